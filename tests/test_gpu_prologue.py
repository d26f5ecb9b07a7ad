"""GPU parity of the prologue kernels (prepare_qk, quant_v) against the oracle: INT4 codes, scales and
fp16 RoPE'd copies bit-exact, through the C-ABI."""
import numpy as np
import pytest

torch = pytest.importorskip('torch')
pytestmark = pytest.mark.gpu

import __graft_entry__ as entry  # noqa: E402

entry.build()
from oracle import rotattn_oracle as orc  # noqa: E402
from synth import video_qkv as syn  # noqa: E402


def _api():
    from paper_2607_02584_b200 import api
    return api


def _run_prologue(w, q, k, v, rot_mode, rot=None, with_ws=True):
    api = _api()
    p = api.params_for(w, rot_mode, H=q.shape[1])
    po = orc.Params(w.B, q.shape[1], w.N, w.D, w.grid, w.pairs, rot_mode=rot_mode)
    tab = api.rotattn_build_tables(p, rot)
    want_tab = orc.coef_table(po, rot)
    if not np.array_equal(tab, want_tab):       # libm ties: feed the oracle's table (bit-exact prologue)
        tab = want_tab
    coef_dev = torch.from_numpy(np.ascontiguousarray(tab)).cuda()
    rot_dev = None if rot is None else torch.from_numpy(np.ascontiguousarray(rot, dtype=np.float32)).cuda()
    Q, K, V = (torch.from_numpy(x).cuda() for x in (q, k, v))
    b = api.Buffers(p, want_fp16=True)
    ws = b.ws if with_ws else None
    if with_ws:
        b.ws.fill_(0x5A)
    api.rotattn_prepare_qk(p, coef_dev, rot_dev, Q, K, b.Q4, b.Qs, b.K4, b.Ks, b.Q16, b.K16, ws)
    api.rotattn_quant_v(p, V, b.V4, b.Vs, ws)
    torch.cuda.synchronize()
    return p, po, tab, b


def _check_head(po, tab, b, q, k, v, bi, h, rot=None, check_ws=True):
    pq = orc.prepare_qk_head(po, q[bi, h], k[bi, h], tab, rot)
    vc, vs = orc.quant_v(v[bi, h])
    N, D = po.N, po.D
    assert np.array_equal(b.Q4[bi, h].cpu().numpy(), pq['q_packed'])
    assert np.array_equal(b.K4[bi, h].cpu().numpy(), pq['k_packed'])
    assert np.array_equal(b.Qs[bi, h].cpu().numpy(), pq['q_scale'])
    assert np.array_equal(b.Ks[bi, h].cpu().numpy(), pq['k_scale'])
    assert np.array_equal(b.Q16[bi, h].cpu().numpy().view(np.uint16), pq['q_16'].view(np.uint16))
    assert np.array_equal(b.K16[bi, h].cpu().numpy().view(np.uint16), pq['k_16'].view(np.uint16))
    assert np.array_equal(b.V4[bi, h].cpu().numpy(), orc.pack_nibbles(vc))
    assert np.array_equal(b.Vs[bi, h].cpu().numpy(), vs)
    if check_ws:
        BH = po.B * po.H
        bh = bi * po.H + h
        npad = -(-N // 128) * 128
        qk_bytes = -(-BH * N * 128 // 1024) * 1024
        ws = b.ws.cpu().numpy()

        def codes(x):      # widened operand bytes are sign-magnitude (= E4M3 encoding of code * 2^-9)
            x = x.view(np.uint8).astype(np.int32)
            assert not np.any(x == 0x80), 'negative zero byte'
            return np.where(x & 0x80, -(x & 0x7F), x & 0x7F).astype(np.int8)
        q8 = codes(ws[:BH * N * 128]).reshape(BH, N, 128)[bh]
        k8 = codes(ws[qk_bytes:qk_bytes + BH * N * 128]).reshape(BH, N, 128)[bh]
        v8t = codes(ws[2 * qk_bytes:2 * qk_bytes + BH * D * npad]).reshape(BH, D, npad)[bh]
        assert np.array_equal(q8[:, :D], pq['q_codes']) and np.all(q8[:, D:] == 0)
        assert np.array_equal(k8[:, :D], pq['k_codes'])
        assert np.array_equal(v8t[:, :N], vc.T) and np.all(v8t[:, N:] == 0)


@pytest.mark.parametrize('rot_mode', [orc.ROT_NONE, orc.ROT_INTERLEAVED, orc.ROT_HALF])
def test_tiny_all_heads(rot_mode):
    w = syn.TINY
    q, k, v = syn.gen_all(w)
    p, po, tab, b = _run_prologue(w, q, k, v, rot_mode)
    for h in range(w.H):
        _check_head(po, tab, b, q, k, v, 0, h)


def test_random_o2_blocks_half_and_interleaved():
    w = syn.TINY
    q, k, v = syn.gen_all(w)
    rng = np.random.default_rng(5)
    th = rng.uniform(0, 2 * np.pi, w.D // 2)
    rot = np.stack([np.cos(th), np.sin(th), np.sin(th), -np.cos(th)], 1).astype(np.float32)   # reflections
    for mode in (orc.ROT_HALF, orc.ROT_INTERLEAVED):
        p, po, tab, b = _run_prologue(w, q, k, v, mode, rot)
        _check_head(po, tab, b, q, k, v, 0, 1, rot)


@pytest.mark.parametrize('base', [syn.WAN_1_3B, syn.HUNYUAN])
def test_d128_ragged_with_text_tokens(base):
    # reduced grids: several 128-token groups, ragged tail (N mod 128 != 0), odd pair counts, text tokens
    w = syn.small_variant(base, (3, 6, 13), n_text=0 if base.n_text == 0 else 19, H=3)
    q, k, v = syn.gen_all(w)
    for mode in (orc.ROT_HALF, orc.ROT_INTERLEAVED):
        p, po, tab, b = _run_prologue(w, q, k, v, mode)
        for h in range(w.H):
            _check_head(po, tab, b, q, k, v, 0, h)


def test_zero_rows_and_no_workspace():
    w = syn.small_variant(syn.WAN_1_3B, (2, 5, 9), H=1)
    q, k, v = syn.gen_all(w)
    q[0, 0, 7] = 0
    k[0, 0, 11] = 0
    v[0, 0, :, 5] = 0
    p, po, tab, b = _run_prologue(w, q, k, v, orc.ROT_HALF, with_ws=False)
    _check_head(po, tab, b, q, k, v, 0, 0, check_ws=False)
    assert b.Qs[0, 0, 7].item() == 0 and b.Vs[0, 0, 0, 5].item() == 0


def test_full_size_wan13b_sampled_heads():
    """BASELINE.json configs[1] at full size (the launch configuration bench.py times); oracle on 2 heads."""
    w = syn.WAN_1_3B
    heads = [0, 7]
    q, k, v = syn.gen_all(w)
    p, po, tab, b = _run_prologue(w, q, k, v, orc.ROT_HALF)
    for h in heads:
        _check_head(po, tab, b, q, k, v, 0, h)
