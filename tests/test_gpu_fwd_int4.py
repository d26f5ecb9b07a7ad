"""GPU parity of rotattn_fwd_int4 against the oracle's same-quantisation attention (O-quant):
int32 S accumulators bit-exact, P codes within +-1 on <= 0.1 % of elements, O within 2e-2 max-abs and
cosine >= 0.9999 (BASELINE.json north_star).  Everything goes through the C-ABI."""
import numpy as np
import pytest

torch = pytest.importorskip('torch')
pytestmark = pytest.mark.gpu

import __graft_entry__ as entry  # noqa: E402

entry.build()
from oracle import rotattn_oracle as orc  # noqa: E402
from synth import video_qkv as syn  # noqa: E402

O_ATOL = 2e-2       # north_star: max-abs 2e-2
O_COS = 0.9999      # north_star: cosine >= 0.9999
P_FRAC = 1e-3       # north_star: P codes differ by +-1 on <= 0.1 % of elements


def _api():
    from paper_2607_02584_b200 import api
    return api


def _oracle_inputs(res, bi, h):
    """codes/scales the kernel consumed (already proven bit-exact against the oracle's prologue in test_gpu_prologue)."""
    qc = orc.unpack_nibbles(res['Q4'][bi, h].cpu().numpy())
    kc = orc.unpack_nibbles(res['K4'][bi, h].cpu().numpy())
    vc = orc.unpack_nibbles(res['V4'][bi, h].cpu().numpy())
    return (qc, res['Qs'][bi, h].cpu().numpy(), kc, res['Ks'][bi, h].cpu().numpy(), vc, res['Vs'][bi, h].cpu().numpy())


def _cos(a, b):
    a, b = a.ravel().astype(np.float64), b.ravel().astype(np.float64)
    return float(a @ b / (np.linalg.norm(a) * np.linalg.norm(b) + 1e-300))


def _check_o(got, want):
    assert np.isfinite(got).all()
    assert np.abs(got - want).max() <= O_ATOL, np.abs(got - want).max()
    assert _cos(got, want) >= O_COS, _cos(got, want)


def _debug_tile(api, res, po, bh, q_tile):
    p = res['p']
    npad = -(-po.N // 128) * 128
    S = torch.zeros((128, npad), dtype=torch.int32, device='cuda')
    P = torch.zeros((128, npad), dtype=torch.uint8, device='cuda')
    Ot = torch.zeros((128, po.D), dtype=torch.float16, device='cuda')
    b = res['buffers']
    api.rotattn_fwd_int4_debug(p, b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, bh, q_tile, S, P, Ot, b.ws,
                               api.WS_HAS_QK | api.WS_HAS_V)
    torch.cuda.synchronize()
    return S.cpu().numpy(), P.cpu().numpy(), Ot.float().cpu().numpy()


def _check_tile(api, res, po, bi, h, q_tile, p_mode, p_norm):
    N = po.N
    rows = np.arange(q_tile * 128, min(N, (q_tile + 1) * 128))
    qc, qs, kc, ks, vc, vs = _oracle_inputs(res, bi, h)
    Ow, acc, codes = orc.o_quant(po, qc, qs, kc, ks, vc, vs, rows=rows, dump=True, p_mode=p_mode, p_norm=p_norm)
    S, P, Ot = _debug_tile(api, res, po, bi * po.H + h, q_tile)
    nr = len(rows)
    assert np.array_equal(S[:nr, :N], acc), 'int32 QK^T accumulators differ'
    diff = np.abs(P[:nr, :N].astype(np.int16) - codes)
    assert diff.max() <= 1
    assert (diff != 0).mean() <= P_FRAC, (diff != 0).mean()
    assert np.all(P[:nr, N:] == 0)
    _check_o(Ot[:nr], Ow)
    full = res['O'][bi, h].float().cpu().numpy()[rows]
    _check_o(full, Ow)


@pytest.mark.parametrize('rot_mode', [orc.ROT_NONE, orc.ROT_INTERLEAVED, orc.ROT_HALF])
@pytest.mark.parametrize('p_mode', [orc.P_ASYM15, orc.P_SYM7])
@pytest.mark.parametrize('p_norm', [orc.NORM_ROWBLOCK, orc.NORM_RUNNING])
def test_tiny_all_modes(rot_mode, p_mode, p_norm):
    api = _api()
    w = syn.TINY
    q, k, v = syn.gen_all(w)
    res = api.run_int4(w, q, k, v, rot_mode=rot_mode, p_mode=p_mode, p_norm=p_norm)
    torch.cuda.synchronize()
    po = orc.Params(w.B, w.H, w.N, w.D, w.grid, w.pairs, rot_mode=rot_mode, p_mode=p_mode, p_norm=p_norm)
    for h in range(w.H):
        for qt in range(2):
            _check_tile(api, res, po, 0, h, qt, p_mode, p_norm)


@pytest.mark.parametrize('base', [syn.WAN_1_3B, syn.HUNYUAN])
def test_d128_ragged_multi_tile(base):
    api = _api()
    w = syn.small_variant(base, (3, 9, 13), n_text=0 if base.n_text == 0 else 21, H=2)   # N = 351 / 372: 3 tiles, ragged
    q, k, v = syn.gen_all(w)
    res = api.run_int4(w, q, k, v, rot_mode=orc.ROT_HALF)
    torch.cuda.synchronize()
    po = orc.Params(w.B, w.H, w.N, w.D, w.grid, w.pairs, rot_mode=orc.ROT_HALF)
    for h in range(w.H):
        for qt in range(3):
            _check_tile(api, res, po, 0, h, qt, orc.P_ASYM15, orc.NORM_ROWBLOCK)


def test_fresh_workspace_unpack_path_and_head_sel():
    """fwd_int4 from the packed public buffers alone (ws_state = 0) and with a head subset."""
    api = _api()
    w = syn.small_variant(syn.WAN_1_3B, (2, 9, 13), H=3)
    q, k, v = syn.gen_all(w)
    res = api.run_int4(w, q, k, v, rot_mode=orc.ROT_HALF, use_ws=False)
    torch.cuda.synchronize()
    po = orc.Params(w.B, w.H, w.N, w.D, w.grid, w.pairs, rot_mode=orc.ROT_HALF)
    qc, qs, kc, ks, vc, vs = _oracle_inputs(res, 0, 1)
    _check_o(res['O'][0, 1].float().cpu().numpy(), orc.o_quant(po, qc, qs, kc, ks, vc, vs))
    b = res['buffers']
    O2 = torch.full_like(b.O, 7.0)
    sel = torch.tensor([2, 0], dtype=torch.int32, device='cuda')
    api.rotattn_fwd_int4(res['p'], b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, O2, b.ws, api.WS_HAS_QK | api.WS_HAS_V, head_sel=sel)
    torch.cuda.synchronize()
    assert torch.equal(O2[0, 0], b.O[0, 0]) and torch.equal(O2[0, 2], b.O[0, 2])
    assert torch.all(O2[0, 1] == 7.0)


def test_diffuse_inputs_codes_cover_range():
    """No outliers (diffuse attention): the case where P-code rounding matters most."""
    api = _api()
    w = syn.small_variant(syn.WAN_1_3B, (4, 8, 12), H=1)
    rng = np.random.default_rng(3)
    shape = (1, 1, w.N, w.D)
    q = (rng.standard_normal(shape) * 0.8).astype(np.float16)
    k = (rng.standard_normal(shape) * 0.8).astype(np.float16)
    v = rng.standard_normal(shape).astype(np.float16)
    res = api.run_int4(w, q, k, v, rot_mode=orc.ROT_HALF)
    torch.cuda.synchronize()
    po = orc.Params(1, 1, w.N, w.D, w.grid, w.pairs, rot_mode=orc.ROT_HALF)
    _check_tile(api, res, po, 0, 0, 1, orc.P_ASYM15, orc.NORM_ROWBLOCK)
    _, P, _ = _debug_tile(api, res, po, 0, 0)
    assert set(np.unique(P[:, :w.N])) == set(range(16))


def test_full_size_wan13b_row_sample():
    """BASELINE.json configs[1] at full size, the launch configuration bench.py times; oracle on a seeded row sample."""
    api = _api()
    w = syn.WAN_1_3B
    q, k, v = syn.gen_all(w)
    res = api.run_int4(w, q, k, v, rot_mode=orc.ROT_HALF)
    torch.cuda.synchronize()
    po = orc.Params(w.B, w.H, w.N, w.D, w.grid, w.pairs, rot_mode=orc.ROT_HALF)
    for h in (0, 5):
        rows = syn.sample_rows(w, n_tiles=3, head=h)
        tiles = sorted(set((rows // 128).tolist()))
        _check_tile(api, res, po, 0, h, tiles[-1], orc.P_ASYM15, orc.NORM_ROWBLOCK)      # ragged last tile, with dumps
        qc, qs, kc, ks, vc, vs = _oracle_inputs(res, 0, h)
        Ow = orc.o_quant(po, qc, qs, kc, ks, vc, vs, rows=rows)
        _check_o(res['O'][0, h].float().cpu().numpy()[rows], Ow)


def _full_size_case(w, heads, p_mode=orc.P_ASYM15, rot_mode=orc.ROT_HALF, n_tiles=3):
    """Full N and D of a BASELINE.json config on a seeded subset of its heads (heads are independent units):
    prologue codes bit-exact on the sampled rows' inputs, S/P dumps on the ragged last tile, O on a seeded row sample."""
    api = _api()
    q, k, v = syn.gen_all(w, heads=heads)
    res = api.run_int4(w, q, k, v, rot_mode=rot_mode, p_mode=p_mode)
    torch.cuda.synchronize()
    po = orc.Params(w.B, len(heads), w.N, w.D, w.grid, w.pairs, rot_mode=rot_mode, p_mode=p_mode)
    for i, h in enumerate(heads):
        rows = syn.sample_rows(w, n_tiles=n_tiles, head=h)
        tiles = sorted(set((rows // 128).tolist()))
        _check_tile(api, res, po, 0, i, tiles[-1], p_mode, orc.NORM_ROWBLOCK)
        qc, qs, kc, ks, vc, vs = _oracle_inputs(res, 0, i)
        Ow = orc.o_quant(po, qc, qs, kc, ks, vc, vs, rows=rows, p_mode=p_mode)
        _check_o(res['O'][0, i].float().cpu().numpy()[rows], Ow)
    return res, po


def test_full_size_wan14b_row_sample():
    """BASELINE.json configs[2] (N = 75600, per-head outlier pairs with magnitudes U(5,25)), heads 0 and 17."""
    _full_size_case(syn.WAN_14B, [0, 17])


def test_full_size_hunyuan_row_sample_with_text_tokens():
    """BASELINE.json configs[3] (N = 118800 video + 256 text tokens without RoPE, split 8/28/28), heads 3 and 11."""
    _full_size_case(syn.HUNYUAN, [3, 11])


def test_sweep_largest_n_and_naive_mode():
    """BASELINE.json configs[4]: the largest sweep point (N = 131072) in the headline mode, and the naive
    symmetric-INT4 / no-rotation baseline (NONE + SYM7) at N = 16384."""
    _full_size_case(syn.SWEEP[4], [1], n_tiles=2)
    _full_size_case(syn.SWEEP[1], [2], p_mode=orc.P_SYM7, rot_mode=orc.ROT_NONE, n_tiles=2)


def test_mixed_precision_step_head_split():
    """configs[4] schedule step: FP16 fallback on a head subset, INT4 on the rest, both through head_sel into one O."""
    api = _api()
    w = syn.small_variant(syn.SWEEP[0], (4, 16, 16), H=5)          # N = 1024
    q, k, v = syn.gen_all(w)
    res = api.run_int4(w, q, k, v, rot_mode=orc.ROT_HALF, want_fp16=True)
    b, p = res['buffers'], res['p']
    pol = dict(n_steps=50, n_blocks=1, first_steps=5, last_steps=0, first_blocks=0, last_blocks=0, fp16_head_mask=[0, 1, 0, 0, 1])
    i4, f16 = api.rotattn_policy_split_heads(pol, 7, 0, w.B, w.H)
    assert i4.tolist() == [0, 2, 3] and f16.tolist() == [1, 4]
    O = torch.full_like(b.O, 9.0)
    api.rotattn_fwd_int4(p, b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, O, b.ws, api.WS_HAS_QK | api.WS_HAS_V,
                         head_sel=torch.from_numpy(i4).cuda())
    api.rotattn_fwd_fp16(p, b.Q16, b.K16, res['V'], O, b.ws16, head_sel=torch.from_numpy(f16).cuda())
    torch.cuda.synchronize()
    for h in range(w.H):
        want = b.O16[0, h] if h in (1, 4) else b.O[0, h]
        assert torch.equal(O[0, h], want)
    i4, f16 = api.rotattn_policy_split_heads(pol, 2, 0, w.B, w.H)   # inside the first 5 steps: everything FP16
    assert len(i4) == 0 and f16.tolist() == [0, 1, 2, 3, 4]


@pytest.mark.parametrize('p_mode', [orc.P_ASYM15, orc.P_SYM7])
def test_d128_running_normaliser_ragged(p_mode):
    """p_norm = RUNNING (the other reading of Eq.12's normaliser) at D = 128 over several ragged tiles."""
    api = _api()
    w = syn.small_variant(syn.HUNYUAN, (3, 9, 13), n_text=21, H=2)
    q, k, v = syn.gen_all(w)
    res = api.run_int4(w, q, k, v, rot_mode=orc.ROT_HALF, p_mode=p_mode, p_norm=orc.NORM_RUNNING)
    torch.cuda.synchronize()
    po = orc.Params(w.B, w.H, w.N, w.D, w.grid, w.pairs, rot_mode=orc.ROT_HALF, p_mode=p_mode, p_norm=orc.NORM_RUNNING)
    for h in range(w.H):
        for qt in range(3):
            _check_tile(api, res, po, 0, h, qt, p_mode, orc.NORM_RUNNING)


def test_batch_of_two_and_d64_many_tiles():
    """B = 2 (unit index = b * H + h) and D = 64 over 9 KV blocks with a ragged tail."""
    api = _api()
    from dataclasses import replace
    w = replace(syn.small_variant(syn.TINY, (4, 16, 17), H=2), B=2)      # N = 1088 = 8 * 128 + 64
    q, k, v = syn.gen_all(w)
    res = api.run_int4(w, q, k, v, rot_mode=orc.ROT_INTERLEAVED)
    torch.cuda.synchronize()
    po = orc.Params(w.B, w.H, w.N, w.D, w.grid, w.pairs, rot_mode=orc.ROT_INTERLEAVED)
    for bi in range(2):
        for h in range(2):
            qc, qs, kc, ks, vc, vs = _oracle_inputs(res, bi, h)
            _check_o(res['O'][bi, h].float().cpu().numpy(), orc.o_quant(po, qc, qs, kc, ks, vc, vs))
    _check_tile(api, res, po, 1, 1, 8, orc.P_ASYM15, orc.NORM_ROWBLOCK)
