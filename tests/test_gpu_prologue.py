"""GPU parity of the prologue kernels (prepare_qk, quant_v, smoothing pre-pass) against the oracle: INT4 codes, scales,
fp16 RoPE'd copies, operand bytes and column means bit-exact, through the C-ABI."""
import numpy as np
import pytest

torch = pytest.importorskip('torch')
pytestmark = pytest.mark.gpu

import __graft_entry__ as entry  # noqa: E402

entry.build()
from oracle import rotattn_oracle as orc  # noqa: E402
from synth import video_qkv as syn  # noqa: E402
import parity_helpers as ph  # noqa: E402


def _run_prologue(w, q, k, v, rot=None, with_ws=True, **modes):
    """prepare_qk + quant_v only (no attention); returns (res-like dict, oracle params, table)."""
    api = ph.api()
    p = api.params_for(w, H=q.shape[1], **modes)
    po = ph.oracle_params(w, q.shape[1], **modes)
    tab = ph.table_for(p, po, rot)
    coef_dev = torch.from_numpy(np.ascontiguousarray(tab)).cuda()
    rot_dev = None if rot is None else torch.from_numpy(np.ascontiguousarray(rot, dtype=np.float32)).cuda()
    Q, K, V = (torch.from_numpy(x).cuda() for x in (q, k, v))
    b = api.Buffers(p, want_fp16=True)
    ws = b.ws if with_ws else None
    if with_ws:
        b.ws.fill_(0x5A)
    if modes.get('smooth'):
        api.rotattn_smooth_stats(p, coef_dev, rot_dev, Q, K, V, b.ws)
    api.rotattn_prepare_qk(p, coef_dev, rot_dev, Q, K, b.Q4, b.Qs, b.K4, b.Ks, b.Q16, b.K16, ws)
    api.rotattn_quant_v(p, V, b.V4, b.Vs, ws)
    torch.cuda.synchronize()
    return dict(p=p, buffers=b), po, tab


MODES = [orc.ROT_NONE, orc.ROT_INTERLEAVED, orc.ROT_HALF, orc.ROT_FULL]


@pytest.mark.parametrize('rot_mode', MODES)
def test_tiny_all_heads(rot_mode):
    w = syn.TINY
    q, k, v = syn.gen_all(w)
    res, po, tab = _run_prologue(w, q, k, v, rot_mode=rot_mode)
    for h in range(w.H):
        ph.check_prologue_head(po, tab, res, q[0, h], k[0, h], v[0, h], 0, h, check_16=True)


def test_random_o2_blocks_half_and_interleaved():
    w = syn.TINY
    q, k, v = syn.gen_all(w)
    rng = np.random.default_rng(5)
    th = rng.uniform(0, 2 * np.pi, w.D // 2)
    rot = np.stack([np.cos(th), np.sin(th), np.sin(th), -np.cos(th)], 1).astype(np.float32)   # reflections
    for mode in (orc.ROT_HALF, orc.ROT_INTERLEAVED):
        res, po, tab = _run_prologue(w, q, k, v, rot=rot, rot_mode=mode)
        ph.check_prologue_head(po, tab, res, q[0, 1], k[0, 1], v[0, 1], 0, 1, rot=rot, check_16=True)


@pytest.mark.parametrize('base', [syn.WAN_1_3B, syn.HUNYUAN])
def test_d128_ragged_with_text_tokens(base):
    # reduced grids: several 128-token groups, ragged tail (N mod 128 != 0), odd pair counts, text tokens
    w = syn.small_variant(base, (3, 6, 13), n_text=0 if base.n_text == 0 else 19, H=3)
    q, k, v = syn.gen_all(w)
    for mode in (orc.ROT_HALF, orc.ROT_INTERLEAVED, orc.ROT_FULL):
        res, po, tab = _run_prologue(w, q, k, v, rot_mode=mode)
        for h in range(w.H):
            ph.check_prologue_head(po, tab, res, q[0, h], k[0, h], v[0, h], 0, h, check_16=True)


@pytest.mark.parametrize('base', [syn.TINY, syn.HUNYUAN])
@pytest.mark.parametrize('qk_group,v_scale', [(128, orc.VSCALE_CHANNEL), (1, orc.VSCALE_GROUP), (128, orc.VSCALE_GROUP)])
def test_granularity_variants(base, qk_group, v_scale):
    """one Q/K scale per 128-token block, one V scale per 128-token group; ragged tail, text tokens."""
    w = syn.small_variant(base, (3, 6, 13), n_text=0 if base.n_text == 0 else 19, H=2)     # N = 234 / 253
    q, k, v = syn.gen_all(w)
    res, po, tab = _run_prologue(w, q, k, v, rot_mode=orc.ROT_HALF, qk_group=qk_group, v_scale=v_scale)
    for h in range(w.H):
        ph.check_prologue_head(po, tab, res, q[0, h], k[0, h], v[0, h], 0, h, check_16=True)
    nG = -(-w.N // 128)
    b = res['buffers']
    assert tuple(b.Qs.shape) == ((1, 2, nG) if qk_group == 128 else (1, 2, w.N))
    assert tuple(b.Vs.shape) == ((1, 2, nG) if v_scale == orc.VSCALE_GROUP else (1, 2, nG, w.D))


@pytest.mark.parametrize('rot_mode', [orc.ROT_NONE, orc.ROT_HALF, orc.ROT_FULL])
def test_smoothing_means_codes_and_correction(rot_mode):
    """fixed-point column means bit-exact, y - mean codes bit-exact, per-key correction within fp32 rounding."""
    w = syn.small_variant(syn.HUNYUAN, (3, 6, 13), n_text=19, H=2)
    q, k, v = syn.gen_all(w)
    rng = np.random.default_rng(9)
    bias = (rng.standard_normal((1, 2, 1, w.D)) * 3).astype(np.float32)          # token-shared bias (the case smoothing is for)
    q = (q.astype(np.float32) + bias).astype(np.float16)
    k = (k.astype(np.float32) - bias).astype(np.float16)
    v = (v.astype(np.float32) + 0.5 * bias).astype(np.float16)
    res, po, tab = _run_prologue(w, q, k, v, rot_mode=rot_mode, smooth=1)
    for h in range(w.H):
        ph.check_prologue_head(po, tab, res, q[0, h], k[0, h], v[0, h], 0, h, check_16=True)


def test_zero_rows_and_no_workspace():
    w = syn.small_variant(syn.WAN_1_3B, (2, 5, 9), H=1)
    q, k, v = syn.gen_all(w)
    q[0, 0, 7] = 0
    k[0, 0, 11] = 0
    v[0, 0, :, 5] = 0
    res, po, tab = _run_prologue(w, q, k, v, with_ws=False, rot_mode=orc.ROT_HALF)
    ph.check_prologue_head(po, tab, res, q[0, 0], k[0, 0], v[0, 0], 0, 0, check_ws=False, check_16=True)
    b = res['buffers']
    assert b.Qs[0, 0, 7].item() == 0 and b.Vs[0, 0, 0, 5].item() == 0


def test_workspace_too_small_is_reported():
    api = ph.api()
    w = syn.TINY
    q, k, v = syn.gen_all(w)
    p = api.params_for(w)
    coef = torch.from_numpy(api.rotattn_build_tables(p)).cuda()
    Q, K, V = (torch.from_numpy(x).cuda() for x in (q, k, v))
    b = api.Buffers(p, want_fp16=True)
    small = b.ws[:b.ws.numel() - 1]
    for call in (lambda: api.rotattn_prepare_qk(p, coef, None, Q, K, b.Q4, b.Qs, b.K4, b.Ks, None, None, small),
                 lambda: api.rotattn_quant_v(p, V, b.V4, b.Vs, small),
                 lambda: api.rotattn_fwd_int4(p, b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, b.O, small, 0)):
        with pytest.raises(RuntimeError, match=r'workspace too small \(-4\)'):
            call()


def test_full_size_wan13b_sampled_heads():
    """BASELINE.json configs[1] at full size (the launch configuration bench.py times); oracle on 2 heads."""
    w = syn.WAN_1_3B
    q, k, v = syn.gen_all(w)
    res, po, tab = _run_prologue(w, q, k, v, rot_mode=orc.ROT_HALF)
    for h in (0, 7):
        ph.check_prologue_head(po, tab, res, q[0, h], k[0, h], v[0, h], 0, h, check_16=True)
