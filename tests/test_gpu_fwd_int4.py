"""GPU parity of rotattn_fwd_int4 against the oracle's same-quantisation attention (O-quant): integer S and P~V accumulators
bit-exact, P codes within +-1 on <= 0.1 % of elements, O within 2e-2 max-abs and cosine >= 0.9999 (BASELINE.json
north_star); at full size the prologue is compared with the oracle from the fp16 inputs first.  Everything goes through
the C-ABI."""
import numpy as np
import pytest

torch = pytest.importorskip('torch')
pytestmark = pytest.mark.gpu

import __graft_entry__ as entry  # noqa: E402

entry.build()
from oracle import rotattn_oracle as orc  # noqa: E402
from synth import video_qkv as syn  # noqa: E402
import parity_helpers as ph  # noqa: E402

F1 = [(128, orc.VSCALE_CHANNEL), (1, orc.VSCALE_GROUP), (128, orc.VSCALE_GROUP)]


@pytest.mark.parametrize('rot_mode', [orc.ROT_NONE, orc.ROT_INTERLEAVED, orc.ROT_HALF, orc.ROT_FULL])
@pytest.mark.parametrize('p_mode', [orc.P_ASYM15, orc.P_SYM7])
@pytest.mark.parametrize('p_norm', [orc.NORM_ROWBLOCK, orc.NORM_RUNNING])
def test_tiny_all_modes(rot_mode, p_mode, p_norm):
    w = syn.TINY
    q, k, v = syn.gen_all(w)
    res, po, tab = ph.run_path(w, q, k, v, rot_mode=rot_mode, p_mode=p_mode, p_norm=p_norm)
    for h in range(w.H):
        pq, vc, vs, _ = ph.check_prologue_head(po, tab, res, q[0, h], k[0, h], v[0, h], 0, h)
        for qt in range(2):
            ph.check_tile(res, po, 0, h, qt, inputs=(pq['q_codes'], pq['q_scale'], pq['k_codes'], pq['k_scale'], vc, vs))


@pytest.mark.parametrize('base', [syn.WAN_1_3B, syn.HUNYUAN])
def test_d128_ragged_multi_tile(base):
    w = syn.small_variant(base, (3, 9, 13), n_text=0 if base.n_text == 0 else 21, H=2)   # N = 351 / 372: 3 tiles, ragged
    q, k, v = syn.gen_all(w)
    res, po, tab = ph.run_path(w, q, k, v, rot_mode=orc.ROT_HALF)
    for h in range(w.H):
        pq, vc, vs, _ = ph.check_prologue_head(po, tab, res, q[0, h], k[0, h], v[0, h], 0, h)
        for qt in range(3):
            ph.check_tile(res, po, 0, h, qt, inputs=(pq['q_codes'], pq['q_scale'], pq['k_codes'], pq['k_scale'], vc, vs))


@pytest.mark.parametrize('grid', [(1, 9, 11), (1, 10, 13), (3, 5, 17), (2, 8, 8)])
@pytest.mark.parametrize('qk_group', [1, 128])
def test_ragged_edge_blocks(grid, qk_group):
    """Degenerate shapes of the masked last KV block: a single ragged block (N = 99: the odd-block softmax group has no work),
    a last block with 2 valid keys (N = 130: every 16-column chunk of it is masked in tensor memory), N = 255 (one key short of
    two full blocks) and an exact multiple (N = 128: no masked column at all)."""
    w = syn.small_variant(syn.WAN_1_3B, grid, H=2)
    q, k, v = syn.gen_all(w)
    res, po, tab = ph.run_path(w, q, k, v, rot_mode=orc.ROT_HALF, qk_group=qk_group)
    for h in range(w.H):
        pq, vc, vs, _ = ph.check_prologue_head(po, tab, res, q[0, h], k[0, h], v[0, h], 0, h)
        for qt in range(-(-w.N // 128)):
            ph.check_tile(res, po, 0, h, qt, inputs=(pq['q_codes'], pq['q_scale'], pq['k_codes'], pq['k_scale'], vc, vs))


@pytest.mark.parametrize('grid', [(1, 9, 11), (1, 10, 13), (3, 9, 13)])
def test_running_normaliser_edge_blocks(grid):
    """p_norm = RUNNING in the one-thread-per-row kernel: the running row max is handed from block j (one softmax group) to
    block j + 1 (the other group).  One ragged block (nobody to hand to), two blocks with 2 valid keys in the second, three
    blocks with a ragged tail."""
    w = syn.small_variant(syn.WAN_1_3B, grid, H=2)
    q, k, v = syn.gen_all(w)
    res, po, tab = ph.run_path(w, q, k, v, rot_mode=orc.ROT_HALF, p_norm=orc.NORM_RUNNING)
    for h in range(w.H):
        pq, vc, vs, _ = ph.check_prologue_head(po, tab, res, q[0, h], k[0, h], v[0, h], 0, h)
        for qt in range(-(-w.N // 128)):
            ph.check_tile(res, po, 0, h, qt, inputs=(pq['q_codes'], pq['q_scale'], pq['k_codes'], pq['k_scale'], vc, vs))


@pytest.mark.parametrize('qk_group,v_scale', F1)
@pytest.mark.parametrize('p_mode', [orc.P_ASYM15, orc.P_SYM7])
def test_granularity_variants_tiny_and_ragged(qk_group, v_scale, p_mode):
    """per-block Q/K scales and per-group V scales, same bounds, all rows of the tiny config plus a
    ragged multi-tile D = 128 case with text tokens."""
    for w in (syn.TINY, syn.small_variant(syn.HUNYUAN, (3, 9, 13), n_text=21, H=2)):
        q, k, v = syn.gen_all(w)
        res, po, tab = ph.run_path(w, q, k, v, rot_mode=orc.ROT_HALF, p_mode=p_mode, qk_group=qk_group, v_scale=v_scale)
        for h in range(w.H):
            pq, vc, vs, _ = ph.check_prologue_head(po, tab, res, q[0, h], k[0, h], v[0, h], 0, h)
            for qt in range(-(-w.N // 128)):
                ph.check_tile(res, po, 0, h, qt, inputs=(pq['q_codes'], pq['q_scale'], pq['k_codes'], pq['k_scale'], vc, vs))


@pytest.mark.parametrize('v_scale', [orc.VSCALE_CHANNEL, orc.VSCALE_GROUP])
def test_zero_block_scales_at_ragged_n(v_scale):
    """qk_group = 128 with an all-zero query tile and an all-zero valid part of the ragged last key block: both block
    scales are exactly 0 (amax = 0 -> zeros), every score of those blocks is 0, and the keys >= N of the last
    block are still masked - 0 * (-inf) must not reach the exponent."""
    w = syn.small_variant(syn.HUNYUAN, (3, 9, 13), n_text=21, H=1)          # N = 372 = 2 * 128 + 116
    q, k, v = syn.gen_all(w)
    q, k = q.copy(), k.copy()
    q[0, 0, 128:256] = 0
    k[0, 0, 256:] = 0
    res, po, tab = ph.run_path(w, q, k, v, rot_mode=orc.ROT_HALF, qk_group=128, v_scale=v_scale)
    pq, vc, vs, _ = ph.check_prologue_head(po, tab, res, q[0, 0], k[0, 0], v[0, 0], 0, 0)
    assert pq['q_scale'][1] == 0 and pq['k_scale'][2] == 0
    assert bool(torch.isfinite(res['O'].float()).all())
    for qt in range(3):
        ph.check_tile(res, po, 0, 0, qt, inputs=(pq['q_codes'], pq['q_scale'], pq['k_codes'], pq['k_scale'], vc, vs))
    ph.check_o(res['O'][0, 0].float().cpu().numpy(),
               orc.o_quant(po, pq['q_codes'], pq['q_scale'], pq['k_codes'], pq['k_scale'], vc, vs))


def test_smooth_needs_the_stats_bit():
    """smooth = 1: fwd_int4 refuses a workspace the caller does not vouch for (ROTATTN_WS_HAS_STATS, include/rotattn.h) instead
    of reading means nobody wrote."""
    api = ph.api()
    w = syn.small_variant(syn.WAN_1_3B, (2, 7, 11), H=1)
    q, k, v = syn.gen_all(w)
    res, po, tab = ph.run_path(w, q, k, v, rot_mode=orc.ROT_HALF, smooth=1)
    b, p = res['buffers'], res['p']
    for state in (0, api.WS_HAS_QK | api.WS_HAS_V, api.WS_HAS_STATS, api.WS_HAS_QK | api.WS_HAS_STATS):
        with pytest.raises(RuntimeError, match='HAS_STATS'):
            api.rotattn_fwd_int4(p, b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, b.O, b.ws, state)
    O2 = torch.zeros_like(b.O)
    api.rotattn_fwd_int4(p, b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, O2, b.ws, api.ws_state_full(p))
    torch.cuda.synchronize()
    assert torch.equal(O2, b.O)


def test_fresh_workspace_unpack_path_and_head_sel():
    """fwd_int4 from the packed public buffers alone (ws_state = 0) and with a head subset."""
    api = ph.api()
    w = syn.small_variant(syn.WAN_1_3B, (2, 9, 13), H=3)
    q, k, v = syn.gen_all(w)
    res, po, tab = ph.run_path(w, q, k, v, rot_mode=orc.ROT_HALF, use_ws=False)
    ph.check_prologue_head(po, tab, res, q[0, 1], k[0, 1], v[0, 1], 0, 1)     # the inputs taken from the GPU below are the oracle's
    qc, qs, kc, ks, vc, vs = ph.gpu_attention_inputs(res, 0, 1)
    ph.check_o(res['O'][0, 1].float().cpu().numpy(), orc.o_quant(po, qc, qs, kc, ks, vc, vs))
    b = res['buffers']
    O2 = torch.full_like(b.O, 7.0)
    sel = torch.tensor([2, 0], dtype=torch.int32, device='cuda')
    api.rotattn_fwd_int4(res['p'], b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, O2, b.ws, api.WS_HAS_QK | api.WS_HAS_V, head_sel=sel)
    torch.cuda.synchronize()
    assert torch.equal(O2[0, 0], b.O[0, 0]) and torch.equal(O2[0, 2], b.O[0, 2])
    assert torch.all(O2[0, 1] == 7.0)


@pytest.mark.parametrize('qk_group,v_scale', [(1, orc.VSCALE_CHANNEL), (128, orc.VSCALE_GROUP)])
def test_diffuse_inputs_codes_cover_range(qk_group, v_scale):
    """No outliers (diffuse attention): the case where P-code rounding matters most - every key of a block lands on a
    non-zero code.  The (128, GROUP) variant evaluates a quarter of its exponentials by a degree-3 polynomial on the FMA pipe
    (fwd_int4_kernel.cuh): same +-1 / 0.1 % bound against the unchanged oracle."""
    w = syn.small_variant(syn.WAN_1_3B, (4, 8, 12), H=1)
    rng = np.random.default_rng(3)
    shape = (1, 1, w.N, w.D)
    q = (rng.standard_normal(shape) * 0.8).astype(np.float16)
    k = (rng.standard_normal(shape) * 0.8).astype(np.float16)
    v = rng.standard_normal(shape).astype(np.float16)
    res, po, tab = ph.run_path(w, q, k, v, rot_mode=orc.ROT_HALF, qk_group=qk_group, v_scale=v_scale)
    stats = []
    for qt in range(3):
        ph.check_tile(res, po, 0, 0, qt, stats=stats)
    print(f'diffuse tiles (qk_group {qk_group}, v_scale {v_scale}): P-code mismatch rates {[f"{x:.2e}" for x in stats]} (bound {ph.P_FRAC:.0e})')
    _, P, _, _ = ph.debug_tile(res, po, 0, 0)
    assert set(np.unique(P[:, :w.N])) == set(range(16))


@pytest.mark.parametrize('rot_mode', [orc.ROT_NONE, orc.ROT_HALF])
def test_smoothing_end_to_end(rot_mode):
    """SURVEY 8f row f2 on inputs with a token-shared bias: prologue bit-exact, S / P / P~V / O within the usual bounds
    (the per-key correction enters S in floating point, so integer S is still the codes' product)."""
    w = syn.small_variant(syn.HUNYUAN, (3, 9, 13), n_text=21, H=2)
    q, k, v = syn.gen_all(w)
    rng = np.random.default_rng(10)
    bias = (rng.standard_normal((1, 2, 1, w.D)) * 2).astype(np.float32)
    q = (q.astype(np.float32) + bias).astype(np.float16)
    k = (k.astype(np.float32) + bias).astype(np.float16)
    v = (v.astype(np.float32) + bias).astype(np.float16)
    res, po, tab = ph.run_path(w, q, k, v, rot_mode=rot_mode, smooth=1)
    for h in range(w.H):
        pq, vc, vs, means = ph.check_prologue_head(po, tab, res, q[0, h], k[0, h], v[0, h], 0, h)
        for qt in range(3):
            ph.check_tile(res, po, 0, h, qt, inputs=(pq['q_codes'], pq['q_scale'], pq['k_codes'], pq['k_scale'], vc, vs),
                          k_corr=pq['k_corr'], v_mean=means[2])


def _crafted(N, D, qc, kc, vc, qs, ks, vs, p_mode=orc.P_ASYM15):
    """Run fwd_int4 on hand-made codes (packed public buffers, fresh workspace): returns (res, po)."""
    api = ph.api()
    w = syn.small_variant(syn.WAN_1_3B if D == 128 else syn.TINY, (1, 1, N), H=1)
    p = api.params_for(w, p_mode=p_mode)
    po = ph.oracle_params(w, 1, p_mode=p_mode)
    b = api.Buffers(p)
    b.Q4.copy_(torch.from_numpy(orc.pack_nibbles(qc))[None, None])
    b.K4.copy_(torch.from_numpy(orc.pack_nibbles(kc))[None, None])
    b.V4.copy_(torch.from_numpy(orc.pack_nibbles(vc))[None, None])
    b.Qs.copy_(torch.from_numpy(qs)[None, None]); b.Ks.copy_(torch.from_numpy(ks)[None, None]); b.Vs.copy_(torch.from_numpy(vs)[None, None])
    api.rotattn_fwd_int4(p, b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, b.O, b.ws, 0)
    torch.cuda.synchronize()
    return dict(p=p, buffers=b, Q4=b.Q4, K4=b.K4, V4=b.V4, Qs=b.Qs, Ks=b.Ks, Vs=b.Vs, O=b.O), po


@pytest.mark.parametrize('unit', [1, -1])
def test_adversarial_integer_exactness_in_the_attention_kernel(unit):
    """Maximum dynamic range inside fwd_int4 itself: S accumulators at +-(49 * 127) receiving one +-1-unit product at
    every position of the contraction, and P~V accumulators at 15 * 7 * 127 receiving unit products (flat softmax: every
    P code is 15) - both dumped and compared bit for bit (the E4M3 path is admissible only if exact)."""
    N, D = 384, 128
    qc = np.full((N, D), 7, dtype=np.int8)
    kc = np.full((N, D), 7, dtype=np.int8)
    idx = np.arange(N)
    qc[idx, idx % D] = 1
    kc[idx, idx % D] = unit                       # key j: unit factor at position j mod D -> meets q's unit when i = j mod D
    kc[1::2] *= -1                                # every other key negative: S = -/+ 6223 +- 1
    vc = np.full((N, D), 7, dtype=np.int8)
    vc[idx, idx % D] = unit                       # one unit code per key, at channel j mod D
    vc[:, 1::2] *= -1
    qs = np.full(N, 1e-4, dtype=np.float32)       # tiny scales: s ~ 0, P^ ~ 1, every code saturates at 15
    ks = np.full(N, 1e-4, dtype=np.float32)
    vs = np.ones((3, D), dtype=np.float32)
    res, po = _crafted(N, D, qc, kc, vc, qs, ks, vs)
    for qt in range(3):
        ph.check_tile(res, po, 0, 0, qt)
    S, P, PV, _ = ph.debug_tile(res, po, 0, 0)
    assert np.abs(S).max() >= 49 * 127 - 1 and set(np.unique(P[:, :N])) == {15}
    assert np.abs(PV).max() >= 15 * (7 * 127 - 1)


def test_random_codes_full_range_through_the_attention_kernel():
    """Random codes over the full ranges with random scales: S, P~V bit-exact, P codes and O within bounds."""
    rng = np.random.default_rng(23)
    N, D = 640, 128
    qc = rng.integers(-7, 8, (N, D)).astype(np.int8)
    kc = rng.integers(-7, 8, (N, D)).astype(np.int8)
    vc = rng.integers(-7, 8, (N, D)).astype(np.int8)
    qs = rng.uniform(0.02, 0.08, N).astype(np.float32)
    ks = rng.uniform(0.02, 0.08, N).astype(np.float32)
    vs = rng.uniform(0.1, 0.5, (5, D)).astype(np.float32)
    res, po = _crafted(N, D, qc, kc, vc, qs, ks, vs)
    for qt in range(5):
        ph.check_tile(res, po, 0, 0, qt)


def test_full_size_wan13b_row_sample():
    """BASELINE.json configs[1] at full size, the launch configuration bench.py times; oracle on a seeded row sample."""
    w = syn.WAN_1_3B
    q, k, v = syn.gen_all(w)
    res, po, tab = ph.run_path(w, q, k, v, rot_mode=orc.ROT_HALF)
    for h in (0, 5):
        pq, vc, vs, _ = ph.check_prologue_head(po, tab, res, q[0, h], k[0, h], v[0, h], 0, h)
        inputs = (pq['q_codes'], pq['q_scale'], pq['k_codes'], pq['k_scale'], vc, vs)
        rows = syn.sample_rows(w, n_tiles=3, head=h)
        tiles = sorted(set((rows // 128).tolist()))
        ph.check_tile(res, po, 0, h, tiles[-1], inputs=inputs)      # ragged last tile, with dumps
        ph.check_o(res['O'][0, h].float().cpu().numpy()[rows], orc.o_quant(po, *inputs, rows=rows))


def _full_size_case(w, heads, n_tiles=3, bi=0, **modes):
    """Full N, D and ALL heads of a BASELINE.json config in one launch (the grid and workspace sizes bench.py uses).  For
    the sampled heads (of batch entry bi): Q/K/V codes, scales and operand bytes against the oracle from the fp16 inputs
    (bit-exact), S / P / P~V dumps on the ragged last tile, O on a seeded row sample."""
    q, k, v = syn.gen_all(w)
    res, po, tab = ph.run_path(w, q, k, v, **modes)
    assert res['O'].shape[:2] == (w.B, w.H)
    for h in heads:
        pq, vc, vs, _ = ph.check_prologue_head(po, tab, res, q[bi, h], k[bi, h], v[bi, h], bi, h)
        inputs = (pq['q_codes'], pq['q_scale'], pq['k_codes'], pq['k_scale'], vc, vs)
        rows = syn.sample_rows(w, n_tiles=n_tiles, head=h)
        tiles = sorted(set((rows // 128).tolist()))
        ph.check_tile(res, po, bi, h, tiles[-1], inputs=inputs)
        ph.check_o(res['O'][bi, h].float().cpu().numpy()[rows], orc.o_quant(po, *inputs, rows=rows))
    # no head was left unwritten / non-finite
    assert bool(torch.isfinite(res['O'].float()).all())
    del res
    torch.cuda.empty_cache()


NAIVE = dict(rot_mode=orc.ROT_NONE, p_mode=orc.P_SYM7)       # north_star: naive symmetric-INT4, no-rotation baseline


def test_full_size_wan14b_all_heads():
    """BASELINE.json configs[2] (H = 40, N = 75600, per-head outlier pairs with magnitudes U(5,25)); heads 0 and 39 checked."""
    _full_size_case(syn.WAN_14B, [0, 39], rot_mode=orc.ROT_HALF)


def test_full_size_wan14b_naive_mode():
    _full_size_case(syn.WAN_14B, [17], n_tiles=2, **NAIVE)


def test_full_size_hunyuan_all_heads_with_text_tokens():
    """BASELINE.json configs[3] (H = 24, N = 118800 video + 256 text tokens without RoPE, split 8/28/28); heads 3 and 23."""
    _full_size_case(syn.HUNYUAN, [3, 23], rot_mode=orc.ROT_HALF)


def test_full_size_hunyuan_naive_mode():
    _full_size_case(syn.HUNYUAN, [11], n_tiles=2, **NAIVE)


@pytest.mark.parametrize('idx', [0, 1, 2, 3, 4])
def test_sweep_points_all_heads(idx):
    """BASELINE.json configs[4]: every sweep point (N = 4096 .. 131072, H = 24, split 8/28/28) in the headline mode."""
    _full_size_case(syn.SWEEP[idx], [1, 22] if idx < 3 else [1], n_tiles=2, rot_mode=orc.ROT_HALF)


def test_sweep_naive_mode_and_granularity_variants_at_16384():
    _full_size_case(syn.SWEEP[1], [2], n_tiles=2, **NAIVE)
    _full_size_case(syn.SWEEP[1], [5], n_tiles=2, rot_mode=orc.ROT_HALF, qk_group=128, v_scale=orc.VSCALE_GROUP)


def test_full_size_d64_and_batch_of_two():
    """SURVEY 8f row f4 at the bench's N = 32760: D = 64 with 24 heads (pairs 12/10/10) and B = 2 (unit = b * H + h, the second
    batch entry checked) - the two shapes bench.py times in its `variants` block."""
    from dataclasses import replace
    _full_size_case(replace(syn.WAN_1_3B, H=24, D=64, pairs=(12, 10, 10), name='wan1.3b-d64'), [0, 23], n_tiles=2, rot_mode=orc.ROT_HALF)
    _full_size_case(replace(syn.WAN_1_3B, B=2, H=6, name='wan1.3b-b2'), [5], n_tiles=2, bi=1, rot_mode=orc.ROT_HALF)


def test_mixed_precision_step_head_split():
    """configs[4] schedule step: FP16 fallback on a head subset, INT4 on the rest, both through head_sel into one O."""
    api = ph.api()
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
    w = syn.small_variant(syn.HUNYUAN, (3, 9, 13), n_text=21, H=2)
    q, k, v = syn.gen_all(w)
    res, po, tab = ph.run_path(w, q, k, v, rot_mode=orc.ROT_HALF, p_mode=p_mode, p_norm=orc.NORM_RUNNING)
    for h in range(w.H):
        pq, vc, vs, _ = ph.check_prologue_head(po, tab, res, q[0, h], k[0, h], v[0, h], 0, h)
        for qt in range(3):
            ph.check_tile(res, po, 0, h, qt, inputs=(pq['q_codes'], pq['q_scale'], pq['k_codes'], pq['k_scale'], vc, vs))


def test_batch_of_two_and_d64_many_tiles():
    """B = 2 (unit index = b * H + h) and D = 64 over 9 KV blocks with a ragged tail."""
    from dataclasses import replace
    w = replace(syn.small_variant(syn.TINY, (4, 16, 17), H=2), B=2)      # N = 1088 = 8 * 128 + 64
    q, k, v = syn.gen_all(w)
    res, po, tab = ph.run_path(w, q, k, v, rot_mode=orc.ROT_INTERLEAVED)
    for bi in range(2):
        for h in range(2):
            pq, vc, vs, _ = ph.check_prologue_head(po, tab, res, q[bi, h], k[bi, h], v[bi, h], bi, h)
            ph.check_o(res['O'][bi, h].float().cpu().numpy(),
                       orc.o_quant(po, pq['q_codes'], pq['q_scale'], pq['k_codes'], pq['k_scale'], vc, vs))
    ph.check_tile(res, po, 1, 1, 8)


def test_cuda_graph_capture_of_the_step():
    """prepare_qk -> quant_v -> fwd_int4 (+ the FP16 head subset on a forked stream) captured once as a
    CUDA graph; the replay reproduces the eager result bit for bit (the library enqueues only, never synchronises)."""
    api = ph.api()
    w = syn.small_variant(syn.SWEEP[0], (4, 16, 16), H=4)          # N = 1024
    q, k, v = syn.gen_all(w)
    p = api.params_for(w, rot_mode=orc.ROT_HALF)
    coef = torch.from_numpy(api.rotattn_build_tables(p)).cuda()
    Q, K, V = (torch.from_numpy(x).cuda() for x in (q, k, v))
    b = api.Buffers(p, want_fp16=True)
    sel4 = torch.tensor([0, 2, 3], dtype=torch.int32, device='cuda')
    sel16 = torch.tensor([1], dtype=torch.int32, device='cuda')
    s2 = torch.cuda.Stream()
    O = torch.zeros_like(b.O)

    def step(out):
        cur = torch.cuda.current_stream()
        api.rotattn_prepare_qk(p, coef, None, Q, K, b.Q4, b.Qs, b.K4, b.Ks, b.Q16, b.K16, b.ws)
        s2.wait_stream(cur)
        with torch.cuda.stream(s2):
            api.rotattn_fwd_fp16(p, b.Q16, b.K16, V, out, b.ws16, head_sel=sel16, stream=s2)
        api.rotattn_quant_v(p, V, b.V4, b.Vs, b.ws)
        api.rotattn_fwd_int4(p, b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, out, b.ws, api.WS_HAS_QK | api.WS_HAS_V, head_sel=sel4)
        cur.wait_stream(s2)
    step(O)                                        # eager (also warms up the per-kernel attribute setup)
    torch.cuda.synchronize()
    want = O.clone()
    O2 = torch.zeros_like(O)
    gs = torch.cuda.Stream()
    with torch.cuda.stream(gs):
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=gs):
            step(O2)
        torch.cuda.synchronize()
        assert torch.all(O2 == 0)                  # capture does not execute
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(O2, want)
        O2.zero_()
        g.replay(); g.replay()
        torch.cuda.synchronize()
        assert torch.equal(O2, want)
