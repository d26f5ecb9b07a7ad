"""Shared machinery of the GPU parity tests: run the C-ABI path on seeded inputs and compare it with the oracle,
stage by stage (prologue codes / scales / operand bytes bit-exact; integer S and P~V accumulators bit-exact; P codes
within +-1 on <= 0.1 %; O within 2e-2 / cosine >= 0.9999 - BASELINE.json north_star).  Imported by tests only."""
import numpy as np
import torch

from oracle import rotattn_oracle as orc

O_ATOL = 2e-2       # north_star: max-abs 2e-2
O_COS = 0.9999      # north_star: cosine >= 0.9999
P_FRAC = 1e-3       # north_star: P codes differ by +-1 on <= 0.1 % of elements


def api():
    from paper_2607_02584_b200 import api as _api
    return _api


def oracle_params(w, H, **kw):
    return orc.Params(w.B, H, w.N, w.D, w.grid, w.pairs, **kw)


def table_for(p, po, rot=None):
    """The library's coefficient table; where libm and NumPy disagree on a rounding tie the oracle's table is fed to the
    kernels instead (bit-exact prologue) - the table itself is compared in tests/test_host_logic.py."""
    tab = api().rotattn_build_tables(p, rot)
    want = orc.coef_table(po, rot)
    return tab if np.array_equal(tab, want) else want


def run_path(w, q, k, v, rot=None, use_ws=True, want_fp16=False, **modes):
    """prepare_qk -> quant_v -> fwd_int4 through the C-ABI on numpy fp16 [B,H',N,D]; modes: rot_mode, p_mode, p_norm,
    qk_group, v_scale, smooth.  Returns (res dict of device tensors, oracle Params, table)."""
    a = api()
    H = q.shape[1]
    p = a.params_for(w, H=H, **modes)
    po = oracle_params(w, H, **modes)
    tab = table_for(p, po, rot)
    res = a.run_int4(w, q, k, v, want_fp16=want_fp16, coef=tab, rot=rot, use_ws=use_ws, **modes)
    torch.cuda.synchronize()
    return res, po, tab


def cos(a, b):
    a, b = a.ravel().astype(np.float64), b.ravel().astype(np.float64)
    return float(a @ b / (np.linalg.norm(a) * np.linalg.norm(b) + 1e-300))


def check_o(got, want):
    assert np.isfinite(got).all()
    assert np.abs(got - want).max() <= O_ATOL, np.abs(got - want).max()
    assert cos(got, want) >= O_COS, cos(got, want)


def _operand_codes(x):
    """operand bytes are sign-magnitude (= E4M3 encoding of code * 2^-9)"""
    x = x.view(np.uint8).astype(np.int32)
    assert not np.any(x == 0x80), 'negative zero byte'
    return np.where(x & 0x80, -(x & 0x7F), x & 0x7F).astype(np.int8)


def oracle_prologue_head(po, tab, q_h, k_h, v_h, rot=None):
    """The oracle's prologue of one head from the fp16 inputs: (pq dict, v codes, v scales, means or None)."""
    means = orc.smooth_means(po, q_h, k_h, v_h, tab, rot) if po.smooth else None
    pq = orc.prepare_qk_head(po, q_h, k_h, tab, rot, means=None if means is None else means[:2])
    vc, vs = orc.quant_v(v_h, po.v_group, po.v_scale, mean=None if means is None else means[2])
    return pq, vc, vs, means


def check_prologue_head(po, tab, res, q_h, k_h, v_h, bi, h, rot=None, check_ws=True, check_16=False):
    """Q/K/V codes, scales, (fp16 copies,) operand bytes and padded key scales of head (bi, h) against the oracle, from
    the fp16 inputs, bit for bit.  Returns the oracle's prologue for use as attention inputs."""
    b = res['buffers']
    pq, vc, vs, means = oracle_prologue_head(po, tab, q_h, k_h, v_h, rot)
    N, D = po.N, po.D
    assert np.array_equal(b.Q4[bi, h].cpu().numpy(), pq['q_packed']), 'Q codes'
    assert np.array_equal(b.K4[bi, h].cpu().numpy(), pq['k_packed']), 'K codes'
    assert np.array_equal(b.Qs[bi, h].cpu().numpy(), pq['q_scale']), 'Q scales'
    assert np.array_equal(b.Ks[bi, h].cpu().numpy(), pq['k_scale']), 'K scales'
    assert np.array_equal(b.V4[bi, h].cpu().numpy(), orc.pack_nibbles(vc)), 'V codes'
    assert np.array_equal(b.Vs[bi, h].cpu().numpy(), vs), 'V scales'
    if check_16:
        assert np.array_equal(b.Q16[bi, h].cpu().numpy().view(np.uint16), pq['q_16'].view(np.uint16))
        assert np.array_equal(b.K16[bi, h].cpu().numpy().view(np.uint16), pq['k_16'].view(np.uint16))
    if means is not None:
        a = api()
        got_means = torch.empty((po.B, po.H, 3, D), dtype=torch.float32, device='cuda')
        got_kc = torch.empty((po.B, po.H, N), dtype=torch.float32, device='cuda')
        a.rotattn_smooth_read(res['p'], b.ws, got_means, got_kc)
        torch.cuda.synchronize()
        assert np.array_equal(got_means[bi, h].cpu().numpy(), np.stack(means)), 'column means'
        want_kc = pq['k_corr'] * (1.4426950408889634 / np.sqrt(D))
        got = got_kc[bi, h].cpu().numpy().astype(np.float64)
        assert np.abs(got - want_kc).max() <= 1e-5 * max(1.0, np.abs(want_kc).max()), 'per-key correction'
    if check_ws:
        BH = po.B * po.H
        bh = bi * po.H + h
        npad = -(-N // 128) * 128
        qk_bytes = -(-BH * N * 128 // 1024) * 1024
        v_bytes = -(-BH * D * npad // 1024) * 1024
        ws = b.ws
        q8 = _operand_codes(ws[bh * N * 128:(bh + 1) * N * 128].cpu().numpy()).reshape(N, 128)
        k8 = _operand_codes(ws[qk_bytes + bh * N * 128:qk_bytes + (bh + 1) * N * 128].cpu().numpy()).reshape(N, 128)
        v8t = _operand_codes(ws[2 * qk_bytes + bh * D * npad:2 * qk_bytes + (bh + 1) * D * npad].cpu().numpy()).reshape(D, npad)
        assert np.array_equal(q8[:, :D], pq['q_codes']) and np.all(q8[:, D:] == 0)
        assert np.array_equal(k8[:, :D], pq['k_codes']) and np.all(k8[:, D:] == 0)
        assert np.array_equal(v8t[:, :N], vc.T) and np.all(v8t[:, N:] == 0)
        if po.qk_group == 1:
            off = 2 * qk_bytes + v_bytes + bh * npad * 4
            ksp = ws[off:off + N * 4].cpu().numpy().view(np.float32)
            assert np.array_equal(ksp, pq['k_scale']), 'padded key scales'
    return pq, vc, vs, means


def gpu_attention_inputs(res, bi, h):
    """codes / scales the attention kernel consumed, unpacked (use only where the prologue was checked bit for bit)."""
    qc = orc.unpack_nibbles(res['Q4'][bi, h].cpu().numpy())
    kc = orc.unpack_nibbles(res['K4'][bi, h].cpu().numpy())
    vc = orc.unpack_nibbles(res['V4'][bi, h].cpu().numpy())
    return (qc, res['Qs'][bi, h].cpu().numpy(), kc, res['Ks'][bi, h].cpu().numpy(), vc, res['Vs'][bi, h].cpu().numpy())


def debug_tile(res, po, bh, q_tile, with_pv=True):
    a = api()
    p = res['p']
    nblk = -(-po.N // 128)
    npad = nblk * 128
    S = torch.zeros((128, npad), dtype=torch.int32, device='cuda')
    P = torch.zeros((128, npad), dtype=torch.uint8, device='cuda')
    PV = torch.zeros((nblk, 128, po.D), dtype=torch.int32, device='cuda') if with_pv else None
    Ot = torch.zeros((128, po.D), dtype=torch.float16, device='cuda')
    b = res['buffers']
    a.rotattn_fwd_int4_debug(p, b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, bh, q_tile, S, P, Ot, b.ws, a.ws_state_full(p),
                             PV_dump=PV)
    torch.cuda.synchronize()
    return S.cpu().numpy(), P.cpu().numpy(), None if PV is None else PV.cpu().numpy(), Ot.float().cpu().numpy()


def check_tile(res, po, bi, h, q_tile, inputs=None, k_corr=None, v_mean=None, stats=None):
    """One query tile of head (bi, h): integer S bit-exact, P codes +-1 on <= 0.1 %, integer P~V bit-exact given the GPU's own
    P codes (so that a tolerated +-1 code does not hide an inexact product), O of the debug launch and of the full launch."""
    N = po.N
    rows = np.arange(q_tile * 128, min(N, (q_tile + 1) * 128))
    qc, qs, kc, ks, vc, vs = gpu_attention_inputs(res, bi, h) if inputs is None else inputs
    Ow, acc, codes = orc.o_quant(po, qc, qs, kc, ks, vc, vs, rows=rows, dump=True, k_corr=k_corr, v_mean=v_mean)
    S, P, PV, Ot = debug_tile(res, po, bi * po.H + h, q_tile, with_pv=po.p_norm == orc.NORM_ROWBLOCK)
    nr = len(rows)
    assert np.array_equal(S[:nr, :N], acc), 'integer QK^T accumulators differ'
    diff = np.abs(P[:nr, :N].astype(np.int16) - codes)
    assert diff.max() <= 1
    frac = float((diff != 0).mean())
    assert frac <= P_FRAC, frac
    assert np.all(P[:nr, N:] == 0)
    if PV is not None:
        nblk = -(-N // 128)
        Ppad = np.zeros((nr, nblk * 128), dtype=np.float64)       # fp64 BLAS on integer-valued codes is exact (< 2^53)
        Ppad[:, :N] = P[:nr, :N]
        vpad = np.zeros((nblk * 128, po.D), dtype=np.float64)
        vpad[:N] = vc
        want_pv = np.matmul(Ppad.reshape(nr, nblk, 128).transpose(1, 0, 2), vpad.reshape(nblk, 128, po.D))
        assert np.array_equal(PV[:, :nr, :].astype(np.float64), want_pv), 'integer P~V accumulators differ'
    check_o(Ot[:nr], Ow)
    full = res['O'][bi, h].float().cpu().numpy()[rows]
    check_o(full, Ow)
    if stats is not None:
        stats.append(frac)
