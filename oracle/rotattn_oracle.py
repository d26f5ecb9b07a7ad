"""CPU oracle for the RotateAttention hot path (arxiv/paper_2607_02584).

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs may import it.  It shares no code
with the CUDA path (paper_2607_02584_b200/): no kernels, headers, helpers, tables or
constants are common; neither imports the other.

Plain NumPy, slow, written so it can be checked against PAPER.md by eye.  Citations are
"PAPER.md:Lnnn" lines of /root/reference/PAPER.md plus the section/equation, and
"DESIGN.md reading n" where the paper is silent/garbled (the readings are listed there).

Two oracles:
  * o_exact  : the plain definition O = softmax(Q_r K_r^T / sqrt(D)) V in fp64
               (Eq.14, S = QK^T/sqrt(D) L157).
  * o_quant  : the INT4 method step by step (an approximation, so the oracle follows the
               algorithm in the paper's order): RoPE (L58-62) -> rotation R (Eq.3-8
               L96-141) -> per-token INT4 Q,K / per-group INT4 V (L190) -> integer
               S = Q4 K4^T (L157) -> block row max / online softmax (L157) ->
               P quantisation (Eq.11 L161 / Eq.12) -> integer P~V with
               zero-point -8 -> fp accumulate -> O / l.
Code-producing arithmetic (RoPE/rotation/quantisers) is fp32, one rounding per
operation, no fused multiply-add (NumPy never contracts), so INT4 codes are
reproducible bit for bit.  Softmax arithmetic is fp64.

Pins: tests/test_oracle_pins.py (-m "not gpu").  Parity status per function:
  hadamard, h2, token_positions (golden triples on an asymmetric grid), rope, coef_table,
  apply_rope_rot (incl. the FULL butterfly), quantisers (per-token / per-block / per-group),
  pack/unpack, integer products, P codes, online softmax, smoothing (column_mean_fixed,
  exactness of the K / Q / V shifts), policy : pinned (see that file).
  INT4-vs-exact *quality numbers* : parity unpinned (paper gives only video-level
  metrics on real weights, Table 1); reported, never asserted.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

ROT_NONE, ROT_INTERLEAVED, ROT_HALF, ROT_FULL = 0, 1, 2, 3
P_ASYM15, P_SYM7 = 0, 1
NORM_ROWBLOCK, NORM_RUNNING = 0, 1
VSCALE_CHANNEL, VSCALE_GROUP = 0, 1

F32 = np.float32
F64 = np.float64


@dataclass
class Params:
    """Problem statement (PAPER.md:L56-62 Q,K,V in R^{N x D}; 3D RoPE split D=D_f+D_h+D_w)."""
    B: int
    H: int
    N: int
    D: int
    grid: tuple            # (T, Hh, W); N_rope = T*Hh*W <= N; tokens >= N_rope carry no RoPE
    pairs: tuple           # (P_t, P_h, P_w), sum == D/2, channel order [t|h|w] (L58, Eq.8)
    rope_base: float = 10000.0
    rot_mode: int = ROT_HALF
    p_mode: int = P_ASYM15
    p_norm: int = NORM_ROWBLOCK
    qk_group: int = 1      # tokens per Q/K scale; 1 = per-token (L190)
    v_group: int = 128     # tokens per V scale group (L190 "per-group"; reading 11)
    kv_block: int = 128    # FlashAttention KV block (L157; reading 18)
    v_scale: int = VSCALE_CHANNEL   # one V scale per (group, channel) (reading 11) | one per group
    smooth: int = 0        # subtract the token mean of Q, K, V before quantisation (L90, L40, L52)

    @property
    def n_rope(self):
        return self.grid[0] * self.grid[1] * self.grid[2]


# ----------------------------------------------------------------------------------
# Hadamard (Eq.4, Eq.13)
# ----------------------------------------------------------------------------------
def h2():
    """H_2 = (1/sqrt 2) [[1,1],[1,-1]]  (Eq.4)."""
    return np.array([[1.0, 1.0], [1.0, -1.0]], dtype=F64) / math.sqrt(2.0)


def hadamard_pm1(n):
    """+-1 Sylvester matrix by the recursion H_{2^k} = H_2 (x) H_{2^{k-1}} (Eq.13), unnormalised."""
    assert n >= 1 and (n & (n - 1)) == 0, "D = 2^n (PAPER.md:L174)"
    H = np.array([[1]], dtype=np.int64)
    H2 = np.array([[1, 1], [1, -1]], dtype=np.int64)
    while H.shape[0] < n:
        H = np.kron(H2, H)
    return H


def hadamard(n):
    """Normalised D x D Hadamard, H H^T = I (Eq.13 with the 1/sqrt2 of Eq.4 in every factor)."""
    return hadamard_pm1(n).astype(F64) / math.sqrt(n)


# ----------------------------------------------------------------------------------
# 3D RoPE (L58-62) and the block-diagonal rotation R (Eq.3)
# ----------------------------------------------------------------------------------
def rope_freqs(P_a, base):
    """f_{a,k} = base^(-k/P_a) = base^(-2k/D_a), k=0..P_a-1, per section (reading 2)."""
    k = np.arange(P_a, dtype=F64)
    return np.power(F64(base), -k / F64(P_a))


def token_positions(N, grid):
    """Token n < N_rope <-> (t,h,w), n = (t*Hh + h)*W + w, w fastest (reading 4).
    Returns int arrays t,h,w of length N and a bool mask is_rope; tokens >= N_rope get pos -1."""
    T, Hh, W = grid
    n = np.arange(N)
    n_rope = T * Hh * W
    is_rope = n < n_rope
    w = np.where(is_rope, n % W, -1)
    h = np.where(is_rope, (n // W) % Hh, -1)
    t = np.where(is_rope, n // (W * Hh), -1)
    return t, h, w, is_rope


def rope_block(theta):
    """M_i in SO(2) (L60), row-vector convention of Eq.7 (x M): M = [[c, s],[-s, c]],
    i.e. y0 = x0 c - x1 s, y1 = x0 s + x1 c on the adjacent pair (2k,2k+1) (reading 1)."""
    c, s = math.cos(theta), math.sin(theta)
    return np.array([[c, s], [-s, c]], dtype=F64)


def default_rot(D):
    """R_i = H_2 for every pair (L100-102, L208)."""
    return np.tile(h2().reshape(1, 4), (D // 2, 1))  # [D/2][r00,r01,r10,r11]


def check_orthogonal(rot, tol=1e-5):
    """R_i in O(2): R_i^T R_i = I (Eq.3; necessity argued L104-120)."""
    R = np.asarray(rot, dtype=F64).reshape(-1, 2, 2)
    err = np.abs(np.einsum('kji,kjl->kil', R, R) - np.eye(2)).max()
    return err <= tol, err


def table_rows(p: Params):
    T, Hh, W = p.grid
    Pt, Ph, Pw = p.pairs
    return (T + 1) * Pt + (Hh + 1) * Ph + (W + 1) * Pw


def coef_table(p: Params, rot=None):
    """Per-axis coefficient table (offline "pre-fusing R into the RoPE weights").
    Layout: for axis a in (t,h,w) with length L_a and P_a pairs: rows pos=0..L_a (row L_a is the
    no-RoPE row for text tokens, reading 7), each with P_a 2x2 blocks [a00,a01,a10,a11].
    NONE/HALF: A = M(theta).  INTERLEAVED: A = M(theta) R_k' (Eq.7), product in fp64.
    Entries rounded once to fp32."""
    D = p.D
    rot64 = default_rot(D) if rot is None else np.asarray(rot, dtype=F64).reshape(D // 2, 4)
    out = np.zeros((table_rows(p), 4), dtype=F64)
    row = 0
    gpair = 0
    for a in range(3):
        L, P = p.grid[a], p.pairs[a]
        f = rope_freqs(P, p.rope_base)
        for pos in range(L + 1):
            for k in range(P):
                M = rope_block(F64(pos) * f[k]) if pos < L else np.eye(2)
                if p.rot_mode == ROT_INTERLEAVED:
                    A = M @ rot64[gpair + k].reshape(2, 2)
                else:
                    A = M
                out[row] = A.reshape(4)
                row += 1
        gpair += P
    return out.astype(F32)


def _gather_coef(p: Params, coef):
    """coef [rows,4] -> per-token blocks [N, D/2, 4] by position lookup."""
    t, h, w, is_rope = token_positions(p.N, p.grid)
    pos = [t, h, w]
    blocks = []
    base = 0
    for a in range(3):
        L, P = p.grid[a], p.pairs[a]
        pa = np.where(is_rope, pos[a], L)          # no-RoPE row for text tokens
        idx = base + pa[:, None] * P + np.arange(P)[None, :]
        blocks.append(coef[idx])                   # [N, P, 4]
        base += (L + 1) * P
    return np.concatenate(blocks, axis=1)


def apply_rope_rot(p: Params, x16, coef, rot=None):
    """Steps 4 of DESIGN.md's algorithm: y = x (M R) in fp32, one rounding per operation.
    x16: fp16 [N, D] (one head).  Returns fp32 [N, D].
      y0 = rn(rn(x0*a00) + rn(x1*a10)),  y1 = rn(rn(x0*a01) + rn(x1*a11))        (Eq.7)
    HALF (Eq.8): within section j, channel o_j+i pairs with o_j+i+D_j/2 through R^j_i,
      u' = rn(rn(u*r00) + rn(v*r10)),  v' = rn(rn(u*r01) + rn(v*r11)), in place (Pi implicit)."""
    N, D = x16.shape
    x = x16.astype(F32)
    A = _gather_coef(p, np.asarray(coef, dtype=F32))  # [N, D/2, 4]
    x0, x1 = x[:, 0::2], x[:, 1::2]
    y = np.empty((N, D), dtype=F32)
    y[:, 0::2] = (x0 * A[..., 0]).astype(F32) + (x1 * A[..., 2]).astype(F32)
    y[:, 1::2] = (x0 * A[..., 1]).astype(F32) + (x1 * A[..., 3]).astype(F32)
    if p.rot_mode == ROT_HALF:
        r = (default_rot(D) if rot is None else np.asarray(rot, dtype=F64).reshape(D // 2, 4)).astype(F32)
        o = 0
        g = 0
        for P in p.pairs:
            u = y[:, o:o + P].copy()
            v = y[:, o + P:o + 2 * P].copy()
            rr = r[g:g + P]
            y[:, o:o + P] = (u * rr[:, 0]).astype(F32) + (v * rr[:, 2]).astype(F32)
            y[:, o + P:o + 2 * P] = (u * rr[:, 1]).astype(F32) + (v * rr[:, 3]).astype(F32)
            o += 2 * P
            g += P
    if p.rot_mode == ROT_FULL:
        y = fwht_fp32(y)
    return y


def fwht_fp32(y):
    """The paper's "Full" rotation baseline (L208: a dense D x D Hadamard applied online after RoPE): y <- y H_D / sqrt(D),
    evaluated as the Sylvester butterfly of Eq.13 (H_{2^n} = H_2 (x) H_{2^{n-1}}) in fp32, one rounding per operation:
    strides 1, 2, ..., D/2 in this order, (a, b) -> (a + b, a - b) with a the lower channel, then one multiplication by
    fl32(1/sqrt(D)).  Pinned against the dense product with hadamard(D) in tests/test_oracle_pins.py."""
    y = np.array(y, dtype=F32, copy=True)
    N, D = y.shape
    s = 1
    while s < D:
        v = y.reshape(N, D // (2 * s), 2, s)
        a, b = v[:, :, 0, :].copy(), v[:, :, 1, :].copy()
        v[:, :, 0, :] = (a + b).astype(F32)
        v[:, :, 1, :] = (a - b).astype(F32)
        y = v.reshape(N, D)
        s *= 2
    return (y * F32(1.0 / math.sqrt(D))).astype(F32)


def rope_fp64(p: Params, x, rot_mode=ROT_NONE, rot=None):
    """fp64 RoPE (and optionally R) on real-valued x [N,D]; used by o_exact and by the pins.
    Independent formulation: builds the dense D x D matrix per token (L60 "block-diagonal M")."""
    N, D = x.shape
    t, h, w, is_rope = token_positions(p.N, p.grid)
    pos = [t, h, w]
    y = np.empty((N, D), dtype=F64)
    R = None
    if rot_mode != ROT_NONE:
        R = dense_rotation(p, rot_mode, rot)
    freqs = [rope_freqs(P, p.rope_base) for P in p.pairs]
    for n in range(N):
        M = np.zeros((D, D), dtype=F64)
        gp = 0
        for a in range(3):
            for k in range(p.pairs[a]):
                th = F64(pos[a][n]) * freqs[a][k] if is_rope[n] else 0.0
                M[2 * gp:2 * gp + 2, 2 * gp:2 * gp + 2] = rope_block(th)
                gp += 1
        v = x[n].astype(F64) @ M
        y[n] = v @ R if R is not None else v
    return y


def rope_fp64_pairs(p: Params, x, rot_mode=ROT_NONE, rot=None):
    """Same map as rope_fp64, evaluated pair by pair (y0 = x0 c - x1 s, y1 = x0 s + x1 c, L60) on whole arrays instead of one
    dense D x D matrix per token: used where N is too large for the dense form (quality references at full size).
    Pinned against rope_fp64 in tests/test_oracle_pins.py."""
    x = np.asarray(x, dtype=F64)
    N, D = x.shape
    t, h, w, is_rope = token_positions(p.N, p.grid)
    pos = [t, h, w]
    y = np.empty((N, D), dtype=F64)
    gp = 0
    for a in range(3):
        P = p.pairs[a]
        th = np.where(is_rope, pos[a], 0).astype(F64)[:, None] * rope_freqs(P, p.rope_base)[None, :]     # [N, P]
        c, sn = np.cos(th), np.sin(th)
        x0, x1 = x[:, 2 * gp:2 * (gp + P):2], x[:, 2 * gp + 1:2 * (gp + P):2]
        y[:, 2 * gp:2 * (gp + P):2] = x0 * c - x1 * sn
        y[:, 2 * gp + 1:2 * (gp + P):2] = x0 * sn + x1 * c
        gp += P
    if rot_mode != ROT_NONE:
        y = y @ dense_rotation(p, rot_mode, rot)
    return y


def dense_rotation(p: Params, rot_mode, rot=None):
    """The D x D orthogonal matrix (Pi R) of Eq.3 (INTERLEAVED) or Eq.8 (HALF) as a dense matrix."""
    D = p.D
    r = default_rot(D) if rot is None else np.asarray(rot, dtype=F64).reshape(D // 2, 4)
    R = np.zeros((D, D), dtype=F64)
    if rot_mode == ROT_INTERLEAVED:
        for k in range(D // 2):
            R[2 * k:2 * k + 2, 2 * k:2 * k + 2] = r[k].reshape(2, 2)
    elif rot_mode == ROT_HALF:
        o = 0
        g = 0
        for P in p.pairs:
            for i in range(P):
                a, b = o + i, o + i + P
                blk = r[g + i].reshape(2, 2)
                R[a, a], R[a, b] = blk[0, 0], blk[0, 1]
                R[b, a], R[b, b] = blk[1, 0], blk[1, 1]
            o += 2 * P
            g += P
    elif rot_mode == ROT_FULL:
        R = hadamard(D)
    else:
        R = np.eye(D)
    return R


# ----------------------------------------------------------------------------------
# Quantisers (L190; readings 10, 11) and nibble packing
# ----------------------------------------------------------------------------------
def _quant_sym7(y, amax):
    """scale = rn(amax/7); inv = rn(7/amax) (0 if amax==0); code = clamp(rne(rn(y*inv)),-7,7).
    All fp32.  amax broadcasts against y."""
    amax = amax.astype(F32)
    scale = (amax / F32(7.0)).astype(F32)
    with np.errstate(divide='ignore'):
        inv = np.where(amax > 0, (F32(7.0) / amax).astype(F32), F32(0.0)).astype(F32)
    q = np.rint((y.astype(F32) * inv).astype(F32))
    codes = np.clip(q, -7, 7).astype(np.int8)
    return codes, scale


def quant_qk(y, qk_group=1):
    """Per-token symmetric INT4 of rotated Q or K (L190 "per-token quantization for Q and K").
    y fp32 [N,D] -> codes int8 [N,D] in [-7,7], scales fp32 [ceil(N/qk_group)]."""
    N, D = y.shape
    if qk_group == 1:
        amax = np.abs(y).max(axis=1)
        codes, scale = _quant_sym7(y, amax[:, None])
        return codes, scale[:, 0]
    ng = -(-N // qk_group)
    codes = np.empty((N, D), dtype=np.int8)
    scales = np.empty(ng, dtype=F32)
    for g in range(ng):
        sl = slice(g * qk_group, min(N, (g + 1) * qk_group))
        amax = np.abs(y[sl]).max()
        c, s = _quant_sym7(y[sl], np.full((1, 1), amax, dtype=F32))
        codes[sl] = c
        scales[g] = s[0, 0]
    return codes, scales


def quant_v(v16, v_group=128, v_scale=VSCALE_CHANNEL, mean=None):
    """Per-group INT4 of Hadamard-domain V (L190 "per-group quantization for V"): one scale per
    (group of v_group consecutive tokens, channel); ragged last group uses the tokens that exist.
    v_scale = VSCALE_GROUP: one scale per group (amax over the group's tokens AND channels).
    mean (smoothing, fp32 [D]): v - mean is quantised (one fp32 subtraction per element).
    v16 fp16 [N,D] -> codes int8 [N,D], scales fp32 [ceil(N/v_group), D]  (VSCALE_GROUP: [ceil(N/v_group)])."""
    N, D = v16.shape
    v = v16.astype(F32)
    if mean is not None:
        v = (v - np.asarray(mean, dtype=F32)[None, :]).astype(F32)
    ng = -(-N // v_group)
    codes = np.empty((N, D), dtype=np.int8)
    scales = np.empty((ng, D) if v_scale == VSCALE_CHANNEL else (ng,), dtype=F32)
    for g in range(ng):
        sl = slice(g * v_group, min(N, (g + 1) * v_group))
        if v_scale == VSCALE_CHANNEL:
            amax = np.abs(v[sl]).max(axis=0)
            c, s = _quant_sym7(v[sl], amax[None, :])
            scales[g] = s[0]
        else:
            amax = np.abs(v[sl]).max()
            c, s = _quant_sym7(v[sl], np.full((1, 1), amax, dtype=F32))
            scales[g] = s[0, 0]
        codes[sl] = c
    return codes, scales


# ----------------------------------------------------------------------------------
# Smoothing (L90 "we first perform smoothing on Q, K, V"; L40 Q - E[Q]; L52): SURVEY 8f row f2
# ----------------------------------------------------------------------------------
FIX_QK = 2.0 ** 20      # fixed-point unit of the column sums of y_Q, y_K
FIX_V = 2.0 ** 24       # fp16 V is a multiple of 2^-24, so its fixed-point sum is exact


def column_mean_fixed(x32, unit):
    """Token mean of every channel, defined through a fixed-point sum so that it does not depend on the order of
    summation (the GPU adds in parallel):  mean = fl32( fp64(sum_n rne(x_n * unit)) / (N * unit) ).
    x32 fp32 [N,D] -> fp32 [D]."""
    x32 = np.asarray(x32, dtype=F32)
    fx = np.rint((x32 * F32(unit)).astype(F32).astype(F64)).astype(np.int64)
    tot = fx.sum(axis=0)                                   # exact integer sums
    return (tot.astype(F64) / (F64(x32.shape[0]) * F64(unit))).astype(F32)


def smooth_means(p: Params, q16, k16, v16, coef, rot=None):
    """Column means of y_Q, y_K (after RoPE and rotation, the tensors that are quantised) and of V."""
    yq = apply_rope_rot(p, q16, coef, rot)
    yk = apply_rope_rot(p, k16, coef, rot)
    return (column_mean_fixed(yq, FIX_QK), column_mean_fixed(yk, FIX_QK),
            column_mean_fixed(v16.astype(F32), FIX_V))


def pack_nibbles(codes):
    """byte d/2 = (code_{2i} & 0xF) | ((code_{2i+1} & 0xF) << 4); two's-complement nibbles."""
    c = codes.astype(np.int16)
    lo = c[..., 0::2] & 0xF
    hi = c[..., 1::2] & 0xF
    return (lo | (hi << 4)).astype(np.uint8)


def unpack_nibbles(packed):
    b = packed.astype(np.int16)
    lo = b & 0xF
    hi = (b >> 4) & 0xF
    lo = np.where(lo >= 8, lo - 16, lo)
    hi = np.where(hi >= 8, hi - 16, hi)
    out = np.empty(packed.shape[:-1] + (packed.shape[-1] * 2,), dtype=np.int8)
    out[..., 0::2] = lo
    out[..., 1::2] = hi
    return out


# ----------------------------------------------------------------------------------
# Prologue = steps a1-a3 for one head
# ----------------------------------------------------------------------------------
def prepare_qk_head(p: Params, q16, k16, coef, rot=None, means=None):
    """One head: RoPE o R in fp32 then per-token INT4.  Returns dict with y (fp32), fp16 copy,
    codes, packed codes, scales for Q and K.
    means = (mean_q, mean_k) (smoothing): y - mean is quantised (one fp32 subtraction per element); k_corr[j] =
    mean_q . (y_K[j] - mean_k) is the rank-1 term that fwd adds back to S (exact: (Q' + 1 mean_q^T) K'^T)."""
    out = {}
    for name, x in (('q', q16), ('k', k16)):
        y = apply_rope_rot(p, x, coef, rot)
        out[name + '_16'] = y.astype(np.float16)            # the FP16 path is never smoothed
        if means is not None:
            y = (y - np.asarray(means[0 if name == 'q' else 1], dtype=F32)[None, :]).astype(F32)
        codes, scale = quant_qk(y, p.qk_group)
        out[name + '_y'] = y
        out[name + '_codes'] = codes
        out[name + '_packed'] = pack_nibbles(codes)
        out[name + '_scale'] = scale
    if means is not None:
        out['k_corr'] = out['k_y'].astype(F64) @ np.asarray(means[0], dtype=F64)
    return out


# ----------------------------------------------------------------------------------
# Attention oracles
# ----------------------------------------------------------------------------------
def o_exact(q_r, k_r, v, rows=None):
    """O* = softmax(Q_r K_r^T / sqrt(D)) V in fp64 — the plain definition (Eq.14).
    rows: optional query-row indices (rows are independent).  Returns fp64 [len(rows), D]."""
    q = np.asarray(q_r, dtype=F64)
    k = np.asarray(k_r, dtype=F64)
    vv = np.asarray(v, dtype=F64)
    if rows is not None:
        q = q[rows]
    D = q.shape[1]
    s = (q @ k.T) / math.sqrt(D)
    s -= s.max(axis=1, keepdims=True)
    e = np.exp(s)
    return (e @ vv) / e.sum(axis=1, keepdims=True)


def p_codes_block(s_blk, m_ref, p_mode):
    """Eq.12 (L166-168): P~ = P/max(P) * 15 - 8 in (-8,7]; returned as unsigned u = c + 8 in {0..15}
    (reading 15).  Eq.11 (L161): * 7 in (0,7].  Round half to even (reading 14).
    s_blk [R, J]; m_ref [R] is the normaliser's exponent (block row max, or running max)."""
    phat = np.exp(s_blk - m_ref[:, None])
    levels = 15.0 if p_mode == P_ASYM15 else 7.0
    u = np.rint(levels * phat)
    return phat, u


def o_quant(p: Params, qc, qs, kc, ks, vc, vs, rows=None, dump=False, quantize=True,
            p_mode=None, p_norm=None, k_corr=None, v_mean=None, dump_pv=False):
    """Steps 7-12 for one head, fp64 softmax arithmetic.
    qc,kc,vc: int8 codes [N,D]; qs,ks: fp32 scales [ceil(N/qk_group)]; vs: fp32 [nG, D].
    rows: query rows to evaluate (default all).  quantize=False switches every quantiser of the
    attention stage off (P^ used unrounded) for the brute-force pin.
    Returns O fp64 [R,D] (and, with dump=True, the int32 S accumulators and the P codes)."""
    p_mode = p.p_mode if p_mode is None else p_mode
    p_norm = p.p_norm if p_norm is None else p_norm
    N, D = kc.shape
    rows = np.arange(qc.shape[0]) if rows is None else np.asarray(rows)
    Rn = len(rows)
    qg = rows // p.qk_group
    q = qc[rows].astype(F64)
    qscale = qs.astype(F64)[qg]
    kscale = ks.astype(F64)[np.arange(N) // p.qk_group]
    levels = 15.0 if p_mode == P_ASYM15 else 7.0
    # step 7: integer scores; fp64 BLAS on integer-valued codes is exact (|acc| <= 49 D << 2^53)
    acc = q @ kc.astype(F64).T                         # [R, N] integers
    s = acc * qscale[:, None] * kscale[None, :] / math.sqrt(D)
    if k_corr is not None:      # smoothing: rank-1 correction mean(Q) K'^T added to S in floating point
        s = s + np.asarray(k_corr, dtype=F64)[None, :] / math.sqrt(D)
    pv_dump = [] if dump_pv else None
    m = np.full(Rn, -np.inf)
    l = np.zeros(Rn)
    O = np.zeros((Rn, D))
    codes_dump = np.zeros((Rn, N), dtype=np.int16) if dump else None
    nblk = -(-N // p.kv_block)
    for J in range(nblk):
        j0, j1 = J * p.kv_block, min(N, (J + 1) * p.kv_block)
        sb = s[:, j0:j1]
        mt = sb.max(axis=1)                            # step 8: block row max (keys < N only)
        m_new = np.maximum(m, mt)                      # step 11 (L157 running max)
        if p_norm == NORM_ROWBLOCK:
            phat, u = p_codes_block(sb, mt, p_mode)    # step 9
            beta = np.exp(mt - m_new)
        else:
            phat, u = p_codes_block(sb, m_new, p_mode)
            beta = np.ones(Rn)
        alpha = np.exp(m - m_new)                      # exp(-inf) = 0 on the first block
        vblk = vc[j0:j1].astype(F64)
        g = j0 // p.v_group
        vscale = np.broadcast_to(np.asarray(vs[g], dtype=F64), (vc.shape[1],))      # [D] (one value repeated for VSCALE_GROUP)
        if quantize:
            pv = u @ vblk                              # step 10, unsigned form
            # signed form with zero-point -8 (L166): sum (u-8) v + 8 sum v — must be the same integer
            pv_signed = (u - 8.0) @ vblk + 8.0 * vblk.sum(axis=0)[None, :]
            assert np.array_equal(pv, pv_signed), "zero-point identity violated"
            contrib = pv * (vscale / levels)[None, :]
            if dump_pv:
                pv_dump.append(pv.astype(np.int64))
        else:
            contrib = phat @ (vblk * vscale[None, :])
        l = alpha * l + beta * phat.sum(axis=1)        # un-rounded P^ (reading 16)
        O = alpha[:, None] * O + beta[:, None] * contrib
        m = m_new
        if dump:
            codes_dump[:, j0:j1] = u.astype(np.int16)
    O = O / l[:, None]                                 # step 12
    if v_mean is not None:      # smoothing: softmax(.)(V - 1 mean^T) + mean^T = softmax(.) V
        O = O + np.asarray(v_mean, dtype=F64)[None, :]
    if dump_pv:
        return O, acc.astype(np.int32), codes_dump, np.stack(pv_dump)
    if dump:
        return O, acc.astype(np.int32), codes_dump
    return O


def int_matmul_loops(a, b):
    """int64 triple loop a[R,K] x b[J,K]^T for the tiny-input pin of the BLAS shortcut."""
    R, K = a.shape
    J = b.shape[0]
    out = np.zeros((R, J), dtype=np.int64)
    for i in range(R):
        for j in range(J):
            acc = 0
            for d in range(K):
                acc += int(a[i, d]) * int(b[j, d])
            out[i, j] = acc
    return out


# ----------------------------------------------------------------------------------
# Incoherence (Eq.1-2) and fallback policy (L192)
# ----------------------------------------------------------------------------------
def incoherence(x):
    """Psi(X) = max_i |X_i,: - E[X]| per channel (Eq.2) with E[X] the token mean (Eq.1)."""
    x = np.asarray(x, dtype=F64)
    return np.abs(x - x.mean(axis=0, keepdims=True)).max(axis=0)


@dataclass
class Policy:
    """FP16 on the first/last sampling steps and first/last DiT blocks, INT4 elsewhere (L192)."""
    n_steps: int
    n_blocks: int
    first_steps: int
    last_steps: int
    first_blocks: int
    last_blocks: int
    fp16_head_mask: tuple = field(default_factory=tuple)

    def select(self, step, block, head=0):
        """0 = INT4, 1 = FP16."""
        if step < self.first_steps or step >= self.n_steps - self.last_steps:
            return 1
        if block < self.first_blocks or block >= self.n_blocks - self.last_blocks:
            return 1
        if self.fp16_head_mask and self.fp16_head_mask[head]:
            return 1
        return 0

    def int4_fraction(self):
        n = sum(1 - self.select(s, b) for s in range(self.n_steps) for b in range(self.n_blocks))
        return n / (self.n_steps * self.n_blocks)


# ----------------------------------------------------------------------------------
# Full pipeline for one head (used by tests / bench cpu_baseline)
# ----------------------------------------------------------------------------------
def int4_attention_head(p: Params, q16, k16, v16, rot=None, rows=None, dump=False, coef=None):
    """prologue + o_quant for one head from fp16 inputs (V already in the Hadamard domain)."""
    coef = coef_table(p, rot) if coef is None else coef
    means = smooth_means(p, q16, k16, v16, coef, rot) if p.smooth else None
    pq = prepare_qk_head(p, q16, k16, coef, rot, means=None if means is None else means[:2])
    vc, vs = quant_v(v16, p.v_group, p.v_scale, mean=None if means is None else means[2])
    res = o_quant(p, pq['q_codes'], pq['q_scale'], pq['k_codes'], pq['k_scale'], vc, vs,
                  rows=rows, dump=dump, k_corr=pq.get('k_corr'), v_mean=None if means is None else means[2])
    pq['means'] = means
    return res, pq, (vc, vs)
