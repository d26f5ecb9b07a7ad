// Prologue kernels (HBM-bound): prepare_qk (a1+a2), quant_v (a3), the smoothing pre-pass (f2) and the unpack helpers.
// Code-producing arithmetic is fp32 with one rounding per operation (__fmul_rn/__fadd_rn/__fsub_rn/__fdiv_rn,
// never contracted) so that the INT4 codes are reproducible bit for bit ("bit-exact prologue").
#include "tc_common.cuh"     // packed fp32x2 arithmetic (mul.rn / add.rn per lane: the same roundings as the scalar forms)

namespace rotattn {

// ------------------------------------------------------------------------------------------------
// prepare_qk: one warp per token; lane l owns channels [CPL*l, CPL*l+CPL) of Q and of K.
// ------------------------------------------------------------------------------------------------
struct PrepArgs {
  const __half* X[2];     // Q, K  [BH*N, D]
  uint8_t* X4[2];         // packed codes [BH*N, D/2]
  float* Xs[2];           // scales [BH*N]  (qk_group = 128: [BH*nG])
  __half* X16[2];         // optional fp16 y
  int8_t* X8[2];          // optional operand bytes [BH*N, 128]
  float* KsP;             // optional: key scales padded to [BH, npad] (per-token mode)
  const float4* coef;     // table rows
  const float4* rot;      // [D/2] blocks or nullptr (H_2)
  long long* sums;        // smoothing: int64 [BH,3,D] fixed-point column sums (stats pass: accumulated; apply pass: unused)
  const float* means;     // smoothing: float [BH,3,D] column means (apply pass)
  float* KcP;             // smoothing: per-key correction, padded [BH, npad]
  float kc_scale;         // log2(e) / sqrt(D)
  int N, n_rope, gt, gh, gw, Pt, Ph, Pw, npad, nG;
};

// Widened MMA operand byte of a code c in [-7,7] (or a P code in [0,15]): sign-magnitude, which is the E4M3
// encoding of c * 2^-9 (E4M3 subnormals are m * 2^-9, and bytes 8..15 are the first normal binade 2^-6 * (1 + m/8)),
// so tcgen05 kind::f8f6f4 multiplies and accumulates the integer codes exactly, scaled by 2^-18, in fp32.
__device__ __forceinline__ uint32_t code_byte(int c) { return (uint32_t)(abs(c) | ((c >> 24) & 0x80)); }

constexpr int kPrepTok = 4;       // tokens per warp iteration: all their loads are issued before any arithmetic (bytes in flight)
constexpr int kPrepWarps = 8;
constexpr float kFixQK = 1048576.f;      // smoothing: y_Q, y_K column sums in fixed point, units of 2^-20 (order-independent, exact)
constexpr float kFixV = 16777216.f;      // smoothing: fp16 V is a multiple of 2^-24: its fixed-point sum is exact

enum { PREP_QUANT = 0, PREP_STATS = 1, PREP_QUANT_SMOOTH = 2 };

// per-lane constants of the RoPE table walk and of the HALF pairing
template <int D, int ROT>
struct PrepLane {
  static constexpr int CPL = D / 32, PPL = CPL / 2;
  int cbase[PPL], cstride[PPL], caxis[PPL];
  int partner[CPL];
  float ca[CPL], cb[CPL];
  __device__ __forceinline__ void init(const PrepArgs& a, int lane) {
    const int secbase[3] = {0, (a.gt + 1) * a.Pt, (a.gt + 1) * a.Pt + (a.gh + 1) * a.Ph};
#pragma unroll
    for (int i = 0; i < PPL; ++i) {
      int g = lane * PPL + i;
      int ax = g < a.Pt ? 0 : (g < a.Pt + a.Ph ? 1 : 2);
      int k = g - (ax == 0 ? 0 : (ax == 1 ? a.Pt : a.Pt + a.Ph));
      int P = ax == 0 ? a.Pt : (ax == 1 ? a.Ph : a.Pw);
      caxis[i] = ax; cbase[i] = secbase[ax] + k; cstride[i] = P;
    }
    if (ROT == ROTATTN_ROT_HALF) {
#pragma unroll
      for (int j = 0; j < CPL; ++j) {
        int c = lane * CPL + j;
        int sec = c < 2 * a.Pt ? 0 : (c < 2 * (a.Pt + a.Ph) ? 1 : 2);
        int o = sec == 0 ? 0 : (sec == 1 ? 2 * a.Pt : 2 * (a.Pt + a.Ph));
        int P = sec == 0 ? a.Pt : (sec == 1 ? a.Ph : a.Pw);
        int goff = o / 2;
        int i = c - o;
        bool role_u = i < P;
        int blk = goff + (role_u ? i : i - P);
        partner[j] = role_u ? c + P : c - P;
        float4 r = a.rot ? a.rot[blk] : make_float4(0.70710678118654752440f, 0.70710678118654752440f,
                                                    0.70710678118654752440f, -0.70710678118654752440f);
        // u' = u r00 + v r10 (this lane holds u), v' = u r01 + v r11 (this lane holds v): own value times ca + partner times cb
        ca[j] = role_u ? r.x : r.w;
        cb[j] = role_u ? r.z : r.y;
      }
    }
  }
};

// Sum of two packed products with one rounding per operation: ptxas contracts mul.rn.f32x2 + add.rn.f32x2 into one FFMA2
// (a single rounding, which would change codes at rounding ties), but it never contracts the scalar add.rn.f32, so the
// products are packed and the additions scalar.
__device__ __forceinline__ float2 add2_rn(float2 a, float2 b) { return make_float2(__fadd_rn(a.x, b.x), __fadd_rn(a.y, b.y)); }

// (t,h,w) of a token index walked with a constant stride: two 32-bit divisions once, then additions with carries
// (the stride is decomposed once; every component of it is smaller than its axis, so one carry per axis suffices).
struct PosWalk {
  int pt, ph, pw, st, sh, sw;
  __device__ __forceinline__ void init(int n0, int stride, int gh, int gw) {
    pw = n0 % gw; int pr = n0 / gw; ph = pr % gh; pt = pr / gh;
    sw = stride % gw; int sr = stride / gw; sh = sr % gh; st = sr / gh;
  }
  __device__ __forceinline__ void advance(int gh, int gw) {
    pw += sw;
    int c = pw >= gw; pw -= c ? gw : 0;
    ph += sh + c;
    c = ph >= gh; ph -= c ? gh : 0;
    pt += st + c;
  }
};

// y = x (M R) for kPrepTok consecutive tokens of one head (Q and K): RoPE through the coefficient table (INTERLEAVED is
// merged into it, Eq.7), then HALF (Eq.8, partner exchange through shared memory) or FULL (the paper's
// "Full" baseline L208: D x D Hadamard as an in-register / shuffle butterfly) in the same register pass.
template <int D, int ROT>
__device__ __forceinline__ void prep_compute_y(const PrepArgs& a, const PrepLane<D, ROT>& ln, float* ybuf_warp, long long head0,
                                               int n0, int pt, int ph, int pw, int lane, __half (&hx)[kPrepTok][2][D / 32],
                                               float (&y)[kPrepTok][2][D / 32]) {
  constexpr int CPL = D / 32, PPL = CPL / 2, TOK = kPrepTok;
  // (pt, ph, pw) = (t,h,w) of token n0 (row-major, reading 4); the following tokens by carry propagation
  // ---- load phase: TOK tokens x (Q, K) + their coefficient rows, all independent
  float4 A[TOK][PPL];
  const bool full = n0 + TOK <= a.N;                     // warp-uniform: no per-token guards on the common path
  const __half* src0 = a.X[0] + (head0 + n0) * D + lane * CPL;
  const __half* src1 = a.X[1] + (head0 + n0) * D + lane * CPL;
#pragma unroll
  for (int t = 0; t < TOK; ++t) {
    const int n = n0 + t;
    if (full || n < a.N) {
      if (CPL == 4) {
        *reinterpret_cast<uint2*>(hx[t][0]) = __ldcs(reinterpret_cast<const uint2*>(src0 + t * D));
        *reinterpret_cast<uint2*>(hx[t][1]) = __ldcs(reinterpret_cast<const uint2*>(src1 + t * D));
      } else {
        *reinterpret_cast<uint32_t*>(hx[t][0]) = __ldcs(reinterpret_cast<const uint32_t*>(src0 + t * D));
        *reinterpret_cast<uint32_t*>(hx[t][1]) = __ldcs(reinterpret_cast<const uint32_t*>(src1 + t * D));
      }
      const bool rope = n < a.n_rope;                    // text tokens use the no-RoPE rows of the table
      const int p0 = rope ? pt : a.gt, p1 = rope ? ph : a.gh, p2 = rope ? pw : a.gw;
#pragma unroll
      for (int i = 0; i < PPL; ++i) {
        const int pos = ln.caxis[i] == 0 ? p0 : (ln.caxis[i] == 1 ? p1 : p2);
        A[t][i] = __ldg(a.coef + ln.cbase[i] + pos * ln.cstride[i]);
      }
    } else {
#pragma unroll
      for (int m = 0; m < 2; ++m)
#pragma unroll
        for (int j = 0; j < CPL; ++j) hx[t][m][j] = __float2half_rn(0.f);
#pragma unroll
      for (int i = 0; i < PPL; ++i) A[t][i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    if (++pw == a.gw) { pw = 0; if (++ph == a.gh) { ph = 0; ++pt; } }
  }
  // ---- RoPE (merged with the interleaved rotation through the table)
#pragma unroll
  for (int t = 0; t < TOK; ++t)
#pragma unroll
    for (int m = 0; m < 2; ++m)
#pragma unroll
      for (int i = 0; i < PPL; ++i) {
        const float x0 = __half2float(hx[t][m][2 * i]), x1 = __half2float(hx[t][m][2 * i + 1]);
        // (y0, y1) = x0 (a, b) + x1 (c, d): two packed multiplies and two adds, every operation rounded once
        const float2 r = add2_rn(fmul2(make_float2(x0, x0), make_float2(A[t][i].x, A[t][i].y)),
                                 fmul2(make_float2(x1, x1), make_float2(A[t][i].z, A[t][i].w)));
        y[t][m][2 * i] = r.x;
        y[t][m][2 * i + 1] = r.y;
      }
  if (ROT == ROTATTN_ROT_HALF) {
    float (*yb)[2][D] = reinterpret_cast<float (*)[2][D]>(ybuf_warp);
#pragma unroll
    for (int t = 0; t < TOK; ++t)
#pragma unroll
      for (int m = 0; m < 2; ++m) {
        if (CPL == 4) *reinterpret_cast<float4*>(&yb[t][m][lane * CPL]) = make_float4(y[t][m][0], y[t][m][1], y[t][m][2], y[t][m][3]);
        else *reinterpret_cast<float2*>(&yb[t][m][lane * CPL]) = make_float2(y[t][m][0], y[t][m][1]);
      }
    __syncwarp();
#pragma unroll
    for (int t = 0; t < TOK; ++t)
#pragma unroll
      for (int m = 0; m < 2; ++m)
#pragma unroll
        for (int j = 0; j < CPL; j += 2) {
          const float2 other = make_float2(yb[t][m][ln.partner[j]], yb[t][m][ln.partner[j + 1]]);
          const float2 r = add2_rn(fmul2(make_float2(y[t][m][j], y[t][m][j + 1]), make_float2(ln.ca[j], ln.ca[j + 1])),
                                   fmul2(other, make_float2(ln.cb[j], ln.cb[j + 1])));             // fp32 addition commutes exactly
          y[t][m][j] = r.x;
          y[t][m][j + 1] = r.y;
        }
    __syncwarp();
  }
  if (ROT == ROTATTN_ROT_FULL) {
    // Sylvester butterfly, strides 1, 2, ..., D/2 in this order: (a, b) -> (a + b, a - b) with a the lower channel; then
    // one multiplication by fl(1/sqrt(D)).  One rounding per operation: the oracle follows the same order bit for bit.
    constexpr float kNorm = D == 128 ? 0.08838834764831845f : 0.125f;
#pragma unroll
    for (int t = 0; t < TOK; ++t)
#pragma unroll
      for (int m = 0; m < 2; ++m) {
        float* v = y[t][m];
#pragma unroll
        for (int s = 1; s < CPL; s <<= 1)
#pragma unroll
          for (int j = 0; j < CPL; ++j)
            if (!(j & s)) { const float p = v[j], q = v[j + s]; v[j] = __fadd_rn(p, q); v[j + s] = __fsub_rn(p, q); }
#pragma unroll
        for (int s = 1; s < 32; s <<= 1)
#pragma unroll
          for (int j = 0; j < CPL; ++j) {
            const float other = __shfl_xor_sync(0xffffffffu, v[j], s);
            v[j] = (lane & s) ? __fsub_rn(other, v[j]) : __fadd_rn(v[j], other);
          }
#pragma unroll
        for (int j = 0; j < CPL; ++j) v[j] = __fmul_rn(v[j], kNorm);
      }
  }
}

// quantise with inv = rn(7 / amax) and store the packed codes, the operand bytes and the optional fp16 copy of one token
template <int D>
__device__ __forceinline__ void prep_store_token(const PrepArgs& a, int m, long long tok, int lane, const float (&yq)[D / 32],
                                                 float inv) {
  constexpr int CPL = D / 32;
  // code = rne(y * inv) is in [-7,7] without clamping (|y| <= amax and inv = rn(7/amax) give |y*inv| < 7.5).
  // fs = q + 1.5*2^23 holds the two's-complement code in its low byte.
  if (CPL == 4) {
    const float2 inv2 = make_float2(inv, inv), magic2 = make_float2(12582912.f, 12582912.f);
    const float2 f01 = add2_rn(fmul2(make_float2(yq[0], yq[1]), inv2), magic2);
    const float2 f23 = add2_rn(fmul2(make_float2(yq[2], yq[3]), inv2), magic2);
    // w = the four codes as two's-complement bytes
    const uint32_t w = __byte_perm(__byte_perm(__float_as_uint(f01.x), __float_as_uint(f01.y), 0x0040),
                                   __byte_perm(__float_as_uint(f23.x), __float_as_uint(f23.y), 0x0040), 0x5410);
    // packed nibbles: byte 0 = (c0 & 0xF) | (c1 & 0xF) << 4, byte 2 = the same of (c2, c3)
    const uint32_t nib = (w & 0x000F000Fu) | ((w >> 4) & 0x00F000F0u);
    *reinterpret_cast<uint16_t*>(a.X4[m] + tok * (D / 2) + lane * 2) = (uint16_t)__byte_perm(nib, nib, 0x0020);
    if (a.X8[m]) {
      // sign-magnitude operand bytes (code_byte): per byte |c| = (c ^ s) + t with t = the sign bit and s = 0xFF t
      // (|c| <= 7: no carry leaves a byte); a zero code has no sign bit, so there is no -0 byte.
      const uint32_t t = (w >> 7) & 0x01010101u;
      const uint32_t mag = (w ^ (t * 0xFFu)) + t;
      *reinterpret_cast<uint32_t*>(a.X8[m] + tok * kQKRowBytes + lane * 4) = mag | (w & 0x80808080u);
    }
  } else {
    uint32_t fs[CPL], fa[CPL], yb[CPL];
#pragma unroll
    for (int j = 0; j < CPL; ++j) {
      const float q = __fmul_rn(yq[j], inv);
      fs[j] = __float_as_uint(__fadd_rn(q, 12582912.f));
      fa[j] = __float_as_uint(__fadd_rn(fabsf(q), 12582912.f));       // |q| + 1.5*2^23: the magnitude in the low byte
      yb[j] = __float_as_uint(q);
    }
    a.X4[m][tok * (D / 2) + lane] = (uint8_t)((fs[0] & 0xFu) | ((fs[1] << 4) & 0xF0u));
    if (a.X8[m]) {
      // magnitude bytes | sign bits of q, the sign only where the magnitude byte is non-zero (no -0 byte)
      int8_t* dst = a.X8[m] + tok * kQKRowBytes;
      const uint32_t mag = __byte_perm(fa[0], fa[1], 0x0040) & 0xFFFFu;
      const uint32_t sgn = __byte_perm(yb[0], yb[1], 0x0073) & 0xFFFFu;
      const uint32_t nz = ((mag + 0x7F7Fu) & 0x8080u);
      *reinterpret_cast<uint16_t*>(dst + lane * 2) = (uint16_t)(mag | (sgn & nz));
      *reinterpret_cast<uint16_t*>(dst + 64 + lane * 2) = 0;      // zero pad to a 128-byte row
    }
  }
}

template <int D>
__device__ __forceinline__ void prep_store_fp16(const PrepArgs& a, int m, long long tok, int lane, const float (&yq)[D / 32]) {
  constexpr int CPL = D / 32;
  __half* dst = a.X16[m] + tok * D + lane * CPL;
  alignas(8) __half hy[CPL];
#pragma unroll
  for (int j = 0; j < CPL; ++j) hy[j] = __float2half_rn(yq[j]);
  if (CPL == 4) *reinterpret_cast<uint2*>(dst) = *reinterpret_cast<uint2*>(hy);
  else *reinterpret_cast<uint32_t*>(dst) = *reinterpret_cast<uint32_t*>(hy);
}

// QKG = 1: per-token scales, warps stride over token chunks.  QKG = 128: one CTA per 128-token group, two passes over the
// group (amax, then quantise; the second pass re-reads its 64 KB from L1/L2).  MODE: PREP_QUANT, PREP_STATS (smoothing
// pre-pass: fixed-point column sums of y only) or PREP_QUANT_SMOOTH (y - column mean is what gets quantised).
template <int D, int ROT, int QKG, int MODE>
__global__ void __launch_bounds__(256, 2) prepare_qk_kernel(const PrepArgs a) {
  constexpr int CPL = D / 32;       // channels per lane
  constexpr int WPB = kPrepWarps;   // warps per block
  constexpr int TOK = kPrepTok;
  __shared__ float ybuf[ROT == ROTATTN_ROT_HALF ? WPB : 1][TOK][2][D];   // HALF-rotation exchange buffer
  __shared__ float gmax[WPB][2];
  __shared__ unsigned long long ssum[MODE == PREP_STATS ? 2 * D : 1];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  PrepLane<D, ROT> ln;
  ln.init(a, lane);
  const long long bh = blockIdx.y;
  const long long head0 = bh * a.N;
  alignas(8) __half hx[TOK][2][CPL];
  float y[TOK][2][CPL];
  float mu[2][CPL];
  if (MODE == PREP_QUANT_SMOOTH) {
#pragma unroll
    for (int m = 0; m < 2; ++m)
#pragma unroll
      for (int j = 0; j < CPL; ++j) mu[m][j] = a.means[(bh * 3 + m) * D + lane * CPL + j];
  }

  if (MODE == PREP_STATS) {
    long long acc[2][CPL];
#pragma unroll
    for (int m = 0; m < 2; ++m)
#pragma unroll
      for (int j = 0; j < CPL; ++j) acc[m][j] = 0;
    for (int i = threadIdx.x; i < 2 * D; i += blockDim.x) ssum[i] = 0;
    __syncthreads();
    const int nstride = gridDim.x * WPB * TOK;
    PosWalk pos;
    pos.init((blockIdx.x * WPB + warp) * TOK, nstride, a.gh, a.gw);
    for (int n0 = (blockIdx.x * WPB + warp) * TOK; n0 < a.N; n0 += nstride, pos.advance(a.gh, a.gw)) {
      prep_compute_y<D, ROT>(a, ln, &ybuf[ROT == ROTATTN_ROT_HALF ? warp : 0][0][0][0], head0, n0, pos.pt, pos.ph, pos.pw, lane, hx, y);
#pragma unroll
      for (int t = 0; t < TOK; ++t)
        if (n0 + t < a.N) {
#pragma unroll
          for (int m = 0; m < 2; ++m)
#pragma unroll
            for (int j = 0; j < CPL; ++j) acc[m][j] += __float2ll_rn(__fmul_rn(y[t][m][j], kFixQK));
        }
    }
#pragma unroll
    for (int m = 0; m < 2; ++m)
#pragma unroll
      for (int j = 0; j < CPL; ++j) atomicAdd(&ssum[m * D + lane * CPL + j], (unsigned long long)acc[m][j]);
    __syncthreads();
    for (int i = threadIdx.x; i < 2 * D; i += blockDim.x)
      atomicAdd(reinterpret_cast<unsigned long long*>(a.sums) + bh * 3 * D + i, ssum[i]);
    return;
  }

  auto smooth_and_corr = [&](int n0) {
    // y' = y - mean (one rounding); per key the correction c_j = mean(Q) . K'_j, stored in the log2 domain
    if (MODE == PREP_QUANT_SMOOTH) {
#pragma unroll
      for (int t = 0; t < TOK; ++t) {
#pragma unroll
        for (int m = 0; m < 2; ++m)
#pragma unroll
          for (int j = 0; j < CPL; ++j) y[t][m][j] = __fsub_rn(y[t][m][j], mu[m][j]);
        float c = 0.f;
#pragma unroll
        for (int j = 0; j < CPL; ++j) c = fmaf(mu[0][j], y[t][1][j], c);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
        if (lane == 0 && n0 + t < a.N && a.KcP) a.KcP[bh * a.npad + n0 + t] = c * a.kc_scale;
      }
    }
  };

  if (QKG == 1) {
    // padded tail of the workspace copies [BH, npad] (read block-wise by fwd_int4's bulk copies): scale 1, correction 0
    if (blockIdx.x == 0 && warp == 0) {
      for (int n = a.N + lane; n < a.npad; n += 32) {
        if (a.KsP) a.KsP[bh * a.npad + n] = 1.f;
        if (MODE == PREP_QUANT_SMOOTH && a.KcP) a.KcP[bh * a.npad + n] = 0.f;
      }
    }
    // blockIdx.y = (b,h); the warps of the grid's x dimension stride over that head's tokens, TOK consecutive ones at a time
    const int nstride = gridDim.x * WPB * TOK;
    PosWalk pos;
    pos.init((blockIdx.x * WPB + warp) * TOK, nstride, a.gh, a.gw);
    for (int n0 = (blockIdx.x * WPB + warp) * TOK; n0 < a.N; n0 += nstride, pos.advance(a.gh, a.gw)) {
      prep_compute_y<D, ROT>(a, ln, &ybuf[ROT == ROTATTN_ROT_HALF ? warp : 0][0][0][0], head0, n0, pos.pt, pos.ph, pos.pw, lane, hx, y);
      if (a.X16[0]) {                                     // fp16 copies for the FP16 path: y before smoothing
#pragma unroll
        for (int t = 0; t < TOK; ++t)
          if (n0 + t < a.N) {
            prep_store_fp16<D>(a, 0, head0 + n0 + t, lane, y[t][0]);
            prep_store_fp16<D>(a, 1, head0 + n0 + t, lane, y[t][1]);
          }
      }
      smooth_and_corr(n0);
      // ---- per-token amax (all TOK x 2 reductions interleaved), quantise, store
      float amax[TOK][2];
#pragma unroll
      for (int t = 0; t < TOK; ++t)
#pragma unroll
        for (int m = 0; m < 2; ++m) {
          float v = 0.f;
#pragma unroll
          for (int j = 0; j < CPL; ++j) v = fmaxf(v, fabsf(y[t][m][j]));
          amax[t][m] = v;
        }
      // Reduction of the TOK x 2 = 8 maxima over the 32 lanes with 9 shuffles instead of 40: at offsets 16, 8, 4 every lane
      // keeps the half of its values that belongs to its side of the exchange and sends the other half, so that lanes
      // [4 i, 4 i + 4) end up with the maximum of value i = 2 t + m (max is exact: the result is the same bit pattern).
      static_assert(TOK == 4, "the transposing reduction is written for 8 values");
      float z;
      {
        const bool h16 = lane & 16, h8 = lane & 8, h4 = lane & 4;
        float w4[4], w2[2];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const float lo = amax[k >> 1][k & 1], hi = amax[(k + 4) >> 1][(k + 4) & 1];
          w4[k] = fmaxf(h16 ? hi : lo, __shfl_xor_sync(0xffffffffu, h16 ? lo : hi, 16));
        }
#pragma unroll
        for (int k = 0; k < 2; ++k) w2[k] = fmaxf(h8 ? w4[k + 2] : w4[k], __shfl_xor_sync(0xffffffffu, h8 ? w4[k] : w4[k + 2], 8));
        z = fmaxf(h4 ? w2[1] : w2[0], __shfl_xor_sync(0xffffffffu, h4 ? w2[0] : w2[1], 4));
        z = fmaxf(z, __shfl_xor_sync(0xffffffffu, z, 2));
        z = fmaxf(z, __shfl_xor_sync(0xffffffffu, z, 1));
      }
      // scale = amax / 7 and inv = 7 / amax are IEEE divisions, computed by the lanes that hold the value (lane >> 2 = 2 t + m)
      const float my_scale = __fdiv_rn(z, 7.0f);
      const float my_inv = z > 0.f ? __fdiv_rn(7.0f, z) : 0.f;
      if ((lane & 3) == 0 && n0 + (lane >> 3) < a.N) {    // lane 4 (2 t + m) stores for (token t, tensor m)
        const int m = (lane >> 2) & 1;
        a.Xs[m][head0 + n0 + (lane >> 3)] = my_scale;
        if (m && a.KsP) a.KsP[bh * a.npad + n0 + (lane >> 3)] = my_scale;
      }
#pragma unroll
      for (int t = 0; t < TOK; ++t) {
        if (n0 + t >= a.N) break;
#pragma unroll
        for (int m = 0; m < 2; ++m)
          prep_store_token<D>(a, m, head0 + n0 + t, lane, y[t][m], __shfl_sync(0xffffffffu, my_inv, 4 * (2 * t + m)));
      }
    }
  } else {
    // one scale per (tensor, 128-token group): CTA = group, warp w owns tokens [16 w, 16 w + 16) of it
    for (int g = blockIdx.x; g < a.nG; g += gridDim.x) {
      const int gbase = g * kTile + warp * (kTile / WPB);
      float am0 = 0.f, am1 = 0.f;
      PosWalk pos;
      pos.init(gbase, TOK, a.gh, a.gw);
      for (int i = 0; i < kTile / WPB / TOK; ++i, pos.advance(a.gh, a.gw)) {
        const int n0 = gbase + i * TOK;
        if (n0 >= a.N) break;
        prep_compute_y<D, ROT>(a, ln, &ybuf[ROT == ROTATTN_ROT_HALF ? warp : 0][0][0][0], head0, n0, pos.pt, pos.ph, pos.pw, lane, hx, y);
#pragma unroll
        for (int t = 0; t < TOK; ++t)
          if (n0 + t < a.N) {
#pragma unroll
            for (int j = 0; j < CPL; ++j) { am0 = fmaxf(am0, fabsf(y[t][0][j])); am1 = fmaxf(am1, fabsf(y[t][1][j])); }
          }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        am0 = fmaxf(am0, __shfl_xor_sync(0xffffffffu, am0, o));
        am1 = fmaxf(am1, __shfl_xor_sync(0xffffffffu, am1, o));
      }
      if (lane == 0) { gmax[warp][0] = am0; gmax[warp][1] = am1; }
      __syncthreads();
      am0 = 0.f; am1 = 0.f;
#pragma unroll
      for (int w = 0; w < WPB; ++w) { am0 = fmaxf(am0, gmax[w][0]); am1 = fmaxf(am1, gmax[w][1]); }
      const float inv0 = am0 > 0.f ? __fdiv_rn(7.0f, am0) : 0.f, inv1 = am1 > 0.f ? __fdiv_rn(7.0f, am1) : 0.f;
      if (threadIdx.x == 0) {
        a.Xs[0][bh * a.nG + g] = __fdiv_rn(am0, 7.0f);
        a.Xs[1][bh * a.nG + g] = __fdiv_rn(am1, 7.0f);
      }
      pos.init(gbase, TOK, a.gh, a.gw);
      for (int i = 0; i < kTile / WPB / TOK; ++i, pos.advance(a.gh, a.gw)) {
        const int n0 = gbase + i * TOK;
        if (n0 >= a.N) break;
        prep_compute_y<D, ROT>(a, ln, &ybuf[ROT == ROTATTN_ROT_HALF ? warp : 0][0][0][0], head0, n0, pos.pt, pos.ph, pos.pw, lane, hx, y);
#pragma unroll
        for (int t = 0; t < TOK; ++t) {
          if (n0 + t >= a.N) break;
          if (a.X16[0]) {
            prep_store_fp16<D>(a, 0, head0 + n0 + t, lane, y[t][0]);
            prep_store_fp16<D>(a, 1, head0 + n0 + t, lane, y[t][1]);
          }
          prep_store_token<D>(a, 0, head0 + n0 + t, lane, y[t][0], inv0);
          prep_store_token<D>(a, 1, head0 + n0 + t, lane, y[t][1], inv1);
        }
      }
      __syncthreads();                                   // gmax is reused by the next group
    }
  }
}

// ------------------------------------------------------------------------------------------------
// quant_v: one CTA per (bh, group of 128 tokens).  V is read once into registers; the per-channel
// amax is reduced through shuffles + shared memory; codes go out packed [N, D/2] and, transposed
// through a swizzled shared tile, as operand bytes [D, npad] (K-major B operand of the P~V MMA).
// VSC = 1: one scale per group (the maximum over the channels as well).  SM = 1: v - column mean is quantised.
// ------------------------------------------------------------------------------------------------
template <int D, int VSC, int SM>
// 4 CTAs per SM cap the kernel at 64 registers (24 bytes of spill); 3 CTAs (80 registers, no spill) measure the same on cfg 2
// (0.0496 vs 0.0497 ms per-channel, 0.0371 vs 0.0351 ms per-group): the spill is not the limiter (round 3).
#ifndef ROTATTN_QV_MINBLOCKS
#define ROTATTN_QV_MINBLOCKS 4
#endif
__global__ void __launch_bounds__(256, ROTATTN_QV_MINBLOCKS) quant_v_kernel(const __half* __restrict__ V, uint8_t* __restrict__ V4,
                                                      float* __restrict__ Vs, int8_t* __restrict__ V8T,
                                                      const float* __restrict__ means, int N, int nG, int npad) {
  constexpr int CR = D / 8;           // 16-byte chunks per row
  constexpr int QPP = 256 / CR;       // row-quads per pass
  constexpr int NPASS = 32 / QPP;     // passes over the 32 row-quads
  constexpr int SW = 32 / CR;         // swizzle multiplier
  __shared__ float amax_s[8][CR][8];
  __shared__ uint32_t tileT[D][32];
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const int cc = t % CR, q0 = t / CR;
  const int g = blockIdx.x % nG;
  const long long bh = blockIdx.x / nG;
  const int row0 = g * kTile;
  const __half* base = V + (bh * N + row0) * (long long)D + cc * 8;

  uint4 raw[NPASS][4];
#pragma unroll
  for (int ps = 0; ps < NPASS; ++ps)
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      int row = (q0 + ps * QPP) * 4 + r;
      raw[ps][r] = (row0 + row < N) ? __ldcs(reinterpret_cast<const uint4*>(base + (long long)row * D)) : make_uint4(0, 0, 0, 0);
    }
  float mu[8];
  if (SM) {
#pragma unroll
    for (int j = 0; j < 8; ++j) mu[j] = means[(bh * 3 + 2) * D + cc * 8 + j];
  }
  float am[8];
  if (!SM) {
    // per-channel amax over this thread's 16 rows on packed halves (max of |fp16| is exact), then across the CTA
    __half2 am2[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) am2[k] = __floats2half2_rn(0.f, 0.f);
#pragma unroll
    for (int ps = 0; ps < NPASS; ++ps)
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const __half2* h2 = reinterpret_cast<const __half2*>(&raw[ps][r]);
#pragma unroll
        for (int k = 0; k < 4; ++k) am2[k] = __hmax2(am2[k], __habs2(h2[k]));
      }
#pragma unroll
    for (int k = 0; k < 4; ++k) { am[2 * k] = __low2float(am2[k]); am[2 * k + 1] = __high2float(am2[k]); }
  } else {
#pragma unroll
    for (int j = 0; j < 8; ++j) am[j] = 0.f;
#pragma unroll
    for (int ps = 0; ps < NPASS; ++ps)
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        if (row0 + (q0 + ps * QPP) * 4 + r < N) {          // rows beyond N do not exist: they must not contribute |0 - mean|
          const __half2* h2 = reinterpret_cast<const __half2*>(&raw[ps][r]);
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const float2 x = __half22float2(h2[k]);
            am[2 * k] = fmaxf(am[2 * k], fabsf(__fsub_rn(x.x, mu[2 * k])));
            am[2 * k + 1] = fmaxf(am[2 * k + 1], fabsf(__fsub_rn(x.y, mu[2 * k + 1])));
          }
        }
      }
  }
#pragma unroll
  for (int o = CR; o < 32; o <<= 1)
#pragma unroll
    for (int j = 0; j < 8; ++j) am[j] = fmaxf(am[j], __shfl_xor_sync(0xffffffffu, am[j], o));
  if (lane < CR) {
#pragma unroll
    for (int j = 0; j < 8; ++j) amax_s[warp][cc][j] = am[j];
  }
  __syncthreads();
  float inv[8];
  if (VSC == 0) {
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      float m = 0.f;
#pragma unroll
      for (int w = 0; w < 8; ++w) m = fmaxf(m, amax_s[w][cc][j]);
      inv[j] = m > 0.f ? __fdiv_rn(7.0f, m) : 0.f;
      if (t < CR) Vs[(bh * nG + g) * D + cc * 8 + j] = __fdiv_rn(m, 7.0f);
    }
  } else {
    float m = 0.f;
    const float* flat = &amax_s[0][0][0];
    for (int i = lane; i < 8 * CR * 8; i += 32) m = fmaxf(m, flat[i]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    const float iv = m > 0.f ? __fdiv_rn(7.0f, m) : 0.f;
#pragma unroll
    for (int j = 0; j < 8; ++j) inv[j] = iv;
    if (t == 0) Vs[bh * nG + g] = __fdiv_rn(m, 7.0f);
  }
  // code = rne(v * inv) in [-7,7] without clamping (|v| <= amax, inv = rn(7/amax)); q + 1.5*2^23 holds the two's-
  // complement code in its low byte, |q| + 1.5*2^23 the magnitude; the operand byte takes the sign of q.
#pragma unroll
  for (int ps = 0; ps < NPASS; ++ps) {
    uint32_t fa[4][8], sg[4][8];
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const __half2* h2 = reinterpret_cast<const __half2*>(&raw[ps][r]);
      uint32_t nb[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        float2 x = __half22float2(h2[k]);
        if (SM) { x.x = __fsub_rn(x.x, mu[2 * k]); x.y = __fsub_rn(x.y, mu[2 * k + 1]); }
        const float qa = __fmul_rn(x.x, inv[2 * k]), qb = __fmul_rn(x.y, inv[2 * k + 1]);
        const uint32_t sa = __float_as_uint(__fadd_rn(qa, 12582912.f)), sb = __float_as_uint(__fadd_rn(qb, 12582912.f));
        fa[r][2 * k] = __float_as_uint(__fadd_rn(fabsf(qa), 12582912.f));
        fa[r][2 * k + 1] = __float_as_uint(__fadd_rn(fabsf(qb), 12582912.f));
        sg[r][2 * k] = __float_as_uint(qa);
        sg[r][2 * k + 1] = __float_as_uint(qb);
        nb[k] = (sa & 0xFu) | ((sb << 4) & 0xF0u);
      }
      const uint32_t pk = __byte_perm(__byte_perm(nb[0], nb[1], 0x0040), __byte_perm(nb[2], nb[3], 0x0040), 0x5410);
      int row = (q0 + ps * QPP) * 4 + r;
      if (row0 + row < N) *reinterpret_cast<uint32_t*>(V4 + (bh * N + row0 + row) * (long long)(D / 2) + cc * 4) = pk;
    }
    if (V8T) {
      const int word = q0 + ps * QPP;
      const bool r1 = row0 + word * 4 + 1 < N, r2 = row0 + word * 4 + 2 < N, r3 = row0 + word * 4 + 3 < N, r0 = row0 + word * 4 < N;
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        // operand byte of (row r, channel j) = magnitude | sign (only where the magnitude is non-zero: no -0 byte)
        uint32_t mag = __byte_perm(__byte_perm(fa[0][j], fa[1][j], 0x0040), __byte_perm(fa[2][j], fa[3][j], 0x0040), 0x5410);
        const uint32_t sgn = __byte_perm(__byte_perm(sg[0][j], sg[1][j], 0x0073), __byte_perm(sg[2][j], sg[3][j], 0x0073), 0x5410);
        if (SM) mag &= (r0 ? 0xFFu : 0u) | (r1 ? 0xFF00u : 0u) | (r2 ? 0xFF0000u : 0u) | (r3 ? 0xFF000000u : 0u);   // pad keys stay 0
        const uint32_t nz = (mag + 0x7F7F7F7Fu) & 0x80808080u;
        tileT[cc * 8 + j][(word ^ (SW * cc)) & 31] = mag | (sgn & nz);
      }
    }
  }
  if (V8T) {
    __syncthreads();
    int8_t* dst = V8T + (bh * D + warp) * (long long)npad + row0 + lane * 4;
#pragma unroll
    for (int i = 0; i < D / 8; ++i) {                       // channel ch = warp + 8 i
      const int ch = warp + 8 * i;
      *reinterpret_cast<uint32_t*>(dst + (long long)(8 * i) * npad) = tileT[ch][(lane ^ (SW * (ch / 8))) & 31];
    }
  }
}

// ------------------------------------------------------------------------------------------------
// smoothing pre-pass helpers (f2): fixed-point column sums of V, and sums -> means
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) smooth_v_stats_kernel(const __half* __restrict__ V, long long* __restrict__ sums, int N, int D,
                                                             int rows_per_cta) {
  // grid (chunks, BH); thread = (row lane, channel pair): V is fp16, so v * 2^24 is an integer and the int64 sum is exact
  const long long bh = blockIdx.y;
  const int cp = threadIdx.x % (D / 2), rl = threadIdx.x / (D / 2), rstep = blockDim.x / (D / 2);
  const int r0 = blockIdx.x * rows_per_cta, r1 = min(N, r0 + rows_per_cta);
  long long s0 = 0, s1 = 0;
  for (int r = r0 + rl; r < r1; r += rstep) {
    const float2 x = __half22float2(*reinterpret_cast<const __half2*>(V + (bh * N + r) * (long long)D + 2 * cp));
    s0 += __float2ll_rn(__fmul_rn(x.x, kFixV));
    s1 += __float2ll_rn(__fmul_rn(x.y, kFixV));
  }
  unsigned long long* dst = reinterpret_cast<unsigned long long*>(sums) + (bh * 3 + 2) * D + 2 * cp;
  atomicAdd(dst, (unsigned long long)s0);
  atomicAdd(dst + 1, (unsigned long long)s1);
}

__global__ void smooth_finalize_kernel(const long long* __restrict__ sums, float* __restrict__ means, int total, int D, int N) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= total) return;
  const int which = (i / D) % 3;
  const double unit = which == 2 ? (double)kFixV : (double)kFixQK;
  means[i] = (float)((double)sums[i] / ((double)N * unit));      // int64 -> fp64 (rn), one fp64 division, one rounding to fp32
}

__global__ void smooth_read_kernel(const float* __restrict__ means, const float* __restrict__ kcp, float* __restrict__ means_out,
                                   float* __restrict__ kc_out, int n_means, long long BH, int N, int npad) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (means_out && i < n_means) means_out[i] = means[i];
  if (kc_out && i < BH * N) kc_out[i] = kcp[(i / N) * npad + i % N];
}

// ------------------------------------------------------------------------------------------------
// unpack helpers: rebuild the widened copies from the packed public buffers (fresh workspace).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int nib2int(uint32_t nib) { return (int)((nib ^ 8u) & 0xFu) - 8; }

__global__ void unpack_qk_kernel(const uint8_t* __restrict__ X4, int8_t* __restrict__ X8, long long tokens, int D) {
  // one thread per output 4-byte word
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long total = tokens * (kQKRowBytes / 4);
  if (idx >= total) return;
  const long long tok = idx / (kQKRowBytes / 4);
  const int w = (int)(idx % (kQKRowBytes / 4));
  uint32_t out = 0;
  if (w * 4 < D) {
    const uint16_t pk = *reinterpret_cast<const uint16_t*>(X4 + tok * (D / 2) + w * 2);
#pragma unroll
    for (int j = 0; j < 4; ++j) out |= code_byte(nib2int((pk >> (4 * j)) & 0xF)) << (8 * j);
  }
  *reinterpret_cast<uint32_t*>(X8 + tok * kQKRowBytes + w * 4) = out;
}

__global__ void unpack_vt_kernel(const uint8_t* __restrict__ V4, int8_t* __restrict__ V8T, int N, int D, int npad) {
  // grid: (npad/128, BH); block 256: transposes one 128-token group through shared memory
  __shared__ int8_t tile[128][128 + 4];
  const long long bh = blockIdx.y;
  const int row0 = blockIdx.x * kTile;
  for (int i = threadIdx.x; i < kTile * (D / 2); i += blockDim.x) {
    int r = i / (D / 2), b = i % (D / 2);
    uint8_t pk = (row0 + r < N) ? V4[(bh * N + row0 + r) * (long long)(D / 2) + b] : 0;
    tile[2 * b][r] = (int8_t)code_byte(nib2int(pk & 0xF));
    tile[2 * b + 1][r] = (int8_t)code_byte(nib2int(pk >> 4));
  }
  __syncthreads();
  for (int i = threadIdx.x; i < D * kTile; i += blockDim.x) {
    int ch = i / kTile, r = i % kTile;
    V8T[(bh * D + ch) * (long long)npad + row0 + r] = tile[ch][r];
  }
}

__global__ void pad_ks_kernel(const float* __restrict__ Ks, float* __restrict__ KsP, long long BH, int N, int npad) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= BH * npad) return;
  const int n = (int)(i % npad);
  KsP[i] = n < N ? Ks[(i / npad) * N + n] : 1.f;       // keys >= N: fwd_int4 masks their accumulators with -inf, the scale must be finite and > 0
}

int launch_unpack_qk(const rotattn_params& p, const uint8_t* X4, int8_t* X8, cudaStream_t st) {
  const long long tokens = (long long)p.B * p.H * p.N;
  const long long total = tokens * (kQKRowBytes / 4);
  unpack_qk_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(X4, X8, tokens, p.D);
  ROTATTN_CUDA_TRY(cudaGetLastError());
  return ROTATTN_OK;
}

int launch_unpack_vt(const rotattn_params& p, const uint8_t* V4, int8_t* V8T, int npad, cudaStream_t st) {
  dim3 grid(npad / kTile, p.B * p.H);
  unpack_vt_kernel<<<grid, 256, 0, st>>>(V4, V8T, p.N, p.D, npad);
  ROTATTN_CUDA_TRY(cudaGetLastError());
  return ROTATTN_OK;
}

int launch_pad_ks(const rotattn_params& p, const float* Ks, float* KsP, int npad, cudaStream_t st) {
  const long long total = (long long)p.B * p.H * npad;
  pad_ks_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(Ks, KsP, (long long)p.B * p.H, p.N, npad);
  ROTATTN_CUDA_TRY(cudaGetLastError());
  return ROTATTN_OK;
}

template <int D, int ROT, int MODE>
static int launch_prepare_rot(const rotattn_params& p, const PrepArgs& a, cudaStream_t st) {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int BH = p.B * p.H;
  const long long cap = ((long long)sms * 2 * 8 + BH - 1) / BH;                             // 2 resident CTAs per SM, 8 waves at most
  if (p.qk_group == 1 || MODE == PREP_STATS) {
    long long blocks_needed = ((long long)a.N + kPrepWarps * kPrepTok - 1) / (kPrepWarps * kPrepTok);     // per (b,h)
    dim3 grid((unsigned)(blocks_needed < cap ? blocks_needed : cap), (unsigned)BH);
    if (grid.x == 0) grid.x = 1;
    prepare_qk_kernel<D, ROT, 1, MODE><<<grid, 256, 0, st>>>(a);
  } else {
    dim3 grid((unsigned)(a.nG < cap ? a.nG : cap), (unsigned)BH);
    prepare_qk_kernel<D, ROT, 128, MODE == PREP_STATS ? PREP_QUANT : MODE><<<grid, 256, 0, st>>>(a);
  }
  ROTATTN_CUDA_TRY(cudaGetLastError());
  return ROTATTN_OK;
}

template <int D, int MODE>
static int launch_prepare(const rotattn_params& p, const PrepArgs& a, cudaStream_t st) {
  switch (p.rot_mode) {
    case ROTATTN_ROT_NONE:
    case ROTATTN_ROT_INTERLEAVED:   // merged into the table: same kernel as plain RoPE
      return launch_prepare_rot<D, ROTATTN_ROT_NONE, MODE>(p, a, st);
    case ROTATTN_ROT_HALF:
      return launch_prepare_rot<D, ROTATTN_ROT_HALF, MODE>(p, a, st);
    default:
      return launch_prepare_rot<D, ROTATTN_ROT_FULL, MODE>(p, a, st);
  }
}

static void fill_prep_args(const rotattn_params* p, PrepArgs& a, const float* coef_dev, const float* rot_dev, const void* Q,
                           const void* K) {
  a.X[0] = (const __half*)Q; a.X[1] = (const __half*)K;
  a.coef = (const float4*)coef_dev; a.rot = (const float4*)rot_dev;
  a.N = p->N; a.n_rope = p->grid_t * p->grid_h * p->grid_w;
  a.gt = p->grid_t; a.gh = p->grid_h; a.gw = p->grid_w;
  a.Pt = p->pairs_t; a.Ph = p->pairs_h; a.Pw = p->pairs_w;
  a.nG = ceil_div(p->N, kTile);
  a.npad = a.nG * kTile;
  a.kc_scale = (float)(1.4426950408889634 / sqrt((double)p->D));
}

}  // namespace rotattn

using namespace rotattn;

extern "C" int rotattn_prepare_qk(const rotattn_params* p, const float* coef_dev, const float* rot_dev,
                                  const void* Q, const void* K, uint8_t* Q4, float* Qs, uint8_t* K4, float* Ks,
                                  void* Qrope16, void* Krope16, void* workspace, size_t ws_bytes, void* stream) {
  int st = rotattn_validate(p);
  if (st != ROTATTN_OK) return st;
  if (!coef_dev || !Q || !K || !Q4 || !Qs || !K4 || !Ks) return ROTATTN_ERR_INVALID_ARG;
  if (p->smooth && !workspace) return ROTATTN_ERR_INVALID_ARG;          // the column means live in the workspace
  if ((st = check_device_sm100()) != ROTATTN_OK) return st;
  PrepArgs a{};
  fill_prep_args(p, a, coef_dev, rot_dev, Q, K);
  a.X4[0] = Q4; a.X4[1] = K4; a.Xs[0] = Qs; a.Xs[1] = Ks;
  a.X16[0] = (__half*)Qrope16; a.X16[1] = (__half*)Krope16;
  if (workspace) {
    WsInt4 ws(*p);
    if (ws_bytes < ws.total) return ROTATTN_ERR_WORKSPACE_TOO_SMALL;
    a.X8[0] = (int8_t*)workspace + ws.q8; a.X8[1] = (int8_t*)workspace + ws.k8;
    a.KsP = (float*)((uint8_t*)workspace + ws.ksp);
    a.means = (const float*)((uint8_t*)workspace + ws.means);
    a.KcP = (float*)((uint8_t*)workspace + ws.kcp);
  }
  cudaStream_t cs = (cudaStream_t)stream;
  if (p->smooth) return p->D == 128 ? launch_prepare<128, PREP_QUANT_SMOOTH>(*p, a, cs) : launch_prepare<64, PREP_QUANT_SMOOTH>(*p, a, cs);
  return p->D == 128 ? launch_prepare<128, PREP_QUANT>(*p, a, cs) : launch_prepare<64, PREP_QUANT>(*p, a, cs);
}

extern "C" int rotattn_smooth_stats(const rotattn_params* p, const float* coef_dev, const float* rot_dev, const void* Q,
                                    const void* K, const void* V, void* workspace, size_t ws_bytes, void* stream) {
  int st = rotattn_validate(p);
  if (st != ROTATTN_OK) return st;
  if (!p->smooth || !coef_dev || !Q || !K || !V || !workspace) return ROTATTN_ERR_INVALID_ARG;
  WsInt4 ws(*p);
  if (ws_bytes < ws.total) return ROTATTN_ERR_WORKSPACE_TOO_SMALL;
  if ((st = check_device_sm100()) != ROTATTN_OK) return st;
  cudaStream_t cs = (cudaStream_t)stream;
  const int BH = p->B * p->H, D = p->D;
  long long* sums = (long long*)((uint8_t*)workspace + ws.sums);
  float* means = (float*)((uint8_t*)workspace + ws.means);
  ROTATTN_CUDA_TRY(cudaMemsetAsync(sums, 0, (size_t)BH * 3 * D * 8, cs));
  PrepArgs a{};
  fill_prep_args(p, a, coef_dev, rot_dev, Q, K);
  a.sums = sums;
  st = D == 128 ? launch_prepare<128, PREP_STATS>(*p, a, cs) : launch_prepare<64, PREP_STATS>(*p, a, cs);
  if (st != ROTATTN_OK) return st;
  {
    const int rows_per_cta = 512;
    dim3 grid((unsigned)ceil_div(p->N, rows_per_cta), (unsigned)BH);
    smooth_v_stats_kernel<<<grid, 256, 0, cs>>>((const __half*)V, sums, p->N, D, rows_per_cta);
    ROTATTN_CUDA_TRY(cudaGetLastError());
  }
  smooth_finalize_kernel<<<ceil_div(BH * 3 * D, 256), 256, 0, cs>>>(sums, means, BH * 3 * D, D, p->N);
  ROTATTN_CUDA_TRY(cudaGetLastError());
  return ROTATTN_OK;
}

extern "C" int rotattn_smooth_read(const rotattn_params* p, const void* workspace, size_t ws_bytes, float* means_out,
                                   float* kcorr_out, void* stream) {
  int st = rotattn_validate(p);
  if (st != ROTATTN_OK) return st;
  if (!p->smooth || !workspace || (!means_out && !kcorr_out)) return ROTATTN_ERR_INVALID_ARG;
  WsInt4 ws(*p);
  if (ws_bytes < ws.total) return ROTATTN_ERR_WORKSPACE_TOO_SMALL;
  const long long BH = (long long)p->B * p->H;
  const long long n = BH * p->N > BH * 3 * p->D ? BH * p->N : BH * 3 * p->D;
  smooth_read_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
      (const float*)((const uint8_t*)workspace + ws.means), (const float*)((const uint8_t*)workspace + ws.kcp), means_out,
      kcorr_out, (int)(BH * 3 * p->D), BH, p->N, ws.npad);
  ROTATTN_CUDA_TRY(cudaGetLastError());
  return ROTATTN_OK;
}

extern "C" int rotattn_quant_v(const rotattn_params* p, const void* V, uint8_t* V4, float* Vs,
                               void* workspace, size_t ws_bytes, void* stream) {
  int st = rotattn_validate(p);
  if (st != ROTATTN_OK) return st;
  if (!V || !V4 || !Vs) return ROTATTN_ERR_INVALID_ARG;
  if (p->smooth && !workspace) return ROTATTN_ERR_INVALID_ARG;
  if ((st = check_device_sm100()) != ROTATTN_OK) return st;
  int8_t* v8t = nullptr;
  const float* means = nullptr;
  WsInt4 ws(*p);
  if (workspace) {
    if (ws_bytes < ws.total) return ROTATTN_ERR_WORKSPACE_TOO_SMALL;
    v8t = (int8_t*)workspace + ws.v8t;
    means = (const float*)((uint8_t*)workspace + ws.means);
  }
  const int nG = ceil_div(p->N, kTile);
  const unsigned grid = (unsigned)((long long)p->B * p->H * nG);
  cudaStream_t cs = (cudaStream_t)stream;
  const __half* v = (const __half*)V;
#define ROTATTN_QV(DD, VSC, SM) quant_v_kernel<DD, VSC, SM><<<grid, 256, 0, cs>>>(v, V4, Vs, v8t, means, p->N, nG, ws.npad)
  if (p->D == 128) {
    if (p->smooth) ROTATTN_QV(128, 0, 1);
    else if (p->v_scale == ROTATTN_VSCALE_GROUP) ROTATTN_QV(128, 1, 0);
    else ROTATTN_QV(128, 0, 0);
  } else {
    if (p->smooth) ROTATTN_QV(64, 0, 1);
    else if (p->v_scale == ROTATTN_VSCALE_GROUP) ROTATTN_QV(64, 1, 0);
    else ROTATTN_QV(64, 0, 0);
  }
#undef ROTATTN_QV
  ROTATTN_CUDA_TRY(cudaGetLastError());
  return ROTATTN_OK;
}
