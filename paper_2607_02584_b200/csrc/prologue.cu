// Prologue kernels (HBM-bound): prepare_qk (a1+a2), quant_v (a3) and the unpack helpers.
// Code-producing arithmetic is fp32 with one rounding per operation (__fmul_rn/__fadd_rn/__fdiv_rn,
// never contracted) so that the INT4 codes are reproducible bit for bit ("bit-exact prologue").
#include "common.cuh"

namespace rotattn {

// ------------------------------------------------------------------------------------------------
// prepare_qk: one warp per token; lane l owns channels [CPL*l, CPL*l+CPL) of Q and of K.
// ------------------------------------------------------------------------------------------------
struct PrepArgs {
  const __half* X[2];     // Q, K  [BH*N, D]
  uint8_t* X4[2];         // packed codes [BH*N, D/2]
  float* Xs[2];           // scales [BH*N]
  __half* X16[2];         // optional fp16 y
  int8_t* X8[2];          // optional widened codes [BH*N, 128]
  const float4* coef;     // table rows
  const float4* rot;      // [D/2] blocks or nullptr (H_2)
  long long total;        // BH*N tokens
  int N, n_rope, gt, gh, gw, Pt, Ph, Pw;
};

__device__ __forceinline__ int quant_code(float y, float inv) {
  int c = __float2int_rn(__fmul_rn(y, inv));       // round half to even
  return max(-7, min(7, c));
}
// Widened MMA operand byte of a code c in [-7,7] (or a P code in [0,15]): sign-magnitude, which is the E4M3
// encoding of c * 2^-9 (E4M3 subnormals are m * 2^-9, and bytes 8..15 are the first normal binade 2^-6 * (1 + m/8)),
// so tcgen05 kind::f8f6f4 multiplies and accumulates the integer codes exactly, scaled by 2^-18, in fp32.
__device__ __forceinline__ uint32_t code_byte(int c) { return (uint32_t)(abs(c) | ((c >> 24) & 0x80)); }

constexpr int kPrepTok = 4;       // tokens per warp iteration: all their loads are issued before any arithmetic (bytes in flight)

template <int D, int ROT>
__global__ void __launch_bounds__(256, 2) prepare_qk_kernel(const PrepArgs a) {
  constexpr int CPL = D / 32;       // channels per lane
  constexpr int PPL = CPL / 2;      // RoPE pairs per lane
  constexpr int WPB = 8;            // warps per block
  constexpr int TOK = kPrepTok;
  __shared__ float ybuf[ROT == ROTATTN_ROT_HALF ? WPB : 1][TOK][2][D];   // HALF-rotation exchange buffer
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

  // ---- per-lane constants ----
  int cbase[PPL], cstride[PPL], caxis[PPL];
  {
    const int secbase[3] = {0, (a.gt + 1) * a.Pt, (a.gt + 1) * a.Pt + (a.gh + 1) * a.Ph};
#pragma unroll
    for (int i = 0; i < PPL; ++i) {
      int g = lane * PPL + i;
      int ax = g < a.Pt ? 0 : (g < a.Pt + a.Ph ? 1 : 2);
      int k = g - (ax == 0 ? 0 : (ax == 1 ? a.Pt : a.Pt + a.Ph));
      int P = ax == 0 ? a.Pt : (ax == 1 ? a.Ph : a.Pw);
      caxis[i] = ax; cbase[i] = secbase[ax] + k; cstride[i] = P;
    }
  }
  int partner[CPL]; float ca[CPL], cb[CPL]; bool role_u[CPL];
  if (ROT == ROTATTN_ROT_HALF) {
#pragma unroll
    for (int j = 0; j < CPL; ++j) {
      int c = lane * CPL + j;
      int sec = c < 2 * a.Pt ? 0 : (c < 2 * (a.Pt + a.Ph) ? 1 : 2);
      int o = sec == 0 ? 0 : (sec == 1 ? 2 * a.Pt : 2 * (a.Pt + a.Ph));
      int P = sec == 0 ? a.Pt : (sec == 1 ? a.Ph : a.Pw);
      int goff = o / 2;
      int i = c - o;
      role_u[j] = i < P;
      int blk = goff + (role_u[j] ? i : i - P);
      partner[j] = role_u[j] ? c + P : c - P;
      float4 r = a.rot ? a.rot[blk] : make_float4(0.70710678118654752440f, 0.70710678118654752440f,
                                                  0.70710678118654752440f, -0.70710678118654752440f);
      // u' = u r00 + v r10 (this lane holds u), v' = u r01 + v r11 (this lane holds v): own value times ca + partner times cb
      ca[j] = role_u[j] ? r.x : r.w;
      cb[j] = role_u[j] ? r.z : r.y;
    }
  }

  // blockIdx.y = (b,h); the warps of the grid's x dimension stride over that head's tokens, TOK consecutive ones at a time
  const long long head0 = (long long)blockIdx.y * a.N;
  const int nstride = gridDim.x * WPB * TOK;
  for (int n0 = (blockIdx.x * WPB + warp) * TOK; n0 < a.N; n0 += nstride) {
    // (t,h,w) of the first token by two 32-bit divisions; the following ones by carry propagation
    int pw = n0 % a.gw, pr = n0 / a.gw;
    int ph = pr % a.gh, pt = pr / a.gh;
    // ---- load phase: TOK tokens x (Q, K) + their coefficient rows, all independent
    float4 A[TOK][PPL];
    __half hx[TOK][2][CPL];
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
          const int pos = caxis[i] == 0 ? p0 : (caxis[i] == 1 ? p1 : p2);
          A[t][i] = __ldg(a.coef + cbase[i] + pos * cstride[i]);
        }
      }
      if (++pw == a.gw) { pw = 0; if (++ph == a.gh) { ph = 0; ++pt; } }
    }
    // ---- RoPE (merged with the interleaved rotation through the table)
    float y[TOK][2][CPL];
#pragma unroll
    for (int t = 0; t < TOK; ++t)
#pragma unroll
      for (int m = 0; m < 2; ++m)
#pragma unroll
        for (int i = 0; i < PPL; ++i) {
          float x0 = __half2float(hx[t][m][2 * i]), x1 = __half2float(hx[t][m][2 * i + 1]);
          y[t][m][2 * i]     = __fadd_rn(__fmul_rn(x0, A[t][i].x), __fmul_rn(x1, A[t][i].z));
          y[t][m][2 * i + 1] = __fadd_rn(__fmul_rn(x0, A[t][i].y), __fmul_rn(x1, A[t][i].w));
        }
    if (ROT == ROTATTN_ROT_HALF) {
#pragma unroll
      for (int t = 0; t < TOK; ++t)
#pragma unroll
        for (int m = 0; m < 2; ++m) {
          if (CPL == 4) *reinterpret_cast<float4*>(&ybuf[warp][t][m][lane * CPL]) = make_float4(y[t][m][0], y[t][m][1], y[t][m][2], y[t][m][3]);
          else *reinterpret_cast<float2*>(&ybuf[warp][t][m][lane * CPL]) = make_float2(y[t][m][0], y[t][m][1]);
        }
      __syncwarp();
#pragma unroll
      for (int t = 0; t < TOK; ++t)
#pragma unroll
        for (int m = 0; m < 2; ++m)
#pragma unroll
          for (int j = 0; j < CPL; ++j) {
            const float other = ybuf[warp][t][m][partner[j]];
            y[t][m][j] = __fadd_rn(__fmul_rn(y[t][m][j], ca[j]), __fmul_rn(other, cb[j]));   // fp32 addition commutes exactly
          }
      __syncwarp();
    }
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
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
      for (int t = 0; t < TOK; ++t)
#pragma unroll
        for (int m = 0; m < 2; ++m) amax[t][m] = fmaxf(amax[t][m], __shfl_xor_sync(0xffffffffu, amax[t][m], o));
    // scale = amax / 7 and inv = 7 / amax are IEEE divisions: lane (2 t + m) computes the pair once, then broadcast
    float my_scale = 0.f, my_inv = 0.f;
    {
      float am = 0.f;
#pragma unroll
      for (int t = 0; t < TOK; ++t)
#pragma unroll
        for (int m = 0; m < 2; ++m) am = (lane == 2 * t + m) ? amax[t][m] : am;
      if (lane < 2 * TOK) {
        my_scale = __fdiv_rn(am, 7.0f);
        my_inv = am > 0.f ? __fdiv_rn(7.0f, am) : 0.f;
        if (n0 + (lane >> 1) < a.N) a.Xs[lane & 1][head0 + n0 + (lane >> 1)] = my_scale;     // lane 2 t + m owns (token t, tensor m)
      }
    }
#pragma unroll
    for (int t = 0; t < TOK; ++t) {
      if (n0 + t >= a.N) break;
      const long long tok = head0 + n0 + t;
#pragma unroll
      for (int m = 0; m < 2; ++m) {
        const float inv = __shfl_sync(0xffffffffu, my_inv, 2 * t + m);
        // code = rne(y * inv) is in [-7,7] without clamping (|y| <= amax and inv = rn(7/amax) give |y*inv| < 7.5).
        // fs = q + 1.5*2^23 holds the two's-complement code in its low byte, fa = |q| + 1.5*2^23 the magnitude.
        uint32_t fs[CPL], fa[CPL], yb[CPL];
#pragma unroll
        for (int j = 0; j < CPL; ++j) {
          const float q = __fmul_rn(y[t][m][j], inv);
          fs[j] = __float_as_uint(__fadd_rn(q, 12582912.f));
          fa[j] = __float_as_uint(__fadd_rn(fabsf(q), 12582912.f));
          yb[j] = __float_as_uint(q);
        }
        if (CPL == 4) {
          const uint32_t n01 = (fs[0] & 0xFu) | ((fs[1] << 4) & 0xF0u), n23 = (fs[2] & 0xFu) | ((fs[3] << 4) & 0xF0u);
          *reinterpret_cast<uint16_t*>(a.X4[m] + tok * (D / 2) + lane * 2) = (uint16_t)__byte_perm(n01, n23, 0x0040);
        } else {
          a.X4[m][tok * (D / 2) + lane] = (uint8_t)((fs[0] & 0xFu) | ((fs[1] << 4) & 0xF0u));
        }
        if (a.X8[m]) {
          // sign-magnitude operand bytes (code_byte): magnitude bytes | sign bits of q (a zero code has q = +-0 or |q| < 0.5:
          // its sign must not be stored, hence the mask with the non-zero test folded into the magnitude: -0 byte is avoided
          // by taking the sign only where the magnitude byte is non-zero)
          int8_t* dst = a.X8[m] + tok * kQKRowBytes;
          if (CPL == 4) {
            const uint32_t mag = __byte_perm(__byte_perm(fa[0], fa[1], 0x0040), __byte_perm(fa[2], fa[3], 0x0040), 0x5410);
            const uint32_t sgn = __byte_perm(__byte_perm(yb[0], yb[1], 0x0073), __byte_perm(yb[2], yb[3], 0x0073), 0x5410);
            const uint32_t nz = ((mag + 0x7F7F7F7Fu) & 0x80808080u);     // 0x80 in every byte whose magnitude is non-zero
            *reinterpret_cast<uint32_t*>(dst + lane * 4) = mag | (sgn & nz);
          } else {
            const uint32_t mag = __byte_perm(fa[0], fa[1], 0x0040) & 0xFFFFu;
            const uint32_t sgn = __byte_perm(yb[0], yb[1], 0x0073) & 0xFFFFu;
            const uint32_t nz = ((mag + 0x7F7Fu) & 0x8080u);
            *reinterpret_cast<uint16_t*>(dst + lane * 2) = (uint16_t)(mag | (sgn & nz));
            *reinterpret_cast<uint16_t*>(dst + 64 + lane * 2) = 0;      // zero pad to a 128-byte row
          }
        }
        if (a.X16[m]) {
          __half* dst = a.X16[m] + tok * D + lane * CPL;
          __half hy[CPL];
#pragma unroll
          for (int j = 0; j < CPL; ++j) hy[j] = __float2half_rn(y[t][m][j]);
          if (CPL == 4) *reinterpret_cast<uint2*>(dst) = *reinterpret_cast<uint2*>(hy);
          else *reinterpret_cast<uint32_t*>(dst) = *reinterpret_cast<uint32_t*>(hy);
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// quant_v: one CTA per (bh, group of 128 tokens).  V is read once into registers; the per-channel
// amax is reduced through shuffles + shared memory; codes go out packed [N, D/2] and, transposed
// through a swizzled shared tile, as int8 [D, npad] (K-major B operand of the P~V MMA).
// ------------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(256, 4) quant_v_kernel(const __half* __restrict__ V, uint8_t* __restrict__ V4,
                                                      float* __restrict__ Vs, int8_t* __restrict__ V8T,
                                                      int N, int nG, int npad) {
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
  float am[8];
#pragma unroll
  for (int k = 0; k < 4; ++k) { am[2 * k] = __low2float(am2[k]); am[2 * k + 1] = __high2float(am2[k]); }
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
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    float m = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) m = fmaxf(m, amax_s[w][cc][j]);
    inv[j] = m > 0.f ? __fdiv_rn(7.0f, m) : 0.f;
    if (t < CR) Vs[(bh * nG + g) * D + cc * 8 + j] = __fdiv_rn(m, 7.0f);
  }
  // code = rne(v * inv) in [-7,7] without clamping (|v| <= amax, inv = rn(7/amax)); q + 1.5*2^23 holds the two's-
  // complement code in its low byte, |q| + 1.5*2^23 the magnitude; the sign of the code is the sign bit of the fp16 input.
#pragma unroll
  for (int ps = 0; ps < NPASS; ++ps) {
    uint32_t fa[4][8];
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const __half2* h2 = reinterpret_cast<const __half2*>(&raw[ps][r]);
      uint32_t nb[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const float2 x = __half22float2(h2[k]);
        const float qa = __fmul_rn(x.x, inv[2 * k]), qb = __fmul_rn(x.y, inv[2 * k + 1]);
        const uint32_t sa = __float_as_uint(__fadd_rn(qa, 12582912.f)), sb = __float_as_uint(__fadd_rn(qb, 12582912.f));
        fa[r][2 * k] = __float_as_uint(__fadd_rn(fabsf(qa), 12582912.f));
        fa[r][2 * k + 1] = __float_as_uint(__fadd_rn(fabsf(qb), 12582912.f));
        nb[k] = (sa & 0xFu) | ((sb << 4) & 0xF0u);
      }
      const uint32_t pk = __byte_perm(__byte_perm(nb[0], nb[1], 0x0040), __byte_perm(nb[2], nb[3], 0x0040), 0x5410);
      int row = (q0 + ps * QPP) * 4 + r;
      if (row0 + row < N) *reinterpret_cast<uint32_t*>(V4 + (bh * N + row0 + row) * (long long)(D / 2) + cc * 4) = pk;
    }
    if (V8T) {
      const int word = q0 + ps * QPP;
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        // operand byte of (row r, channel j) = magnitude | sign (only where the magnitude is non-zero: no -0 byte)
        const uint32_t mag = __byte_perm(__byte_perm(fa[0][j], fa[1][j], 0x0040), __byte_perm(fa[2][j], fa[3][j], 0x0040), 0x5410);
        const uint32_t* w0 = reinterpret_cast<const uint32_t*>(&raw[ps][0]);
        const uint32_t* w1 = reinterpret_cast<const uint32_t*>(&raw[ps][1]);
        const uint32_t* w2 = reinterpret_cast<const uint32_t*>(&raw[ps][2]);
        const uint32_t* w3 = reinterpret_cast<const uint32_t*>(&raw[ps][3]);
        const uint32_t sel = (j & 1) ? 0x0073u : 0x0051u;          // byte 3 (odd channel) / byte 1 (even channel) of the half2 word
        const uint32_t sgn = __byte_perm(__byte_perm(w0[j >> 1], w1[j >> 1], sel), __byte_perm(w2[j >> 1], w3[j >> 1], sel), 0x5410);
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

template <int D>
static int launch_prepare(const rotattn_params& p, const PrepArgs& a, cudaStream_t st) {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int BH = p.B * p.H;
  long long blocks_needed = ((long long)a.N + 8 * kPrepTok - 1) / (8 * kPrepTok);     // per (b,h)
  long long cap = ((long long)sms * 2 * 8 + BH - 1) / BH;                             // 2 resident CTAs per SM, 8 waves at most
  dim3 grid((unsigned)(blocks_needed < cap ? blocks_needed : cap), (unsigned)BH);
  if (grid.x == 0) grid.x = 1;
  switch (p.rot_mode) {
    case ROTATTN_ROT_NONE:
    case ROTATTN_ROT_INTERLEAVED:   // merged into the table: same kernel as plain RoPE
      prepare_qk_kernel<D, ROTATTN_ROT_NONE><<<grid, 256, 0, st>>>(a); break;
    default:
      prepare_qk_kernel<D, ROTATTN_ROT_HALF><<<grid, 256, 0, st>>>(a); break;
  }
  ROTATTN_CUDA_TRY(cudaGetLastError());
  return ROTATTN_OK;
}

}  // namespace rotattn

using namespace rotattn;

extern "C" int rotattn_prepare_qk(const rotattn_params* p, const float* coef_dev, const float* rot_dev,
                                  const void* Q, const void* K, uint8_t* Q4, float* Qs, uint8_t* K4, float* Ks,
                                  void* Qrope16, void* Krope16, void* workspace, size_t ws_bytes, void* stream) {
  int st = rotattn_validate(p);
  if (st != ROTATTN_OK) return st;
  if (!coef_dev || !Q || !K || !Q4 || !Qs || !K4 || !Ks) return ROTATTN_ERR_INVALID_ARG;
  if ((st = check_device_sm100()) != ROTATTN_OK) return st;
  PrepArgs a{};
  a.X[0] = (const __half*)Q; a.X[1] = (const __half*)K;
  a.X4[0] = Q4; a.X4[1] = K4; a.Xs[0] = Qs; a.Xs[1] = Ks;
  a.X16[0] = (__half*)Qrope16; a.X16[1] = (__half*)Krope16;
  if (workspace) {
    WsInt4 ws(*p);
    if (ws_bytes < ws.total) return ROTATTN_ERR_WORKSPACE_TOO_SMALL;
    a.X8[0] = (int8_t*)workspace + ws.q8; a.X8[1] = (int8_t*)workspace + ws.k8;
  }
  a.coef = (const float4*)coef_dev; a.rot = (const float4*)rot_dev;
  a.total = (long long)p->B * p->H * p->N;
  a.N = p->N; a.n_rope = p->grid_t * p->grid_h * p->grid_w;
  a.gt = p->grid_t; a.gh = p->grid_h; a.gw = p->grid_w;
  a.Pt = p->pairs_t; a.Ph = p->pairs_h; a.Pw = p->pairs_w;
  return p->D == 128 ? launch_prepare<128>(*p, a, (cudaStream_t)stream) : launch_prepare<64>(*p, a, (cudaStream_t)stream);
}

extern "C" int rotattn_quant_v(const rotattn_params* p, const void* V, uint8_t* V4, float* Vs,
                               void* workspace, size_t ws_bytes, void* stream) {
  int st = rotattn_validate(p);
  if (st != ROTATTN_OK) return st;
  if (!V || !V4 || !Vs) return ROTATTN_ERR_INVALID_ARG;
  if ((st = check_device_sm100()) != ROTATTN_OK) return st;
  int8_t* v8t = nullptr;
  WsInt4 ws(*p);
  if (workspace) {
    if (ws_bytes < ws.total) return ROTATTN_ERR_WORKSPACE_TOO_SMALL;
    v8t = (int8_t*)workspace + ws.v8t;
  }
  const int nG = ceil_div(p->N, kTile);
  const unsigned grid = (unsigned)((long long)p->B * p->H * nG);
  if (p->D == 128)
    quant_v_kernel<128><<<grid, 256, 0, (cudaStream_t)stream>>>((const __half*)V, V4, Vs, v8t, p->N, nG, ws.npad);
  else
    quant_v_kernel<64><<<grid, 256, 0, (cudaStream_t)stream>>>((const __half*)V, V4, Vs, v8t, p->N, nG, ws.npad);
  ROTATTN_CUDA_TRY(cudaGetLastError());
  return ROTATTN_OK;
}
