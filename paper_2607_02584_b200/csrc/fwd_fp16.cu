// rotattn_fwd_fp16 (step a10): FP16 FlashAttention forward on tcgen05 kind::f16 — the fallback precision
// and the speed baseline the INT4 kernel is compared with (L267 "custom FP16 attention").
//
// One CTA = TWO 128-row query tiles (X = 0, 1) of one (b,h) sharing every K / V tile (V is read as it lies in memory,
// [keys, D], as an MN-major B operand - no transposed copy); 16 warps, warp-specialised:
//   warps 0-3 / 4-7  softmax group of tile 0 / 1: one thread per query row, the whole 128-key row of S in registers
//                    (single pass over tensor memory), fp16 P written back over S (TMEM A operand of P V)
//   warps 8-11       correction group: lazy rescale of the fp32 O accumulators that live in TMEM across KV blocks,
//                    epilogue O/l for both tiles
//   warp 12          TMEM allocator        warp 13  TMA producer
//   warp 14          MMA issuer 2: O_X += P_X V        warp 15  MMA issuer 1: S_X = Q_X K^T
// TMEM (512 columns): S_0, S_1 at 0/128 (fp16 P aliases the first 64 columns of its S), O_0, O_1 at 256/384.
// While one tile is in its softmax the tensor pipe works for the other one.  The running reference max only moves
// when a block max exceeds it by more than 2^8 (exact: P and l are relative to the same reference), so the O rescale is
// rare after the first blocks.
#include <cmath>
#include <cstdio>
#include "tc_common.cuh"

namespace rotattn {

constexpr int F_STAGES = 2;
constexpr int F_RING = 4;
constexpr int kFp16Threads = 512;
constexpr int kFWarpAlloc = 12, kFWarpTma = 13, kFWarpMmaPV = 14, kFWarpMmaS = 15;

struct FwdFp16Args {
  __half* O;
  float* O32;               // F32OUT flavour only (rotattn_debug.h): O/l before the rounding to fp16
  const int32_t* head_sel;
  int N, nblk;
  float scale_log2;
};

template <int D>
struct SmemFp16 {
  static constexpr int PANELS = D / 64;                 // 64 fp16 = one 128-byte swizzle row
  static constexpr int Q_BYTES = 128 * D * 2;           // one query tile
  static constexpr int K_BYTES = 128 * D * 2;
  static constexpr int V_BYTES = D * 128 * 2;           // V^T tile: D rows x 128 keys
  static constexpr int OFF_Q = 0;                       // [2 tiles]
  static constexpr int OFF_K = OFF_Q + 2 * Q_BYTES;
  static constexpr int OFF_V = OFF_K + F_STAGES * K_BYTES;
  static constexpr int OFF_AL = OFF_V + F_STAGES * V_BYTES;   // float [2 tiles][F_RING][128] alpha
  static constexpr int OFF_L = OFF_AL + 2 * F_RING * 128 * 4; // float [2 tiles][128]
  static constexpr int OFF_BAR = OFF_L + 2 * 128 * 4;
  static constexpr int NBAR = 1 + 4 * F_STAGES + 2 * (1 + 1 + 1 + 1 + F_RING + 1);
  static constexpr int OFF_TMEM = OFF_BAR + NBAR * 8;
  static constexpr int TOTAL = OFF_TMEM + 16;
};

__device__ __forceinline__ float ex2f(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ uint32_t pack_half2(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

template <int D, bool F32OUT = false>
__global__ void __launch_bounds__(kFp16Threads, 1)
fwd_fp16_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                const __grid_constant__ CUtensorMap tmV, const FwdFp16Args a) {
  using L = SmemFp16<D>;
  extern __shared__ __align__(1024) uint8_t smem[];      // no static shared memory in this kernel: base is 1024-aligned
  uint8_t* sQ = smem + L::OFF_Q;
  uint8_t* sK = smem + L::OFF_K;
  uint8_t* sV = smem + L::OFF_V;
  float* sAl = (float*)(smem + L::OFF_AL);
  float* sL = (float*)(smem + L::OFF_L);
  uint64_t* bars = (uint64_t*)(smem + L::OFF_BAR);
  uint64_t* q_full = bars;
  uint64_t* k_full = q_full + 1;
  uint64_t* k_empty = k_full + F_STAGES;
  uint64_t* v_full = k_empty + F_STAGES;
  uint64_t* v_empty = v_full + F_STAGES;
  uint64_t* s_full = v_empty + F_STAGES;      // [2 tiles] MMA -> softmax
  uint64_t* p_full = s_full + 2;              // [2] softmax -> MMA (count 128)
  uint64_t* pv_done = p_full + 2;             // [2] O_X += P_X V (block j) complete: -> S issuer (S_X / P_X buffer free), correction
  uint64_t* o_ready = pv_done + 2;            // [2] correction -> MMA: O_X rescaled for block j (count 128)
  uint64_t* al_full = o_ready + 2;            // [2][F_RING] softmax -> correction (count 128)
  uint64_t* l_full = al_full + 2 * F_RING;    // [2] softmax -> correction (count 128)
  uint32_t* tmem_slot = (uint32_t*)(smem + L::OFF_TMEM);

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);   // warp-uniform
  const int lane = threadIdx.x & 31;
  const int q0 = blockIdx.x * 2 * kTile;
  const int bh = a.head_sel ? a.head_sel[blockIdx.y] : (int)blockIdx.y;
  const int nblk = a.nblk;

  if (threadIdx.x == 0) {
    if (smem_u32(smem) & 1023u) __trap();
    mbar_init(q_full, 1);
    for (int i = 0; i < F_STAGES; ++i) { mbar_init(&k_full[i], 1); mbar_init(&k_empty[i], 1); mbar_init(&v_full[i], 1); mbar_init(&v_empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&s_full[i], 1); mbar_init(&p_full[i], 128); mbar_init(&pv_done[i], 1); mbar_init(&o_ready[i], 128); mbar_init(&l_full[i], 128); }
    for (int i = 0; i < 2 * F_RING; ++i) mbar_init(&al_full[i], 128);
    fence_mbar_init();
  }
  if (warp == kFWarpAlloc) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  constexpr uint32_t TM_S = 0, TM_O = 256;

  // register pool of the CTA = 512 x 128; after redistribution 128 x 40 + 128 x 88 + 256 x 184 = 63488
  if (warp >= 12) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
    if (warp == kFWarpTma) {
      // ---------------------------------------------------------------- TMA producer
      if (elect_one()) {
        tma_prefetch_desc(&tmQ); tma_prefetch_desc(&tmK); tma_prefetch_desc(&tmV);
        mbar_arrive_expect_tx(q_full, 2 * L::Q_BYTES);
#pragma unroll
        for (int x = 0; x < 2; ++x)
#pragma unroll
          for (int pn = 0; pn < L::PANELS; ++pn)
            tma_load_3d(sQ + x * L::Q_BYTES + pn * 16384, &tmQ, q_full, pn * 64, q0 + x * kTile, bh);
      }
      __syncwarp();
      for (int j = 0; j < nblk; ++j) {
        const int s = j % F_STAGES;
        const uint32_t ph = (j / F_STAGES) & 1;
        mbar_wait(&k_empty[s], ph ^ 1);
        if (elect_one()) {
          mbar_arrive_expect_tx(&k_full[s], L::K_BYTES);
#pragma unroll
          for (int pn = 0; pn < L::PANELS; ++pn)
            tma_load_3d(sK + s * L::K_BYTES + pn * 16384, &tmK, &k_full[s], pn * 64, j * kTile, bh);
        }
        __syncwarp();
        mbar_wait(&v_empty[s], ph ^ 1);
        if (elect_one()) {
          mbar_arrive_expect_tx(&v_full[s], L::V_BYTES);
#pragma unroll
          for (int pn = 0; pn < L::PANELS; ++pn)   // V as it lies in memory, [keys, D]: channel panels of 64, 128 keys each (keys >= N arrive as zeros)
            tma_load_3d(sV + s * L::V_BYTES + pn * 16384, &tmV, &v_full[s], pn * 64, j * kTile, bh);
        }
        __syncwarp();
      }
    } else if (warp == kFWarpMmaS) {
      // ---------------------------------------------------------------- MMA issuer 1: S_X(j) = Q_X K(j)^T
      constexpr uint32_t idesc_s = umma_idesc(1, 0, 0, 128, 128);     // f32 <- f16 x f16
      mbar_wait(q_full, 0);
      for (int j = 0; j < nblk; ++j) {
        const int st = j % F_STAGES;
        mbar_wait(&k_full[st], (j / F_STAGES) & 1);
#pragma unroll
        for (int x = 0; x < 2; ++x) {
          if (j > 0) mbar_wait(&pv_done[x], (j - 1) & 1);              // P_X(j-1), which aliases S_X, has been consumed
          // Stagger the two tiles by one softmax: tile 1 starts when tile 0 has left its first exp2 phase, so that from
          // then on one tile is in its softmax (MUFU) while the tensor pipe works for the other one.
          if (j == 0 && x == 1) mbar_wait(&p_full[0], 0);
          tc_fence_after();
          if (elect_one()) {
            const uint32_t q_addr = smem_u32(sQ + x * L::Q_BYTES), k_addr = smem_u32(sK + st * L::K_BYTES);
#pragma unroll
            for (int kk = 0; kk < D / 16; ++kk) {
              const uint32_t off = (kk >> 2) * 16384 + (kk & 3) * 32;
              mma_ss<MmaKind::F16>(tmem_base + TM_S + x * 128, umma_desc_k128(q_addr + off), umma_desc_k128(k_addr + off), idesc_s, kk != 0);
            }
            tc_commit(&s_full[x]);
            if (x == 1) tc_commit(&k_empty[st]);
          }
          __syncwarp();
        }
      }
    } else if (warp == kFWarpMmaPV) {
      // ---------------------------------------------------------------- MMA issuer 2: O_X += P_X(j) V(j)
      constexpr uint32_t idesc_pv = umma_idesc(1, 0, 0, 128, D) | (1u << 16);     // f32 <- f16 (TMEM) x f16, B MN-major
      for (int j = 0; j < nblk; ++j) {
        const int st = j % F_STAGES;
        mbar_wait(&v_full[st], (j / F_STAGES) & 1);
#pragma unroll
        for (int x = 0; x < 2; ++x) {
          mbar_wait(&p_full[x], j & 1);
          mbar_wait(&o_ready[x], j & 1);
          tc_fence_after();
          if (elect_one()) {
            const uint32_t v_addr = smem_u32(sV + st * L::V_BYTES);
#pragma unroll
            for (int kk = 0; kk < 8; ++kk) {
              // B operand = the V tile [128 keys, D], MN-major (D contiguous): 16 keys per step = two 8-row atoms
              mma_ts<MmaKind::F16>(tmem_base + TM_O + x * 128, tmem_base + TM_S + x * 128 + 8 * kk,
                                   umma_desc_mn128(v_addr + kk * 2048, 16384, 1024), idesc_pv, (j | kk) != 0);
            }
            tc_commit(&pv_done[x]);
            if (x == 1) tc_commit(&v_empty[st]);
          }
          __syncwarp();
        }
      }
    }
  }
  else if (warp < 8) {
    // ------------------------------------------------------------------ softmax group of tile x (1 thread = 1 query row)
    asm volatile("setmaxnreg.inc.sync.aligned.u32 184;");
    const int x = warp >> 2;
    const int r = (warp & 3) * 32 + lane;
    const uint32_t s_addr = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + TM_S + x * 128;
    float* al = sAl + x * F_RING * 128;
    const float c = a.scale_log2;
    const float2 c2 = make_float2(c, c);
    float m_ref = -INFINITY, l_run = 0.f;
    for (int j = 0; j < nblk; ++j) {
      const int nvalid = min(kTile, a.N - j * kTile);
      mbar_wait(&s_full[x], j & 1);
      tc_fence_after();
      uint32_t t[128];
      {
        uint32_t(&t0)[32] = *reinterpret_cast<uint32_t(*)[32]>(&t[0]);
        uint32_t(&t1)[32] = *reinterpret_cast<uint32_t(*)[32]>(&t[32]);
        uint32_t(&t2)[32] = *reinterpret_cast<uint32_t(*)[32]>(&t[64]);
        uint32_t(&t3)[32] = *reinterpret_cast<uint32_t(*)[32]>(&t[96]);
        tmem_ld32(s_addr, t0); tmem_ld32(s_addr + 32, t1); tmem_ld32(s_addr + 64, t2); tmem_ld32(s_addr + 96, t3);
        tmem_wait_ld();
      }
      if (nvalid < kTile) {                                             // ragged last block: keys >= N never win the max, P = 0
#pragma unroll
        for (int i = 0; i < 128; ++i) if (i >= nvalid) t[i] = 0xff800000u;
      }
      float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;
#pragma unroll
      for (int i = 0; i < 128; i += 8) {
        mx0 = fmax3(mx0, __uint_as_float(t[i]), __uint_as_float(t[i + 1]));
        mx1 = fmax3(mx1, __uint_as_float(t[i + 2]), __uint_as_float(t[i + 3]));
        mx2 = fmax3(mx2, __uint_as_float(t[i + 4]), __uint_as_float(t[i + 5]));
        mx3 = fmax3(mx3, __uint_as_float(t[i + 6]), __uint_as_float(t[i + 7]));
      }
      const float mt = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * c;
      float alpha = 1.f, m_new = m_ref;
      if (mt > m_ref + 8.f) { m_new = mt; alpha = ex2f(m_ref - m_new); }     // first block: m_ref = -inf -> alpha = 0
      al[(j % F_RING) * 128 + r] = alpha;
      mbar_arrive(&al_full[x * F_RING + j % F_RING]);
      const float2 nm2 = make_float2(-m_new, -m_new);
      float2 ls0 = make_float2(0.f, 0.f), ls1 = make_float2(0.f, 0.f);
#pragma unroll
      for (int cc = 0; cc < 4; ++cc) {                                  // 32 keys -> 16 columns of fp16 pairs
        uint32_t pw[16];
#pragma unroll
        for (int g = 0; g < 16; g += 2) {
          const int i = cc * 32 + 2 * g;
          const float2 e0 = ffma2(make_float2(__uint_as_float(t[i]), __uint_as_float(t[i + 1])), c2, nm2);
          const float2 e1 = ffma2(make_float2(__uint_as_float(t[i + 2]), __uint_as_float(t[i + 3])), c2, nm2);
          const float2 p0 = make_float2(ex2f(e0.x), ex2f(e0.y)), p1 = make_float2(ex2f(e1.x), ex2f(e1.y));
          ls0 = fadd2(ls0, p0);
          ls1 = fadd2(ls1, p1);
          pw[g] = pack_half2(p0.x, p0.y);
          pw[g + 1] = pack_half2(p1.x, p1.y);
        }
        tmem_st16(s_addr + cc * 16, pw);                                // fp16 P aliases S columns [0,64): the row is in registers
      }
      l_run = alpha * l_run + ((ls0.x + ls0.y) + (ls1.x + ls1.y));
      m_ref = m_new;
      tmem_wait_st();
      tc_fence_before();
      mbar_arrive(&p_full[x]);
    }
    sL[x * 128 + r] = l_run;
    mbar_arrive(&l_full[x]);
  } else if (warp < 12) {
    // ------------------------------------------------------------------ correction group (both tiles)
    asm volatile("setmaxnreg.dec.sync.aligned.u32 88;");
    const int r = (warp & 3) * 32 + lane;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    for (int j = 0; j < nblk; ++j) {
#pragma unroll
      for (int x = 0; x < 2; ++x) {
        mbar_wait(&al_full[x * F_RING + j % F_RING], (j / F_RING) & 1);
        const float alpha = sAl[(x * F_RING + j % F_RING) * 128 + r];
        if (j > 0 && __any_sync(0xffffffffu, alpha != 1.f)) {
          mbar_wait(&pv_done[x], (j - 1) & 1);
          tc_fence_after();
#pragma unroll
          for (int cc = 0; cc < D / 32; ++cc) {
            uint32_t v[32];
            tmem_ld32(tmem_base + lane_off + TM_O + x * 128 + cc * 32, v);
            tmem_wait_ld();
#pragma unroll
            for (int i = 0; i < 32; ++i) v[i] = __float_as_uint(__uint_as_float(v[i]) * alpha);
            tmem_st32(tmem_base + lane_off + TM_O + x * 128 + cc * 32, v);
          }
          tmem_wait_st();
        }
        tc_fence_before();
        mbar_arrive(&o_ready[x]);
      }
    }
#pragma unroll
    for (int x = 0; x < 2; ++x) {
      const int row = q0 + x * kTile + r;
      mbar_wait(&pv_done[x], (nblk - 1) & 1);
      tc_fence_after();
      mbar_wait(&l_full[x], 0);
      const float inv_l = 1.f / sL[x * 128 + r];
#pragma unroll
      for (int cc = 0; cc < D / 32; ++cc) {
        uint32_t v[32];
        tmem_ld32(tmem_base + lane_off + TM_O + x * 128 + cc * 32, v);
        tmem_wait_ld();
        if (F32OUT) {                        // test flavour: the quotient itself, so that the kernel's arithmetic can be
          if (row < a.N) {                   // held to the strict bound without the rounding of the fp16 output
            float* dst = a.O32 + ((size_t)bh * a.N + row) * D + cc * 32;
#pragma unroll
            for (int d = 0; d < 32; d += 4)
              *reinterpret_cast<float4*>(dst + d) =
                  make_float4(__uint_as_float(v[d]) * inv_l, __uint_as_float(v[d + 1]) * inv_l,
                              __uint_as_float(v[d + 2]) * inv_l, __uint_as_float(v[d + 3]) * inv_l);
          }
        } else if (row < a.N) {
          __half* dst = a.O + ((size_t)bh * a.N + row) * D + cc * 32;
#pragma unroll
          for (int d = 0; d < 32; d += 8) {
            uint4 o;
            o.x = pack_half2(__uint_as_float(v[d]) * inv_l, __uint_as_float(v[d + 1]) * inv_l);
            o.y = pack_half2(__uint_as_float(v[d + 2]) * inv_l, __uint_as_float(v[d + 3]) * inv_l);
            o.z = pack_half2(__uint_as_float(v[d + 4]) * inv_l, __uint_as_float(v[d + 5]) * inv_l);
            o.w = pack_half2(__uint_as_float(v[d + 6]) * inv_l, __uint_as_float(v[d + 7]) * inv_l);
            *reinterpret_cast<uint4*>(dst + d) = o;
          }
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kFWarpAlloc) tmem_dealloc(tmem_base, 512);
}

}  // namespace rotattn

using namespace rotattn;

template <int D, bool F32OUT>
static int launch_fp16(const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv, const FwdFp16Args& a, dim3 grid,
                       cudaStream_t cs) {
  constexpr int smem = SmemFp16<D>::TOTAL;
  static PerDeviceOnce once;    // per device: ptxas must have allocated exactly the register pool setmaxnreg redistributes,
  int dev = 0;                  // and the dynamic shared-memory opt-in is a per-device attribute
  ROTATTN_CUDA_TRY(cudaGetDevice(&dev));
  if (!once.done(dev)) {
    cudaFuncAttributes fa;
    ROTATTN_CUDA_TRY(cudaFuncGetAttributes(&fa, fwd_fp16_kernel<D, F32OUT>));
    if (fa.numRegs != 128) {
      set_error_text("fwd_fp16_kernel: unexpected register allocation (setmaxnreg pool assumes 128 registers per thread)");
      return ROTATTN_ERR_UNSUPPORTED;
    }
    ROTATTN_CUDA_TRY(cudaFuncSetAttribute(fwd_fp16_kernel<D, F32OUT>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    once.mark(dev);
  }
  fwd_fp16_kernel<D, F32OUT><<<grid, kFp16Threads, smem, cs>>>(tq, tk, tv, a);
  ROTATTN_CUDA_TRY(cudaGetLastError());
  return ROTATTN_OK;
}

static int fwd_fp16_common(const rotattn_params* p, const void* Q16, const void* K16, const void* V16, void* O, bool f32out,
                           const int32_t* head_sel, int32_t n_sel, void* workspace, size_t ws_bytes, void* stream) {
  int st = rotattn_validate(p);
  if (st != ROTATTN_OK) return st;
  if (!Q16 || !K16 || !V16 || !O) return ROTATTN_ERR_INVALID_ARG;
  if (((uintptr_t)Q16 & 15) || ((uintptr_t)K16 & 15) || ((uintptr_t)V16 & 15) || ((uintptr_t)O & 15)) return ROTATTN_ERR_INVALID_ARG;   // TMA / 16-byte stores
  (void)workspace; (void)ws_bytes;      // no scratch any more (V is read in place); the arguments stay for the ABI
  const int BH = p->B * p->H;
  if (head_sel && (n_sel < 1 || n_sel > BH)) return ROTATTN_ERR_INVALID_ARG;
  if ((st = check_device_sm100()) != ROTATTN_OK) return st;
  cudaStream_t cs = (cudaStream_t)stream;
  const uint64_t N = p->N, D = p->D;
  CUtensorMap tq, tk, tv;
  if ((st = make_tmap_3d(&tq, Q16, 2, D, N, BH, D * 2, N * D * 2, 64, 128)) != ROTATTN_OK) return st;
  if ((st = make_tmap_3d(&tk, K16, 2, D, N, BH, D * 2, N * D * 2, 64, 128)) != ROTATTN_OK) return st;
  if ((st = make_tmap_3d(&tv, V16, 2, D, N, BH, D * 2, N * D * 2, 64, 128)) != ROTATTN_OK) return st;
  FwdFp16Args a{};
  a.O = f32out ? nullptr : (__half*)O; a.O32 = f32out ? (float*)O : nullptr;
  a.head_sel = head_sel; a.N = p->N; a.nblk = ceil_div(p->N, kTile);
  a.scale_log2 = (float)(1.4426950408889634 / std::sqrt((double)p->D));
  dim3 grid(ceil_div(p->N, 2 * kTile), head_sel ? n_sel : BH);     // one CTA per pair of 128-row query tiles
  if (f32out) return p->D == 128 ? launch_fp16<128, true>(tq, tk, tv, a, grid, cs) : launch_fp16<64, true>(tq, tk, tv, a, grid, cs);
  return p->D == 128 ? launch_fp16<128, false>(tq, tk, tv, a, grid, cs) : launch_fp16<64, false>(tq, tk, tv, a, grid, cs);
}

extern "C" int rotattn_fwd_fp16(const rotattn_params* p, const void* Q16, const void* K16, const void* V16, void* O,
                                const int32_t* head_sel, int32_t n_sel, void* workspace, size_t ws_bytes, void* stream) {
  return fwd_fp16_common(p, Q16, K16, V16, O, false, head_sel, n_sel, workspace, ws_bytes, stream);
}

// rotattn_debug.h: the same kernel with O/l stored as fp32 (test aid, never on the timed path)
extern "C" int rotattn_fwd_fp16_debug_f32(const rotattn_params* p, const void* Q16, const void* K16, const void* V16, float* O32,
                                          const int32_t* head_sel, int32_t n_sel, void* workspace, size_t ws_bytes, void* stream) {
  return fwd_fp16_common(p, Q16, K16, V16, O32, true, head_sel, n_sel, workspace, ws_bytes, stream);
}
