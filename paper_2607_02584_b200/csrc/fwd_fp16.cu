// rotattn_fwd_fp16 (step a10): FP16 FlashAttention forward on tcgen05 kind::f16 — the fallback precision
// and the speed baseline the INT4 kernel is compared with (L267 "custom FP16 attention").
//
// One CTA = one 128-row query tile of one (b,h); same warp roles as fwd_int4:
//   warp 0 TMA producer, warp 1 MMA issuer, warp 2 TMEM allocator,
//   warps 4-7 softmax group (S fp32 -> P fp16 in TMEM), warps 8-11 correction group (lazy rescale of the fp32 O
//   accumulator that lives in TMEM across KV blocks; epilogue O/l).
// TMEM: S[2] at 0/128 (fp16 P aliases the first 64 columns of its S buffer), O at 256.
// The running reference max is only moved when the block max exceeds it by more than 2^8 (exact: P and l are
// expressed relative to the same reference), so the O rescale is rare after the first blocks.
#include <cmath>
#include <cstdio>
#include "tc_common.cuh"

namespace rotattn {

constexpr int F_STAGES = 2;
constexpr int F_RING = 4;

struct FwdFp16Args {
  __half* O;
  const int32_t* head_sel;
  int N, nblk;
  float scale_log2;
};

template <int D>
struct SmemFp16 {
  static constexpr int PANELS = D / 64;                 // 64 fp16 = one 128-byte swizzle row
  static constexpr int Q_BYTES = 128 * D * 2;
  static constexpr int K_BYTES = 128 * D * 2;
  static constexpr int V_BYTES = D * 128 * 2;           // V^T tile: D rows x 128 keys
  static constexpr int OFF_Q = 0;
  static constexpr int OFF_K = OFF_Q + Q_BYTES;
  static constexpr int OFF_V = OFF_K + F_STAGES * K_BYTES;
  static constexpr int OFF_AL = OFF_V + F_STAGES * V_BYTES;   // float [F_RING][128] alpha
  static constexpr int OFF_L = OFF_AL + F_RING * 128 * 4;
  static constexpr int OFF_BAR = OFF_L + 128 * 4;
  static constexpr int NBAR = 1 + 4 * F_STAGES + 2 + 2 + 1 + 1 + F_RING + 1;
  static constexpr int OFF_TMEM = OFF_BAR + NBAR * 8;
  static constexpr int TOTAL = OFF_TMEM + 16 + 1024;
};

__device__ __forceinline__ float ex2f(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

template <int D>
__global__ void __launch_bounds__(384, 1)
fwd_fp16_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                const __grid_constant__ CUtensorMap tmV, const FwdFp16Args a) {
  using L = SmemFp16<D>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
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
  uint64_t* s_full = v_empty + F_STAGES;      // [2]
  uint64_t* p_full = s_full + 2;              // [2] count 128
  uint64_t* pv_done = p_full + 2;             // [1] MMA -> correction: P V(j) accumulated
  uint64_t* o_ready = pv_done + 1;            // [1] correction -> MMA: O rescaled for block j (count 128)
  uint64_t* al_full = o_ready + 1;            // [F_RING] softmax -> correction (count 128)
  uint64_t* l_full = al_full + F_RING;
  uint32_t* tmem_slot = (uint32_t*)(smem + L::OFF_TMEM);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int q0 = blockIdx.x * kTile;
  const int bh = a.head_sel ? a.head_sel[blockIdx.y] : (int)blockIdx.y;
  const int nblk = a.nblk;

  if (threadIdx.x == 0) {
    mbar_init(q_full, 1);
    for (int i = 0; i < F_STAGES; ++i) { mbar_init(&k_full[i], 1); mbar_init(&k_empty[i], 1); mbar_init(&v_full[i], 1); mbar_init(&v_empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&s_full[i], 1); mbar_init(&p_full[i], 128); }
    mbar_init(pv_done, 1);
    mbar_init(o_ready, 128);
    for (int i = 0; i < F_RING; ++i) mbar_init(&al_full[i], 128);
    mbar_init(l_full, 128);
    fence_mbar_init();
  }
  if (warp == 2) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  constexpr uint32_t TM_S = 0, TM_O = 256;

  if (warp < 4) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
    if (warp == 0) {
      // ---------------------------------------------------------------- TMA producer
      if (lane == 0) {
        tma_prefetch_desc(&tmQ); tma_prefetch_desc(&tmK); tma_prefetch_desc(&tmV);
        mbar_arrive_expect_tx(q_full, L::Q_BYTES);
#pragma unroll
        for (int pn = 0; pn < L::PANELS; ++pn) tma_load_3d(sQ + pn * 16384, &tmQ, q_full, pn * 64, q0, bh);
        int s = 0; uint32_t ph = 0;
        for (int j = 0; j < nblk; ++j) {
          mbar_wait(&k_empty[s], ph ^ 1);
          mbar_arrive_expect_tx(&k_full[s], L::K_BYTES);
#pragma unroll
          for (int pn = 0; pn < L::PANELS; ++pn)
            tma_load_3d(sK + s * L::K_BYTES + pn * 16384, &tmK, &k_full[s], pn * 64, j * kTile, bh);
          mbar_wait(&v_empty[s], ph ^ 1);
          mbar_arrive_expect_tx(&v_full[s], L::V_BYTES);
#pragma unroll
          for (int pn = 0; pn < 2; ++pn)      // key panels of 64
            tma_load_3d(sV + s * L::V_BYTES + pn * (D * 128), &tmV, &v_full[s], j * kTile + pn * 64, 0, bh);
          if (++s == F_STAGES) { s = 0; ph ^= 1; }
        }
      }
    } else if (warp == 1) {
      // ---------------------------------------------------------------- MMA issuer
      if (lane == 0) {
        constexpr uint32_t idesc_s = umma_idesc(1, 0, 0, 128, 128);     // f32 <- f16 x f16
        constexpr uint32_t idesc_pv = umma_idesc(1, 0, 0, 128, D);
        const uint32_t q_addr = smem_u32(sQ);
        auto issue_s = [&](int stage, int buf) {
          const uint32_t k_addr = smem_u32(sK + stage * L::K_BYTES);
#pragma unroll
          for (int kk = 0; kk < D / 16; ++kk) {
            const uint32_t off = (kk >> 2) * 16384 + (kk & 3) * 32;
            mma_ss<MmaKind::F16>(tmem_base + TM_S + buf * 128, umma_desc_k128(q_addr + off), umma_desc_k128(k_addr + off),
                                 idesc_s, kk != 0);
          }
        };
        mbar_wait(q_full, 0);
        mbar_wait(&k_full[0], 0);
        tc_fence_after();
        issue_s(0, 0);
        tc_commit(&k_empty[0]);
        tc_commit(&s_full[0]);
        int ks = 1; uint32_t kph = 0;
        int vs = 0; uint32_t vph = 0;
        for (int j = 0; j < nblk; ++j) {
          const int b = j & 1;
          if (j + 1 < nblk) {
            if (ks == F_STAGES) { ks = 0; kph ^= 1; }
            mbar_wait(&k_full[ks], kph);
            tc_fence_after();
            issue_s(ks, b ^ 1);
            tc_commit(&k_empty[ks]);
            tc_commit(&s_full[b ^ 1]);
            ++ks;
          }
          mbar_wait(&p_full[b], (j >> 1) & 1);
          mbar_wait(&v_full[vs], vph);
          mbar_wait(o_ready, j & 1);
          tc_fence_after();
          const uint32_t v_addr = smem_u32(sV + vs * L::V_BYTES);
#pragma unroll
          for (int kk = 0; kk < 8; ++kk) {
            const uint32_t off = (kk >> 2) * (D * 128) + (kk & 3) * 32;
            mma_ts<MmaKind::F16>(tmem_base + TM_O, tmem_base + TM_S + b * 128 + 8 * kk, umma_desc_k128(v_addr + off),
                                 idesc_pv, (j | kk) != 0);
          }
          tc_commit(&v_empty[vs]);
          tc_commit(pv_done);
          if (++vs == F_STAGES) { vs = 0; vph ^= 1; }
        }
      }
    }
  } else if (warp < 8) {
    // ------------------------------------------------------------------ softmax group (1 thread = 1 query row)
    asm volatile("setmaxnreg.inc.sync.aligned.u32 216;");
    const int r = threadIdx.x - 128;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    const float c = a.scale_log2;
    float m_ref = -INFINITY, l_run = 0.f;
    for (int j = 0; j < nblk; ++j) {
      const int b = j & 1;
      const int nvalid = min(kTile, a.N - j * kTile);
      mbar_wait(&s_full[b], (j >> 1) & 1);
      tc_fence_after();
      float t[128];
      float mx[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
      for (int cc = 0; cc < 4; ++cc) {
        uint32_t v[32];
        tmem_ld32(tmem_base + lane_off + TM_S + b * 128 + cc * 32, v);
        tmem_wait_ld();
#pragma unroll
        for (int i = 0; i < 32; ++i) {
          const float x = __uint_as_float(v[i]);
          t[cc * 32 + i] = x;
          if (cc * 32 + i < nvalid) mx[i & 3] = fmaxf(mx[i & 3], x);
        }
      }
      const float mt = fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3])) * c;
      float alpha = 1.f, m_new = m_ref;
      if (mt > m_ref + 8.f) { m_new = mt; alpha = ex2f(m_ref - m_new); }     // first block: m_ref = -inf -> alpha = 0
      sAl[(j % F_RING) * 128 + r] = alpha;
      mbar_arrive(&al_full[j % F_RING]);
      float ls[4] = {0.f, 0.f, 0.f, 0.f};
      uint32_t pw[64];
#pragma unroll
      for (int g = 0; g < 64; ++g) {
        float e0 = fmaf(t[2 * g], c, -m_new), e1 = fmaf(t[2 * g + 1], c, -m_new);
        if (2 * g >= nvalid) e0 = -INFINITY;
        if (2 * g + 1 >= nvalid) e1 = -INFINITY;
        const float p0 = ex2f(e0), p1 = ex2f(e1);
        ls[g & 3] += p0 + p1;
        __half2 h = __floats2half2_rn(p0, p1);
        pw[g] = *reinterpret_cast<uint32_t*>(&h);
      }
      {
        uint32_t(&lo)[32] = *reinterpret_cast<uint32_t(*)[32]>(&pw[0]);
        uint32_t(&hi)[32] = *reinterpret_cast<uint32_t(*)[32]>(&pw[32]);
        tmem_st32(tmem_base + lane_off + TM_S + b * 128, lo);            // fp16 P aliases S columns [0,64)
        tmem_st32(tmem_base + lane_off + TM_S + b * 128 + 32, hi);
      }
      l_run = alpha * l_run + ((ls[0] + ls[1]) + (ls[2] + ls[3]));
      m_ref = m_new;
      tmem_wait_st();
      tc_fence_before();
      mbar_arrive(&p_full[b]);
    }
    sL[r] = l_run;
    mbar_arrive(l_full);
  } else {
    // ------------------------------------------------------------------ correction group
    asm volatile("setmaxnreg.inc.sync.aligned.u32 216;");
    const int r = threadIdx.x - 256;
    const int row = q0 + r;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    for (int j = 0; j < nblk; ++j) {
      mbar_wait(&al_full[j % F_RING], (j / F_RING) & 1);
      const float alpha = sAl[(j % F_RING) * 128 + r];
      if (j > 0 && __any_sync(0xffffffffu, alpha != 1.f)) {
        mbar_wait(pv_done, (j - 1) & 1);
        tc_fence_after();
#pragma unroll
        for (int cc = 0; cc < D / 32; ++cc) {
          uint32_t v[32];
          tmem_ld32(tmem_base + lane_off + TM_O + cc * 32, v);
          tmem_wait_ld();
#pragma unroll
          for (int i = 0; i < 32; ++i) v[i] = __float_as_uint(__uint_as_float(v[i]) * alpha);
          tmem_st32(tmem_base + lane_off + TM_O + cc * 32, v);
        }
        tmem_wait_st();
      }
      tc_fence_before();
      mbar_arrive(o_ready);
    }
    mbar_wait(pv_done, (nblk - 1) & 1);
    tc_fence_after();
    mbar_wait(l_full, 0);
    const float inv_l = 1.f / sL[r];
#pragma unroll
    for (int cc = 0; cc < D / 32; ++cc) {
      uint32_t v[32];
      tmem_ld32(tmem_base + lane_off + TM_O + cc * 32, v);
      tmem_wait_ld();
      if (row < a.N) {
        __half* dst = a.O + ((size_t)bh * a.N + row) * D + cc * 32;
#pragma unroll
        for (int d = 0; d < 32; d += 8) {
          __half2 h[4];
#pragma unroll
          for (int i = 0; i < 4; ++i)
            h[i] = __floats2half2_rn(__uint_as_float(v[d + 2 * i]) * inv_l, __uint_as_float(v[d + 2 * i + 1]) * inv_l);
          *reinterpret_cast<uint4*>(dst + d) = *reinterpret_cast<uint4*>(h);
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem_base, 512);
}

// V [BH, N, D] fp16 -> V^T [BH, D, npad] fp16 (zero padded): K-major B operand of the P V product.
__global__ void transpose_v_kernel(const __half* __restrict__ V, __half* __restrict__ VT, int N, int D, int npad) {
  __shared__ __half tile[64][64 + 2];
  const long long bh = blockIdx.z;
  const int n0 = blockIdx.x * 64, d0 = blockIdx.y * 64;
  for (int i = threadIdx.x; i < 64 * 32; i += blockDim.x) {
    const int rr = i / 32, c2 = i % 32;
    __half2 v = __floats2half2_rn(0.f, 0.f);
    if (n0 + rr < N) v = *reinterpret_cast<const __half2*>(V + (bh * N + n0 + rr) * (long long)D + d0 + 2 * c2);
    tile[rr][2 * c2] = __low2half(v);
    tile[rr][2 * c2 + 1] = __high2half(v);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < 64 * 32; i += blockDim.x) {
    const int dd = i / 32, n2 = i % 32;
    __half2 v = __halves2half2(tile[2 * n2][dd], tile[2 * n2 + 1][dd]);
    *reinterpret_cast<__half2*>(VT + (bh * D + d0 + dd) * (long long)npad + n0 + 2 * n2) = v;
  }
}

}  // namespace rotattn

using namespace rotattn;

template <int D>
static int launch_fp16(const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv, const FwdFp16Args& a, dim3 grid,
                       cudaStream_t cs) {
  constexpr int smem = SmemFp16<D>::TOTAL;
  ROTATTN_CUDA_TRY(cudaFuncSetAttribute(fwd_fp16_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  fwd_fp16_kernel<D><<<grid, 384, smem, cs>>>(tq, tk, tv, a);
  ROTATTN_CUDA_TRY(cudaGetLastError());
  return ROTATTN_OK;
}

extern "C" int rotattn_fwd_fp16(const rotattn_params* p, const void* Q16, const void* K16, const void* V16, void* O,
                                const int32_t* head_sel, int32_t n_sel, void* workspace, size_t ws_bytes, void* stream) {
  int st = rotattn_validate(p);
  if (st != ROTATTN_OK) return st;
  if (!Q16 || !K16 || !V16 || !O || !workspace) return ROTATTN_ERR_INVALID_ARG;
  const int BH = p->B * p->H;
  if (head_sel && (n_sel < 1 || n_sel > BH)) return ROTATTN_ERR_INVALID_ARG;
  WsFp16 ws(*p);
  if (ws_bytes < ws.total) return ROTATTN_ERR_WORKSPACE_TOO_SMALL;
  if ((st = check_device_sm100()) != ROTATTN_OK) return st;
  cudaStream_t cs = (cudaStream_t)stream;
  __half* vt = (__half*)((uint8_t*)workspace + ws.vt);
  {
    dim3 g(ws.npad / 64, p->D / 64, BH);
    transpose_v_kernel<<<g, 256, 0, cs>>>((const __half*)V16, vt, p->N, p->D, ws.npad);
    ROTATTN_CUDA_TRY(cudaGetLastError());
  }
  const uint64_t N = p->N, D = p->D;
  CUtensorMap tq, tk, tv;
  if ((st = make_tmap_3d(&tq, Q16, 2, D, N, BH, D * 2, N * D * 2, 64, 128)) != ROTATTN_OK) return st;
  if ((st = make_tmap_3d(&tk, K16, 2, D, N, BH, D * 2, N * D * 2, 64, 128)) != ROTATTN_OK) return st;
  if ((st = make_tmap_3d(&tv, vt, 2, ws.npad, D, BH, (uint64_t)ws.npad * 2, D * ws.npad * 2, 64, (uint32_t)D)) != ROTATTN_OK) return st;
  FwdFp16Args a{};
  a.O = (__half*)O; a.head_sel = head_sel; a.N = p->N; a.nblk = ceil_div(p->N, kTile);
  a.scale_log2 = (float)(1.4426950408889634 / std::sqrt((double)p->D));
  dim3 grid(a.nblk, head_sel ? n_sel : BH);
  return p->D == 128 ? launch_fp16<128>(tq, tk, tv, a, grid, cs) : launch_fp16<64>(tq, tk, tv, a, grid, cs);
}
