// fwd_int4_sync: INT4 FlashAttention forward with the softmax serialised over KV blocks (2 threads per query row,
// running max kept by the softmax threads).  Used for p_norm = RUNNING (codes relative to the running max,
// SURVEY 8c reading 13 alternative), where block j cannot be normalised before block j-1 is known.
// Same operand path as fwd_int4_kernel.cuh: tcgen05 kind::f8f6f4 on integer-exact E4M3 code bytes, TMA, TMEM.
#include <cmath>
#include <cstdio>
#include "fwd_int4.cuh"

namespace rotattn {

constexpr int KS_STAGES = 3;
constexpr int KS_RING = 4;

template <int D>
struct SmemInt4Sync {
  static constexpr int Q_BYTES = 128 * 128;
  static constexpr int K_BYTES = 128 * 128;
  static constexpr int V_BYTES = D * 128;
  static constexpr int OFF_Q = 0;
  static constexpr int OFF_K = OFF_Q + Q_BYTES;
  static constexpr int OFF_V = OFF_K + KS_STAGES * K_BYTES;
  static constexpr int OFF_KS = OFF_V + KS_STAGES * V_BYTES;          // float [2][128]
  static constexpr int OFF_VS = OFF_KS + 2 * 128 * 4;                 // float [2][D]
  static constexpr int OFF_AB = OFF_VS + 2 * D * 4;                   // float2 [KS_RING][128]
  static constexpr int OFF_MX = OFF_AB + KS_RING * 128 * 8;           // float [2 parity][2 halves][128]
  static constexpr int OFF_L = OFF_MX + 2 * 2 * 128 * 4;              // float [2 halves][128]
  static constexpr int OFF_BAR = OFF_L + 2 * 128 * 4;                 // mbarriers
  static constexpr int NBAR = 1 + 4 * KS_STAGES + 2 + 2 + 2 + 2 + KS_RING + 1;
  static constexpr int OFF_TMEM = OFF_BAR + NBAR * 8;
  static constexpr int TOTAL = OFF_TMEM + 16 + 1024;                  // + alignment slack
};

template <int D, int P_MODE, int P_NORM, bool DEBUG>
__global__ void __launch_bounds__(kInt4Threads, 1)
fwd_int4_sync_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                const __grid_constant__ CUtensorMap tmV, const FwdInt4Args a) {
  using L = SmemInt4Sync<D>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint8_t* sQ = smem + L::OFF_Q;
  uint8_t* sK = smem + L::OFF_K;
  uint8_t* sV = smem + L::OFF_V;
  float* sKs = (float*)(smem + L::OFF_KS);
  float* sVs = (float*)(smem + L::OFF_VS);
  float2* sAB = (float2*)(smem + L::OFF_AB);
  float* sMx = (float*)(smem + L::OFF_MX);
  float* sL = (float*)(smem + L::OFF_L);
  uint64_t* bars = (uint64_t*)(smem + L::OFF_BAR);
  uint64_t* q_full = bars;
  uint64_t* k_full = q_full + 1;
  uint64_t* k_empty = k_full + KS_STAGES;
  uint64_t* v_full = k_empty + KS_STAGES;
  uint64_t* v_empty = v_full + KS_STAGES;
  uint64_t* s_full = v_empty + KS_STAGES;     // [2] MMA -> softmax
  uint64_t* p_full = s_full + 2;              // [2] softmax -> MMA (count 256)
  uint64_t* pv_full = p_full + 2;             // [2] MMA -> drain
  uint64_t* pv_empty = pv_full + 2;           // [2] drain -> MMA (count 256)
  uint64_t* ab_full = pv_empty + 2;           // [KS_RING] softmax (half 0) -> drain (count 128)
  uint64_t* l_full = ab_full + KS_RING;       // softmax -> drain (count 256)
  uint32_t* tmem_slot = (uint32_t*)(smem + L::OFF_TMEM);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int qtile = DEBUG ? a.dbg_qtile : blockIdx.x;
  const int bh = DEBUG ? a.dbg_bh : (a.head_sel ? a.head_sel[blockIdx.y] : (int)blockIdx.y);
  const int q0 = qtile * kTile;
  const int nblk = a.nblk;

  if (threadIdx.x == 0) {
    mbar_init(q_full, 1);
    for (int i = 0; i < KS_STAGES; ++i) { mbar_init(&k_full[i], 1); mbar_init(&k_empty[i], 1); mbar_init(&v_full[i], 1); mbar_init(&v_empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&s_full[i], 1); mbar_init(&p_full[i], 256); mbar_init(&pv_full[i], 1); mbar_init(&pv_empty[i], 256); }
    for (int i = 0; i < KS_RING; ++i) mbar_init(&ab_full[i], 128);
    mbar_init(l_full, 256);
    fence_mbar_init();
  }
  if (warp == 2) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  constexpr uint32_t TM_S = 0, TM_PV = 256;

  // register pool of the CTA = 640 x 96; after redistribution 128 x 32 + 256 x 104 + 256 x 120 = 61440 (must not exceed it)
  if (warp < 4) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 32;");
    if (warp == 0) {
      // ---------------------------------------------------------------- TMA producer
      if (lane == 0) {
        tma_prefetch_desc(&tmQ); tma_prefetch_desc(&tmK); tma_prefetch_desc(&tmV);
        mbar_arrive_expect_tx(q_full, L::Q_BYTES);
        tma_load_3d(sQ, &tmQ, q_full, 0, q0, bh);
        int s = 0; uint32_t ph = 0;
        for (int j = 0; j < nblk; ++j) {
          mbar_wait(&k_empty[s], ph ^ 1);
          mbar_arrive_expect_tx(&k_full[s], L::K_BYTES);
          tma_load_3d(sK + s * L::K_BYTES, &tmK, &k_full[s], 0, j * kTile, bh);
          mbar_wait(&v_empty[s], ph ^ 1);
          mbar_arrive_expect_tx(&v_full[s], L::V_BYTES);
          tma_load_3d(sV + s * L::V_BYTES, &tmV, &v_full[s], j * kTile, 0, bh);
          if (++s == KS_STAGES) { s = 0; ph ^= 1; }
        }
      }
    } else if (warp == 1) {
      // ---------------------------------------------------------------- MMA issuer
      if (lane == 0) {
        constexpr uint32_t idesc_s = umma_idesc(1, 0, 0, 128, 128);      // f32 <- e4m3 x e4m3 (integer codes * 2^-9)
        constexpr uint32_t idesc_pv = umma_idesc(1, 0, 0, 128, D);       // f32 <- e4m3 x e4m3
        constexpr int KSTEPS_S = D / 32;                                 // D=64 rows are zero-padded to 128 B
        const uint64_t qd = umma_desc_k128(smem_u32(sQ));
        mbar_wait(q_full, 0);
        mbar_wait(&k_full[0], 0);
        tc_fence_after();
        {
          const uint64_t kd = umma_desc_k128(smem_u32(sK));
#pragma unroll
          for (int k = 0; k < KSTEPS_S; ++k) mma_ss<MmaKind::F8F6F4>(tmem_base + TM_S, qd + 2 * k, kd + 2 * k, idesc_s, k != 0);
          tc_commit(&k_empty[0]);
          tc_commit(&s_full[0]);
        }
        int ks = 1; uint32_t kph = 0;       // K ring position of block j+1
        int vs = 0; uint32_t vph = 0;       // V ring position of block j
        for (int j = 0; j < nblk; ++j) {
          const int b = j & 1;
          if (j + 1 < nblk) {
            if (ks == KS_STAGES) { ks = 0; kph ^= 1; }
            mbar_wait(&k_full[ks], kph);
            tc_fence_after();
            const uint64_t kd = umma_desc_k128(smem_u32(sK + ks * L::K_BYTES));
#pragma unroll
            for (int k = 0; k < KSTEPS_S; ++k)
              mma_ss<MmaKind::F8F6F4>(tmem_base + TM_S + (b ^ 1) * 128, qd + 2 * k, kd + 2 * k, idesc_s, k != 0);
            tc_commit(&k_empty[ks]);
            tc_commit(&s_full[b ^ 1]);
            ++ks;
          }
          mbar_wait(&p_full[b], (j >> 1) & 1);
          mbar_wait(&v_full[vs], vph);
          mbar_wait(&pv_empty[b], ((j >> 1) & 1) ^ 1);
          tc_fence_after();
          const uint64_t vd = umma_desc_k128(smem_u32(sV + vs * L::V_BYTES));
#pragma unroll
          for (int k = 0; k < 4; ++k)
            mma_ts<MmaKind::F8F6F4>(tmem_base + TM_PV + b * 128, tmem_base + TM_S + b * 128 + 8 * k, vd + 2 * k, idesc_pv, k != 0);
          tc_commit(&v_empty[vs]);
          tc_commit(&pv_full[b]);
          if (++vs == KS_STAGES) { vs = 0; vph ^= 1; }
        }
      }
    }
  } else if (warp < 12) {
    // ------------------------------------------------------------------ softmax: 2 threads per query row
    asm volatile("setmaxnreg.inc.sync.aligned.u32 104;");
    const int tsm = threadIdx.x - 128;
    const int h = tsm >> 7, r = tsm & 127;          // h: which 64-key half of the block this thread owns
    const int cb = 64 * h;
    const int row = q0 + r;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    // qs >= 1e-30 keeps (-inf) * qs well defined for masked keys; an all-zero query row still gives s == 0 everywhere
    const float qs = (row < a.N) ? fmaxf(a.Qs[(size_t)bh * a.N + row], 1e-30f) : 1e-30f;
    const float2 qs2 = make_float2(qs, qs);
    const float* ksrc = a.Ks + (size_t)bh * a.N;
    constexpr float LEVELS = P_MODE == ROTATTN_P_ASYM15 ? 15.f : 7.f;
    const float2 lev2 = make_float2(LEVELS, LEVELS), magic2 = make_float2(12582912.f, 12582912.f);
    float m_run = -INFINITY, l_run = 0.f;
    if (h == 0) sKs[r] = (r < a.N) ? ksrc[r] * a.scale_log2 : 0.f;
    for (int j = 0; j < nblk; ++j) {
      const int b = j & 1;
      bar_sync(1, 256);                                  // ks'(j) visible; everyone is past block j-1
      float ks_next = 0.f;
      if (h == 0 && j + 1 < nblk) { int kj = (j + 1) * kTile + r; ks_next = (kj < a.N) ? ksrc[kj] * a.scale_log2 : 0.f; }
      const float2* ksb2 = reinterpret_cast<const float2*>(sKs + b * 128 + cb);
      const int nvalid = min(kTile, a.N - j * kTile);    // < 128 only on the ragged last block
      mbar_wait(&s_full[b], (j >> 1) & 1);
      tc_fence_after();
      float2 t2[32];
      {
        uint32_t v0[32], v1[32];
        tmem_ld32(tmem_base + lane_off + TM_S + b * 128 + cb, v0);
        tmem_ld32(tmem_base + lane_off + TM_S + b * 128 + cb + 32, v1);
        tmem_wait_ld();
        if (DEBUG) {
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            a.S_dump[(size_t)r * a.npad + j * kTile + cb + i] = (int32_t)(__uint_as_float(v0[i]) * kAccScale);
            a.S_dump[(size_t)r * a.npad + j * kTile + cb + 32 + i] = (int32_t)(__uint_as_float(v1[i]) * kAccScale);
          }
        }
#pragma unroll
        for (int i = 0; i < 16; ++i) {                                 // t = acc * Ks_j * log2e/sqrt(D)
          t2[i] = fmul2(make_float2(__uint_as_float(v0[2 * i]), __uint_as_float(v0[2 * i + 1])), ksb2[i]);
          t2[16 + i] = fmul2(make_float2(__uint_as_float(v1[2 * i]), __uint_as_float(v1[2 * i + 1])), ksb2[16 + i]);
        }
      }
      if (nvalid < kTile) {                                            // keys >= N: masked out of max, sum and codes
#pragma unroll
        for (int i = 0; i < 32; ++i) {
          if (cb + 2 * i >= nvalid) t2[i].x = -INFINITY;
          if (cb + 2 * i + 1 >= nvalid) t2[i].y = -INFINITY;
        }
      }
      float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
      for (int i = 0; i < 32; i += 2) { mx0 = fmax3(mx0, t2[i].x, t2[i].y); mx1 = fmax3(mx1, t2[i + 1].x, t2[i + 1].y); }
      float tmax = fmaxf(mx0, mx1);
      sMx[((j & 1) * 2 + h) * 128 + r] = tmax;
      bar_sync(3 + (warp & 3), 64);                                    // the two warps that share these 32 rows
      tmax = fmaxf(tmax, sMx[((j & 1) * 2 + (h ^ 1)) * 128 + r]);
      // online softmax bookkeeping (log2 domain): mt = qs * tmax is the block row max of s*log2e
      const float mt = qs * tmax;
      const float m_new = fmaxf(m_run, mt);
      const float ref = P_NORM == ROTATTN_NORM_ROWBLOCK ? mt : m_new;
      const float alpha = ex2_approx(m_run - m_new);                   // first block: exp2(-inf) = 0
      const float beta = P_NORM == ROTATTN_NORM_ROWBLOCK ? ex2_approx(mt - m_new) : 1.f;
      const float2 nref2 = make_float2(-ref, -ref);
      float2 ls0 = make_float2(0.f, 0.f), ls1 = make_float2(0.f, 0.f);
      uint32_t pw[16];
#pragma unroll
      for (int g = 0; g < 16; ++g) {
        const float2 e0 = ffma2(t2[2 * g], qs2, nref2), e1 = ffma2(t2[2 * g + 1], qs2, nref2);
        const float2 p0 = make_float2(ex2_approx(e0.x), ex2_approx(e0.y));
        const float2 p1 = make_float2(ex2_approx(e1.x), ex2_approx(e1.y));
        ls0 = fadd2(ls0, p0);
        ls1 = fadd2(ls1, p1);
        const float2 f0 = ffma2(p0, lev2, magic2), f1 = ffma2(p1, lev2, magic2);   // low byte = rne(LEVELS * p)
        const uint32_t lo = __byte_perm(__float_as_uint(f0.x), __float_as_uint(f0.y), 0x0040);
        const uint32_t hi = __byte_perm(__float_as_uint(f1.x), __float_as_uint(f1.y), 0x0040);
        pw[g] = __byte_perm(lo, hi, 0x5410);
      }
      if (DEBUG) {
#pragma unroll
        for (int g = 0; g < 16; ++g) *reinterpret_cast<uint32_t*>(a.P_dump + (size_t)r * a.npad + j * kTile + cb + g * 4) = pw[g];
      }
      tmem_st16(tmem_base + lane_off + TM_S + b * 128 + 16 * h, pw);   // u8 P tile aliases S columns [0,32)
      if (h == 0) sAB[(j % KS_RING) * 128 + r] = make_float2(alpha, beta * (kAccScale / LEVELS));
      l_run = alpha * l_run + beta * ((ls0.x + ls0.y) + (ls1.x + ls1.y));
      m_run = m_new;
      tmem_wait_st();
      tc_fence_before();
      mbar_arrive(&p_full[b]);
      if (h == 0) {
        mbar_arrive(&ab_full[j % KS_RING]);
        if (j + 1 < nblk) sKs[(b ^ 1) * 128 + r] = ks_next;
      }
    }
    sL[h * 128 + r] = l_run;
    mbar_arrive(l_full);
  } else {
    // ------------------------------------------------------------------ drain: 2 threads per query row of O
    asm volatile("setmaxnreg.inc.sync.aligned.u32 120;");
    constexpr int DH = D / 2;                      // channels per thread
    const int tdr = threadIdx.x - 384;
    const int h = tdr >> 7, r = tdr & 127;
    const int row = q0 + r;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    const float* vsrc = a.Vs + (size_t)bh * nblk * D;
    float2 o2[DH / 2];
#pragma unroll
    for (int d = 0; d < DH / 2; ++d) o2[d] = make_float2(0.f, 0.f);
    if (tdr < D) sVs[tdr] = vsrc[tdr];
    for (int j = 0; j < nblk; ++j) {
      const int b = j & 1;
      bar_sync(2, 256);
      float vs_next = 0.f;
      if (j + 1 < nblk && tdr < D) vs_next = vsrc[(size_t)(j + 1) * D + tdr];
      const float2* vsb2 = reinterpret_cast<const float2*>(sVs + b * D + h * DH);
      mbar_wait(&ab_full[j % KS_RING], (j / KS_RING) & 1);
      const float2 ab = sAB[(j % KS_RING) * 128 + r];
      mbar_wait(&pv_full[b], (j >> 1) & 1);
      tc_fence_after();
      const float2 c2 = make_float2(ab.y, ab.y), a2 = make_float2(ab.x, ab.x);
      const bool keep = __all_sync(0xffffffffu, ab.x == 1.f);          // no new row max in this warp's 32 rows
#pragma unroll
      for (int cc = 0; cc < DH / 32; ++cc) {
        uint32_t v[32];
        tmem_ld32(tmem_base + lane_off + TM_PV + b * 128 + h * DH + cc * 32, v);
        tmem_wait_ld();
        if (cc == DH / 32 - 1) {                                       // PV buffer is in registers now
          tc_fence_before();
          mbar_arrive(&pv_empty[b]);
        }
        if (keep) {
#pragma unroll
          for (int d = 0; d < 16; ++d) {
            const float2 y = fmul2(make_float2(__uint_as_float(v[2 * d]), __uint_as_float(v[2 * d + 1])), vsb2[cc * 16 + d]);
            o2[cc * 16 + d] = ffma2(y, c2, o2[cc * 16 + d]);           // O += (beta/levels) * pv * Vs[g][d]
          }
        } else {
#pragma unroll
          for (int d = 0; d < 16; ++d) {
            const float2 y = fmul2(make_float2(__uint_as_float(v[2 * d]), __uint_as_float(v[2 * d + 1])), vsb2[cc * 16 + d]);
            o2[cc * 16 + d] = ffma2(o2[cc * 16 + d], a2, fmul2(y, c2));   // O = alpha O + (beta/levels) * pv * Vs[g][d]
          }
        }
      }
      if (j + 1 < nblk && tdr < D) sVs[(b ^ 1) * D + tdr] = vs_next;
    }
    mbar_wait(l_full, 0);
    const float inv_l = 1.f / (sL[r] + sL[128 + r]);
    if (row < a.N) {
      __half* dst = (DEBUG ? a.O + (size_t)r * D : a.O + ((size_t)bh * a.N + row) * D) + h * DH;
#pragma unroll
      for (int d = 0; d < DH; d += 8) {
        __half2 hh[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) hh[i] = __floats2half2_rn(o2[d / 2 + i].x * inv_l, o2[d / 2 + i].y * inv_l);
        *reinterpret_cast<uint4*>(dst + d) = *reinterpret_cast<uint4*>(hh);
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem_base, 512);
}


template <int D, bool DEBUG>
static int launch_sync_variant(const rotattn_params& p, const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv,
                               const FwdInt4Args& a, dim3 grid, cudaStream_t cs) {
  constexpr int smem = SmemInt4Sync<D>::TOTAL;
#define ROTATTN_LAUNCH(PM, PN)                                                                                      \
  do {                                                                                                              \
    cudaFuncAttributes fa;                                                                                          \
    ROTATTN_CUDA_TRY(cudaFuncGetAttributes(&fa, fwd_int4_sync_kernel<D, PM, PN, DEBUG>));                           \
    if (fa.numRegs != 96) {       /* the setmaxnreg redistribution assumes a pool of 640 x 96 registers */          \
      set_error_text("fwd_int4_sync_kernel: unexpected register allocation (setmaxnreg pool assumes 96 per thread)"); \
      return ROTATTN_ERR_UNSUPPORTED;                                                                               \
    }                                                                                                               \
    ROTATTN_CUDA_TRY(cudaFuncSetAttribute(fwd_int4_sync_kernel<D, PM, PN, DEBUG>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)); \
    fwd_int4_sync_kernel<D, PM, PN, DEBUG><<<grid, kInt4Threads, smem, cs>>>(tq, tk, tv, a);                        \
  } while (0)
  if (p.p_mode == ROTATTN_P_ASYM15) ROTATTN_LAUNCH(ROTATTN_P_ASYM15, ROTATTN_NORM_RUNNING);
  else ROTATTN_LAUNCH(ROTATTN_P_SYM7, ROTATTN_NORM_RUNNING);
#undef ROTATTN_LAUNCH
  ROTATTN_CUDA_TRY(cudaGetLastError());
  return ROTATTN_OK;
}

int launch_fwd_int4_sync(const rotattn_params& p, const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv,
                         const FwdInt4Args& a, dim3 grid, bool debug, cudaStream_t cs) {
  if (p.D == 128) return debug ? launch_sync_variant<128, true>(p, tq, tk, tv, a, grid, cs) : launch_sync_variant<128, false>(p, tq, tk, tv, a, grid, cs);
  return debug ? launch_sync_variant<64, true>(p, tq, tk, tv, a, grid, cs) : launch_sync_variant<64, false>(p, tq, tk, tv, a, grid, cs);
}

}  // namespace rotattn
