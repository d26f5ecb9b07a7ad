// rotattn_fwd_int4 (steps a4-a9): INT4 FlashAttention forward on tcgen05 (kind::f8f6f4 on integer-exact E4M3 code
// bytes, see fwd_int4.cuh), row-block P normaliser.
//
// One CTA = one 128-row query tile of one (b,h); 28 warps, warp-specialised:
//   warp 0        TMA producer : Q tile once, K tiles (4-stage ring) and V^T tiles (3-stage ring)
//   warp 1        MMA issuer   : S = Q K^T (codes x codes, exact, TMEM), P~V (P codes from TMEM x V codes, TMEM)
//   warp 2        TMEM allocator, then V-scale loader (Vs[g][:] -> shared ring)
//   warp 3        K-scale loader (Ks[j] * 2^18 log2e/sqrt(D) -> shared ring)
//   warps 4-11    softmax group 0: even KV blocks; warps 4-7 own keys [0,64) of the block, warps 8-11 keys [64,128)
//   warps 12-19   softmax group 1: odd KV blocks, same split  (two threads per query row and block)
//   warps 20-27   drain: 2 threads per query row (D/2 channels each): online-softmax bookkeeping (m, l, alpha, beta),
//                 P~V block -> fp32 O registers, epilogue O/l
// With the row-block normaliser (reading 13) the codes of block j depend only on block j, so the two softmax
// groups work on different blocks concurrently and the running max lives in the drain threads.  Each softmax thread
// makes two passes over its half row of S in tensor memory (pass 1: block row max, exchanged with the partner thread
// through shared memory; pass 2: exp2 / row sum / codes) in 16-column chunks.
// TMEM (512 columns): S[2] at 0/128, PV at 256, four P-code slots of 32 columns at 384.  P has its own slots so that
// an S buffer is released as soon as pass 2 has read it (S(j+2) is issued before P~V(j), hiding the MMA latency).
// The per-block drain is forced by the method: beta (row, block) and Vs (channel, block) change every KV block
// (PAPER.md:L157 online softmax, L190 per-group V scales), so P~V cannot accumulate across blocks in tensor memory.
#include <cmath>
#include <cstdio>
#include "fwd_int4.cuh"

namespace rotattn {

constexpr int kFwdThreads = 896;
constexpr int K_STAGES = 4;
constexpr int V_STAGES = 3;
constexpr int P_SLOTS = 4;
constexpr int AB_RING = 8;
constexpr int KS_RING = 4;
constexpr int VS_RING = 4;

template <int D>
struct SmemInt4 {
  static constexpr int Q_BYTES = 128 * 128;
  static constexpr int K_BYTES = 128 * 128;
  static constexpr int V_BYTES = D * 128;
  static constexpr int OFF_Q = 0;
  static constexpr int OFF_K = OFF_Q + Q_BYTES;
  static constexpr int OFF_V = OFF_K + K_STAGES * K_BYTES;
  static constexpr int OFF_KS = OFF_V + V_STAGES * V_BYTES;           // float [KS_RING][128]
  static constexpr int OFF_VS = OFF_KS + KS_RING * 128 * 4;           // float [VS_RING][D]
  static constexpr int OFF_AB = OFF_VS + VS_RING * D * 4;             // float2 [AB_RING][2 halves][128]  (block max, half-row sum)
  static constexpr int OFF_MX = OFF_AB + AB_RING * 2 * 128 * 8;       // float [2 groups][2 parities][2 halves][128]
  static constexpr int OFF_BAR = OFF_MX + 2 * 2 * 2 * 128 * 4;        // mbarriers
  static constexpr int NBAR = 1 + 2 * K_STAGES + 2 * V_STAGES + 2 + 2 + 2 * P_SLOTS + 2 + AB_RING + 2 * KS_RING + 2 * VS_RING;
  static constexpr int OFF_TMEM = OFF_BAR + NBAR * 8;
  static constexpr int TOTAL = OFF_TMEM + 16;
};

// ---- per-chunk element-wise work of the softmax threads (16 S columns of one query row) -------------------------
// t = S * (Ks_j * 2^18 log2e/sqrt(D)) (the query scale Qs_i > 0 is applied after the max); keys >= N are masked to -inf.
template <bool MASK>
__device__ __forceinline__ void chunk_scale(const uint32_t (&v)[16], const float2* ks2, int nvalid_rel, float2 (&t2)[8]) {
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    t2[i] = fmul2(make_float2(__uint_as_float(v[2 * i]), __uint_as_float(v[2 * i + 1])), ks2[i]);
    if (MASK) {
      if (2 * i >= nvalid_rel) t2[i].x = -INFINITY;
      if (2 * i + 1 >= nvalid_rel) t2[i].y = -INFINITY;
    }
  }
}

template <bool MASK>
__device__ __forceinline__ void chunk_max(const uint32_t (&v)[16], const float2* ks2, int nvalid_rel, float& mx0, float& mx1) {
  float2 t2[8];
  chunk_scale<MASK>(v, ks2, nvalid_rel, t2);
#pragma unroll
  for (int i = 0; i < 8; i += 2) { mx0 = fmax3(mx0, t2[i].x, t2[i].y); mx1 = fmax3(mx1, t2[i + 1].x, t2[i + 1].y); }
}

// LEVELS * P^ = exp2(t * Qs_i - mt + log2(LEVELS)); codes u = rne(LEVELS * P^) taken from the low byte of
// (LEVELS * P^) + 1.5 * 2^23 (Eq.12 L166-168 with the fixed scale 15 / Eq.11 L161 with 7); four codes per TMEM column.
template <bool MASK>
__device__ __forceinline__ void chunk_exp(const uint32_t (&v)[16], const float2* ks2, int nvalid_rel, float2 qs2, float2 nref2,
                                          float2& ls0, float2& ls1, uint32_t (&pw)[4]) {
  const float2 magic2 = make_float2(12582912.f, 12582912.f);
  float2 t2[8];
  chunk_scale<MASK>(v, ks2, nvalid_rel, t2);
#pragma unroll
  for (int g = 0; g < 4; ++g) {
    const float2 e0 = ffma2(t2[2 * g], qs2, nref2), e1 = ffma2(t2[2 * g + 1], qs2, nref2);
    const float2 p0 = make_float2(ex2_approx(e0.x), ex2_approx(e0.y));
    const float2 p1 = make_float2(ex2_approx(e1.x), ex2_approx(e1.y));
    ls0 = fadd2(ls0, p0);
    ls1 = fadd2(ls1, p1);
    const float2 f0 = fadd2(p0, magic2), f1 = fadd2(p1, magic2);
    const uint32_t lo = __byte_perm(__float_as_uint(f0.x), __float_as_uint(f0.y), 0x0040);
    const uint32_t hi = __byte_perm(__float_as_uint(f1.x), __float_as_uint(f1.y), 0x0040);
    pw[g] = __byte_perm(lo, hi, 0x5410);
  }
}

template <int D, int P_MODE, bool DEBUG>
__global__ void __launch_bounds__(kFwdThreads, 1)
fwd_int4_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                const __grid_constant__ CUtensorMap tmV, const FwdInt4Args a) {
  using L = SmemInt4<D>;
  extern __shared__ __align__(1024) uint8_t smem[];      // no static shared memory in this kernel: base is 1024-aligned
  uint8_t* sQ = smem + L::OFF_Q;
  uint8_t* sK = smem + L::OFF_K;
  uint8_t* sV = smem + L::OFF_V;
  float* sKs = (float*)(smem + L::OFF_KS);
  float* sVs = (float*)(smem + L::OFF_VS);
  float2* sAB = (float2*)(smem + L::OFF_AB);
  float* sMx = (float*)(smem + L::OFF_MX);
  uint64_t* bars = (uint64_t*)(smem + L::OFF_BAR);
  uint64_t* q_full = bars;
  uint64_t* k_full = q_full + 1;
  uint64_t* k_empty = k_full + K_STAGES;
  uint64_t* v_full = k_empty + K_STAGES;
  uint64_t* v_empty = v_full + V_STAGES;
  uint64_t* s_full = v_empty + V_STAGES;      // [2] MMA -> softmax group (buffer b belongs to group b)
  uint64_t* s_empty = s_full + 2;             // [2] softmax group -> MMA (count 256): S buffer has been read
  uint64_t* p_full = s_empty + 2;             // [P_SLOTS] softmax group -> MMA (count 256)
  uint64_t* p_empty = p_full + P_SLOTS;       // [P_SLOTS] MMA -> softmax: P~V has consumed the slot
  uint64_t* pv_full = p_empty + P_SLOTS;      // MMA -> drain
  uint64_t* pv_empty = pv_full + 1;           // drain -> MMA (count 256)
  uint64_t* ab_full = pv_empty + 1;           // [AB_RING] softmax -> drain (count 256)
  uint64_t* ks_full = ab_full + AB_RING;      // [KS_RING] loader -> softmax (count 32)
  uint64_t* ks_empty = ks_full + KS_RING;     // [KS_RING] softmax -> loader (count 256)
  uint64_t* vs_full = ks_empty + KS_RING;     // [VS_RING] loader -> drain (count 32)
  uint64_t* vs_empty = vs_full + VS_RING;     // [VS_RING] drain -> loader (count 256)
  uint32_t* tmem_slot = (uint32_t*)(smem + L::OFF_TMEM);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int qtile = DEBUG ? a.dbg_qtile : blockIdx.x;
  const int bh = DEBUG ? a.dbg_bh : (a.head_sel ? a.head_sel[blockIdx.y] : (int)blockIdx.y);
  const int q0 = qtile * kTile;
  const int nblk = a.nblk;

  if (threadIdx.x == 0) {
    if (smem_u32(smem) & 1023u) __trap();     // SWIZZLE_128B operand tiles need 1024-byte alignment
    mbar_init(q_full, 1);
    for (int i = 0; i < K_STAGES; ++i) { mbar_init(&k_full[i], 1); mbar_init(&k_empty[i], 1); }
    for (int i = 0; i < V_STAGES; ++i) { mbar_init(&v_full[i], 1); mbar_init(&v_empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&s_full[i], 1); mbar_init(&s_empty[i], 256); }
    for (int i = 0; i < P_SLOTS; ++i) { mbar_init(&p_full[i], 256); mbar_init(&p_empty[i], 1); }
    mbar_init(pv_full, 1); mbar_init(pv_empty, 256);
    for (int i = 0; i < AB_RING; ++i) mbar_init(&ab_full[i], 256);
    for (int i = 0; i < KS_RING; ++i) { mbar_init(&ks_full[i], 32); mbar_init(&ks_empty[i], 256); }
    for (int i = 0; i < VS_RING; ++i) { mbar_init(&vs_full[i], 32); mbar_init(&vs_empty[i], 256); }
    fence_mbar_init();
  }
  if (warp == 2) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  constexpr uint32_t TM_S = 0, TM_PV = 256, TM_P = 384;

  // register pool of the CTA = 896 x 72; after redistribution 128 x 24 + 512 x 72 + 256 x 96 = 64512 (exactly the pool)
  if (warp < 4) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
    if (warp == 0) {
      // ---------------------------------------------------------------- TMA producer
      if (lane == 0) {
        tma_prefetch_desc(&tmQ); tma_prefetch_desc(&tmK); tma_prefetch_desc(&tmV);
        mbar_arrive_expect_tx(q_full, L::Q_BYTES);
        tma_load_3d(sQ, &tmQ, q_full, 0, q0, bh);
        auto load_k = [&](int m) {
          const int s = m % K_STAGES;
          mbar_wait(&k_empty[s], ((m / K_STAGES) & 1) ^ 1);
          mbar_arrive_expect_tx(&k_full[s], L::K_BYTES);
          tma_load_3d(sK + s * L::K_BYTES, &tmK, &k_full[s], 0, m * kTile, bh);
        };
        load_k(0);
        if (nblk > 1) load_k(1);
        for (int j = 0; j < nblk; ++j) {
          if (j + 2 < nblk) load_k(j + 2);
          const int s = j % V_STAGES;
          mbar_wait(&v_empty[s], ((j / V_STAGES) & 1) ^ 1);
          mbar_arrive_expect_tx(&v_full[s], L::V_BYTES);
          tma_load_3d(sV + s * L::V_BYTES, &tmV, &v_full[s], j * kTile, 0, bh);
        }
      }
    } else if (warp == 1) {
      // ---------------------------------------------------------------- MMA issuer
      if (lane == 0) {
        constexpr uint32_t idesc_s = umma_idesc(1, 0, 0, 128, 128);      // f32 <- e4m3 x e4m3 (integer codes * 2^-9)
        constexpr uint32_t idesc_pv = umma_idesc(1, 0, 0, 128, D);
        constexpr int KSTEPS_S = D / 32;                                 // D=64 rows are zero-padded to 128 B
        const uint64_t qd = umma_desc_k128(smem_u32(sQ));
        auto issue_s = [&](int m) {                                      // S(m) -> buffer m & 1
          const int st = m % K_STAGES, b = m & 1;
          mbar_wait(&k_full[st], (m / K_STAGES) & 1);
          if (m >= 2) mbar_wait(&s_empty[b], ((m >> 1) - 1) & 1);        // softmax has read S(m-2) out of this buffer
          tc_fence_after();
          const uint64_t kd = umma_desc_k128(smem_u32(sK + st * L::K_BYTES));
#pragma unroll
          for (int k = 0; k < KSTEPS_S; ++k)
            mma_ss<MmaKind::F8F6F4>(tmem_base + TM_S + b * 128, qd + 2 * k, kd + 2 * k, idesc_s, k != 0);
          tc_commit(&k_empty[st]);
          tc_commit(&s_full[b]);
        };
        mbar_wait(q_full, 0);
        issue_s(0);
        if (nblk > 1) issue_s(1);
        for (int j = 0; j < nblk; ++j) {
          if (j + 2 < nblk) issue_s(j + 2);                              // goes ahead of P~V(j): only needs S(j) to be read
          const int slot = j % P_SLOTS, vst = j % V_STAGES;
          mbar_wait(&p_full[slot], (j / P_SLOTS) & 1);
          mbar_wait(&v_full[vst], (j / V_STAGES) & 1);
          mbar_wait(pv_empty, (j & 1) ^ 1);
          tc_fence_after();
          const uint64_t vd = umma_desc_k128(smem_u32(sV + vst * L::V_BYTES));
#pragma unroll
          for (int k = 0; k < 4; ++k)
            mma_ts<MmaKind::F8F6F4>(tmem_base + TM_PV, tmem_base + TM_P + slot * 32 + 8 * k, vd + 2 * k, idesc_pv, k != 0);
          tc_commit(&v_empty[vst]);
          tc_commit(&p_empty[slot]);
          tc_commit(pv_full);
        }
      }
    } else if (warp == 2) {
      // ---------------------------------------------------------------- V-scale loader
      const float* vsrc = a.Vs + (size_t)bh * nblk * D;
      for (int j = 0; j < nblk; ++j) {
        const int s = j % VS_RING;
        mbar_wait(&vs_empty[s], ((j / VS_RING) & 1) ^ 1);
#pragma unroll
        for (int i = 0; i < D / 32; ++i) sVs[s * D + i * 32 + lane] = vsrc[(size_t)j * D + i * 32 + lane];
        mbar_arrive(&vs_full[s]);
      }
    } else {
      // ---------------------------------------------------------------- K-scale loader: Ks_j * 2^18 log2e/sqrt(D)
      const float* ksrc = a.Ks + (size_t)bh * a.N;
      for (int j = 0; j < nblk; ++j) {
        const int s = j % KS_RING;
        mbar_wait(&ks_empty[s], ((j / KS_RING) & 1) ^ 1);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int kj = j * kTile + i * 32 + lane;
          sKs[s * 128 + i * 32 + lane] = (kj < a.N) ? ksrc[kj] * a.scale_log2 : 0.f;
        }
        mbar_arrive(&ks_full[s]);
      }
    }
  } else if (warp < 20) {
    // ------------------------------------------------------------------ softmax groups: 0 = even blocks, 1 = odd blocks
    constexpr float LOG2_LEVELS = P_MODE == ROTATTN_P_ASYM15 ? 3.9068905956085187f : 2.8073549220576042f;
    const int tsm = threadIdx.x - 128;
    const int g = tsm >> 8;                          // group index = S buffer index
    const int h = (tsm >> 7) & 1;                    // which 64 keys of the block
    const int r = tsm & 127;
    const int row = q0 + r;
    const int cb = 64 * h;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    // qs >= 1e-30 keeps (-inf) * qs well defined for masked keys; an all-zero query row still gives s == 0 everywhere
    const float qs = (row < a.N) ? fmaxf(a.Qs[(size_t)bh * a.N + row], 1e-30f) : 1e-30f;
    const float2 qs2 = make_float2(qs, qs);
    const uint32_t s_addr = tmem_base + lane_off + TM_S + g * 128 + cb;
    const int pair_bar = 1 + 4 * g + (warp & 3);     // named barrier of the two warps that share these 32 rows
    for (int j = g; j < nblk; j += 2) {
      const int n = j >> 1;
      const int ring = j % KS_RING, slot = j % P_SLOTS, abslot = j % AB_RING;
      const float2* ks2 = reinterpret_cast<const float2*>(sKs + ring * 128 + cb);
      const int nvalid = min(kTile, a.N - j * kTile) - cb;   // valid keys of this half; < 64 only on the ragged last block
      const bool ragged = nvalid < 64;
      mbar_wait(&ks_full[ring], (j / KS_RING) & 1);
      mbar_wait(&s_full[g], n & 1);
      tc_fence_after();
      uint32_t va[16], vb[16];
      // ---- pass 1: block row max over this half
      float mx0 = -INFINITY, mx1 = -INFINITY;
      tmem_ld16(s_addr, va);
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        tmem_wait_ld();
        uint32_t(&cur)[16] = (c & 1) ? vb : va;
        uint32_t(&nxt)[16] = (c & 1) ? va : vb;
        tmem_ld16(s_addr + ((c + 1) & 3) * 16, nxt);     // chunk c+1 (after chunk 3: chunk 0 again, for pass 2)
        if (ragged) chunk_max<true>(cur, ks2 + c * 8, nvalid - c * 16, mx0, mx1);
        else chunk_max<false>(cur, ks2 + c * 8, 16, mx0, mx1);
      }
      float tmax = fmaxf(mx0, mx1);
      float* mxbuf = sMx + ((g * 2 + (n & 1)) * 2) * 128;
      mxbuf[h * 128 + r] = tmax;
      bar_sync(pair_bar, 64);
      tmax = fmaxf(tmax, mxbuf[(h ^ 1) * 128 + r]);
      const float mt = qs * tmax;                        // block row max of s * log2e
      const float nref = LOG2_LEVELS - mt;
      const float2 nref2 = make_float2(nref, nref);
      mbar_wait(&p_empty[slot], ((j / P_SLOTS) & 1) ^ 1);
      // ---- pass 2: LEVELS * P^, row sum, codes -> u8 P tile slot
      float2 ls0 = make_float2(0.f, 0.f), ls1 = make_float2(0.f, 0.f);
      const uint32_t p_addr = tmem_base + lane_off + TM_P + slot * 32 + 16 * h;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        tmem_wait_ld();
        uint32_t(&cur)[16] = (c & 1) ? vb : va;
        uint32_t(&nxt)[16] = (c & 1) ? va : vb;
        if (c < 3) tmem_ld16(s_addr + (c + 1) * 16, nxt);
        else { tc_fence_before(); mbar_arrive(&s_empty[g]); }          // this thread is done with the S buffer
        if (DEBUG) {
#pragma unroll
          for (int i = 0; i < 16; ++i)
            a.S_dump[(size_t)r * a.npad + j * kTile + cb + c * 16 + i] = (int32_t)(__uint_as_float(cur[i]) * kAccScale);
        }
        uint32_t pw[4];
        if (ragged) chunk_exp<true>(cur, ks2 + c * 8, nvalid - c * 16, qs2, nref2, ls0, ls1, pw);
        else chunk_exp<false>(cur, ks2 + c * 8, 16, qs2, nref2, ls0, ls1, pw);
        if (DEBUG) {
#pragma unroll
          for (int q = 0; q < 4; ++q) *reinterpret_cast<uint32_t*>(a.P_dump + (size_t)r * a.npad + j * kTile + cb + c * 16 + q * 4) = pw[q];
        }
        tmem_st4(p_addr + c * 4, pw);
      }
      sAB[(abslot * 2 + h) * 128 + r] = make_float2(mt, (ls0.x + ls0.y) + (ls1.x + ls1.y));
      tmem_wait_st();
      tc_fence_before();
      mbar_arrive(&p_full[slot]);
      mbar_arrive(&ab_full[abslot]);
      mbar_arrive(&ks_empty[ring]);
    }
  } else {
    // ------------------------------------------------------------------ drain: 2 threads per query row of O
    asm volatile("setmaxnreg.inc.sync.aligned.u32 96;");
    constexpr int DH = D / 2;                      // channels per thread
    const int tdr = threadIdx.x - 640;
    const int h = tdr >> 7, r = tdr & 127;
    const int row = q0 + r;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    float2 o2[DH / 2];
#pragma unroll
    for (int d = 0; d < DH / 2; ++d) o2[d] = make_float2(0.f, 0.f);
    float m_run = -INFINITY, l_run = 0.f;
    for (int j = 0; j < nblk; ++j) {
      // online softmax bookkeeping (L157): m' = max(m, mt); alpha = exp(m - m'); beta = exp(mt - m'); l = alpha l + beta sum(P^)
      const int abslot = j % AB_RING;
      mbar_wait(&ab_full[abslot], (j / AB_RING) & 1);
      const float2 ms0 = sAB[(abslot * 2 + 0) * 128 + r], ms1 = sAB[(abslot * 2 + 1) * 128 + r];
      const float m_new = fmaxf(m_run, ms0.x);
      const float alpha = ex2_approx(m_run - m_new);                   // first block: exp2(-inf) = 0
      const float beta = ex2_approx(ms0.x - m_new);
      l_run = alpha * l_run + beta * (ms0.y + ms1.y);                  // in units of LEVELS (cancels in O/l)
      m_run = m_new;
      const float cf = beta * kAccScale;                               // undoes the 2^-18 of the E4M3 code products
      const float2 c2 = make_float2(cf, cf), a2 = make_float2(alpha, alpha);
      const bool keep = __all_sync(0xffffffffu, alpha == 1.f);         // no new row max in this warp's 32 rows
      const int vring = j % VS_RING;
      mbar_wait(&vs_full[vring], (j / VS_RING) & 1);
      const float2* vsb2 = reinterpret_cast<const float2*>(sVs + vring * D + h * DH);
      mbar_wait(pv_full, j & 1);
      tc_fence_after();
#pragma unroll
      for (int cc = 0; cc < DH / 16; ++cc) {
        uint32_t v[16];
        tmem_ld16(tmem_base + lane_off + TM_PV + h * DH + cc * 16, v);
        tmem_wait_ld();
        if (cc == DH / 16 - 1) {                                       // PV buffer is in registers now
          tc_fence_before();
          mbar_arrive(pv_empty);
        }
        if (keep) {
#pragma unroll
          for (int d = 0; d < 8; ++d) {
            const float2 y = fmul2(make_float2(__uint_as_float(v[2 * d]), __uint_as_float(v[2 * d + 1])), vsb2[cc * 8 + d]);
            o2[cc * 8 + d] = ffma2(y, c2, o2[cc * 8 + d]);             // O += beta * pv * Vs[g][d]
          }
        } else {
#pragma unroll
          for (int d = 0; d < 8; ++d) {
            const float2 y = fmul2(make_float2(__uint_as_float(v[2 * d]), __uint_as_float(v[2 * d + 1])), vsb2[cc * 8 + d]);
            o2[cc * 8 + d] = ffma2(o2[cc * 8 + d], a2, fmul2(y, c2));  // O = alpha O + beta * pv * Vs[g][d]
          }
        }
      }
      mbar_arrive(&vs_empty[vring]);
    }
    const float inv_l = 1.f / l_run;
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

}  // namespace rotattn

using namespace rotattn;

namespace {

template <int D, bool DEBUG>
int launch_variant(const rotattn_params& p, const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv,
                   const FwdInt4Args& a, dim3 grid, cudaStream_t cs) {
  constexpr int smem = SmemInt4<D>::TOTAL;
  if (p.p_mode == ROTATTN_P_ASYM15) {
    ROTATTN_CUDA_TRY(cudaFuncSetAttribute(fwd_int4_kernel<D, ROTATTN_P_ASYM15, DEBUG>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    fwd_int4_kernel<D, ROTATTN_P_ASYM15, DEBUG><<<grid, kFwdThreads, smem, cs>>>(tq, tk, tv, a);
  } else {
    ROTATTN_CUDA_TRY(cudaFuncSetAttribute(fwd_int4_kernel<D, ROTATTN_P_SYM7, DEBUG>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    fwd_int4_kernel<D, ROTATTN_P_SYM7, DEBUG><<<grid, kFwdThreads, smem, cs>>>(tq, tk, tv, a);
  }
  ROTATTN_CUDA_TRY(cudaGetLastError());
  return ROTATTN_OK;
}

int fwd_int4_common(const rotattn_params* p, const uint8_t* Q4, const float* Qs, const uint8_t* K4, const float* Ks,
                    const uint8_t* V4, const float* Vs, void* O, const int32_t* head_sel, int32_t n_sel,
                    void* workspace, size_t ws_bytes, int32_t ws_state, void* stream,
                    bool debug, int32_t bh, int32_t q_tile, int32_t* S_dump, uint8_t* P_dump) {
  int st = rotattn_validate(p);
  if (st != ROTATTN_OK) return st;
  if (!Q4 || !Qs || !K4 || !Ks || !V4 || !Vs || !O || !workspace) return ROTATTN_ERR_INVALID_ARG;
  const int BH = p->B * p->H;
  const int nblk = ceil_div(p->N, kTile);
  if (head_sel && (n_sel < 1 || n_sel > BH)) return ROTATTN_ERR_INVALID_ARG;
  if (debug && (bh < 0 || bh >= BH || q_tile < 0 || q_tile >= nblk || !S_dump || !P_dump)) return ROTATTN_ERR_INVALID_ARG;
  WsInt4 ws(*p);
  if (ws_bytes < ws.total) return ROTATTN_ERR_WORKSPACE_TOO_SMALL;
  if ((st = check_device_sm100()) != ROTATTN_OK) return st;
  cudaStream_t cs = (cudaStream_t)stream;
  int8_t* q8 = (int8_t*)workspace + ws.q8;
  int8_t* k8 = (int8_t*)workspace + ws.k8;
  int8_t* v8t = (int8_t*)workspace + ws.v8t;
  if (!(ws_state & ROTATTN_WS_HAS_QK)) {
    if ((st = launch_unpack_qk(*p, Q4, q8, cs)) != ROTATTN_OK) return st;
    if ((st = launch_unpack_qk(*p, K4, k8, cs)) != ROTATTN_OK) return st;
  }
  if (!(ws_state & ROTATTN_WS_HAS_V)) {
    if ((st = launch_unpack_vt(*p, V4, v8t, ws.npad, cs)) != ROTATTN_OK) return st;
  }
  CUtensorMap tq, tk, tv;
  const uint64_t N = p->N, D = p->D;
  if ((st = make_tmap_3d(&tq, q8, 1, kQKRowBytes, N, BH, kQKRowBytes, N * kQKRowBytes, 128, 128)) != ROTATTN_OK) return st;
  if ((st = make_tmap_3d(&tk, k8, 1, kQKRowBytes, N, BH, kQKRowBytes, N * kQKRowBytes, 128, 128)) != ROTATTN_OK) return st;
  if ((st = make_tmap_3d(&tv, v8t, 1, ws.npad, D, BH, ws.npad, D * ws.npad, 128, (uint32_t)D)) != ROTATTN_OK) return st;
  FwdInt4Args a{};
  a.Qs = Qs; a.Ks = Ks; a.Vs = Vs; a.O = (__half*)O; a.head_sel = head_sel;
  a.S_dump = S_dump; a.P_dump = P_dump;
  a.N = p->N; a.nblk = nblk; a.npad = ws.npad; a.dbg_bh = bh; a.dbg_qtile = q_tile;
  a.scale_log2 = (float)(1.4426950408889634 / std::sqrt((double)p->D) * (double)kAccScale);   // S arrives as acc * 2^-18
  dim3 grid(debug ? 1 : nblk, debug ? 1 : (head_sel ? n_sel : BH));
  if (p->p_norm == ROTATTN_NORM_RUNNING) return launch_fwd_int4_sync(*p, tq, tk, tv, a, grid, debug, cs);
  if (p->D == 128) return debug ? launch_variant<128, true>(*p, tq, tk, tv, a, grid, cs) : launch_variant<128, false>(*p, tq, tk, tv, a, grid, cs);
  return debug ? launch_variant<64, true>(*p, tq, tk, tv, a, grid, cs) : launch_variant<64, false>(*p, tq, tk, tv, a, grid, cs);
}

}  // namespace

extern "C" int rotattn_fwd_int4(const rotattn_params* p, const uint8_t* Q4, const float* Qs, const uint8_t* K4,
                                const float* Ks, const uint8_t* V4, const float* Vs, void* O, const int32_t* head_sel,
                                int32_t n_sel, void* workspace, size_t ws_bytes, int32_t ws_state, void* stream) {
  return fwd_int4_common(p, Q4, Qs, K4, Ks, V4, Vs, O, head_sel, n_sel, workspace, ws_bytes, ws_state, stream,
                         false, 0, 0, nullptr, nullptr);
}

extern "C" int rotattn_fwd_int4_debug(const rotattn_params* p, const uint8_t* Q4, const float* Qs, const uint8_t* K4,
                                      const float* Ks, const uint8_t* V4, const float* Vs, int32_t bh, int32_t q_tile,
                                      int32_t* S_dump, uint8_t* P_dump, void* O_tile, void* workspace, size_t ws_bytes,
                                      int32_t ws_state, void* stream) {
  return fwd_int4_common(p, Q4, Qs, K4, Ks, V4, Vs, O_tile, nullptr, 0, workspace, ws_bytes, ws_state, stream,
                         true, bh, q_tile, S_dump, P_dump);
}
