// fwd_int4_kernel (steps a4-a9): INT4 FlashAttention forward on tcgen05 (kind::f8f6f4 on integer-exact E4M3 code
// bytes, see fwd_int4.cuh), row-block P normaliser (reading 13).
//
// One CTA = one 128-row query tile of one (b,h); 16 warps, warp-specialised, ONE THREAD PER QUERY ROW in every
// element-wise role (the tcgen05.ld 32x32b shape gives a thread its whole row, so no row reduction crosses threads):
//   warps 0-3     softmax group 0: even KV blocks.  The thread reads the 128 accumulators of its row of S into
//                 registers with one wait, releases the S buffer at once, and then works from registers only:
//                 key scales + block row max, exp2 / row sum / codes, codes -> shared-memory P tile
//   warps 4-7     softmax group 1: odd KV blocks, same code
//   warps 8-11    drain: online-softmax bookkeeping (m, l, alpha, beta), P~V block -> fp32 O registers, epilogue O/l
//   warp 12       TMEM allocator
//   warp 13       TMA producer  : Q tile once, K tiles (4-stage ring) and V^T tiles (3-stage ring); with them the key
//                 scales of the block and Vs[g][:] as 512-byte bulk copies into 8-deep shared rings
//   warp 14       MMA issuer 2  : P~V (P codes x V codes, both from shared memory, TMEM accumulators)
//   warp 15       MMA issuer 1  : S = Q K^T (codes x codes, exact, TMEM)
// With the row-block normaliser the codes of block j depend only on block j, so the two softmax groups work on
// different blocks concurrently and the running max lives in the drain threads.  Each SM sub-partition hosts one warp
// of each softmax group, one drain warp and one service warp; the exponentials (16 per clock and SM) are the busiest
// pipe, and the two softmax warps of a sub-partition keep it fed in turn: while one is in its load / scale / max phase
// the other is in its exp2 phase (per-token variants: enforced by a token passed through two named barriers per pair of
// warps; the per-block variants, whose non-exp2 phase is short, run free - DESIGN.md section 12 has the measurements).
// Registers: 512 x 128 at launch, redistributed by setmaxnreg to 24 (service) / 152 (softmax) / 184 (drain).
// Template switches (PAPER.md:L190 granularity; all parity-tested against the same oracle flags):
//   QKG = 1   per-token Q/K scales (the paper's setting): t = S * Ks_j in registers, block row max, e = t * Qs_i - ref
//   QKG = 128 one Q scale per query tile and one K scale per KV block: bare max over the raw accumulators (no multiply,
//             no key-scale ring); the scalar folds into the exp2 argument.
//   VSC = 0   one V scale per (128-token group, channel) (reading 11): drain = multiply + fma per element pair
//   VSC = 1   one V scale per 128-token group: the scalar folds into beta, drain = one fma per element pair.
//   SM = 1    smoothing (f2): t = S * Ks_j * Qs_i + kc_j with the per-key rank-1 correction, mean(V) added in the epilogue
// TMEM (512 columns): S[2] at 0/128 and four half-width (D/2 channels) P~V accumulators of 64 columns at 256 (block
// parity x channel half), so that the P~V MMAs run a block ahead of the drain instead of alternating with it.  The u8 P
// codes go to four shared-memory tiles (128-byte swizzle, A operand from shared memory).
// The per-block drain is forced by the method: beta (row, block) and Vs (channel, block) change every KV block
// (PAPER.md:L157 online softmax, L190 per-group V scales), so P~V cannot accumulate across blocks in tensor memory.
// Keys >= N (ragged last block): the softmax thread first overwrites those columns of its S row with -inf in tensor
// memory (a rolled loop, executed once per CTA), so the common path carries no mask; the padded key scales are 1
// (written by prepare_qk / pad_ks into the workspace copy KsP [BH, npad] the bulk copies read).
#pragma once
#include <cmath>
#include <cstdio>
#include <type_traits>
#include "fwd_int4.cuh"

namespace rotattn {

// Warp roles (role indices; the map from physical warps to roles is in the kernel, it depends on the variant).
constexpr int kWarpDrain = 8, kWarpAlloc = 12, kWarpTma = 13, kWarpMmaPV = 14, kWarpMmaS = 15;
constexpr int K_STAGES = 4;
constexpr int V_STAGES = 3;
constexpr int P_SLOTS = 4;       // P-code tiles in shared memory (A operand of the P~V MMA)
constexpr int PV_BUFS = 4;       // half-width (D/2 channel) P~V accumulators in rotation: buffer 2 * (j & 1) + h
constexpr int AB_RING = 8;
constexpr int KS_RING = 8;       // key-scale blocks in flight (bulk copies issued with the K tiles, released by the softmax threads)
constexpr int VS_RING = 8;
constexpr int RUN_RING = 4;      // p_norm = RUNNING: running row maxima handed from block j to block j + 1 (the other softmax group)
static_assert(K_STAGES == 4 && P_SLOTS == 4 && PV_BUFS == 4 && V_STAGES <= P_SLOTS, "ring sizes are tied together by the shared completion barriers");

template <int D>
struct SmemInt4 {
  static constexpr int Q_BYTES = 128 * 128;
  static constexpr int K_BYTES = 128 * 128;
  static constexpr int V_BYTES = D * 128;
  static constexpr int OFF_Q = 0;
  static constexpr int OFF_K = OFF_Q + Q_BYTES;
  static constexpr int OFF_V = OFF_K + K_STAGES * K_BYTES;
  static constexpr int P_BYTES = 128 * 128;                           // u8 codes [128 query rows][128 keys], 128-byte swizzle
  static constexpr int OFF_P = OFF_V + V_STAGES * V_BYTES;
  static constexpr int OFF_KS = OFF_P + P_SLOTS * P_BYTES;            // float [KS_RING][128]
  static constexpr int OFF_KC = OFF_KS + KS_RING * 128 * 4;           // float [KS_RING][128]  smoothing: per-key correction
  static constexpr int OFF_VS = OFF_KC + KS_RING * 128 * 4;           // float [VS_RING][D]
  static constexpr int OFF_AB = OFF_VS + VS_RING * D * 4;             // float [AB_RING][2][128]: block max, block row sum
  static constexpr int OFF_RUN = OFF_AB + AB_RING * 2 * 128 * 4;      // float [RUN_RING][128]  p_norm = RUNNING: running row max after block j
  static constexpr int OFF_BAR = OFF_RUN + RUN_RING * 128 * 4;        // mbarriers
  static constexpr int NBAR = 1 + 2 * K_STAGES + V_STAGES + 2 + 2 * P_SLOTS + 2 * PV_BUFS + AB_RING + 2 * KS_RING + 2 * VS_RING + RUN_RING;
  static constexpr int OFF_TMEM = OFF_BAR + NBAR * 8;
  static constexpr int TOTAL = OFF_TMEM + 16;
};

// exp2 of a pair on the FMA pipe instead of the exp2 unit (MUFU.EX2 issues one warp instruction per 8 clk; where the
// exp2 unit is the limiter a share of the exponentials is cheaper as arithmetic).  Cody-Waite: x = n + f with n = rne(x)
// taken from the low mantissa bits of x + 1.5 * 2^23, f in [-0.5, 0.5]; 2^f by a minimax polynomial in relative error
// (degree 4: 2.7e-6, degree 3: 7.5e-5, evaluated in fp32); 2^n by adding n to the exponent field.  Valid for
// -125 <= x < 128; smaller arguments (masked keys carry -inf) are clamped, 2^-125 is 0 for every later use.
#ifndef ROTATTN_POLY_DEG
#define ROTATTN_POLY_DEG 3
#endif
__device__ __forceinline__ float2 ex2_fma_pipe2(float2 x) {
  x.x = fmaxf(x.x, -125.f);
  x.y = fmaxf(x.y, -125.f);
  const float2 magic = make_float2(12582912.f, 12582912.f);
  const float2 t = fadd2(x, magic);
  const float2 n = fadd2(t, make_float2(-12582912.f, -12582912.f));
  const float2 fr = ffma2(n, make_float2(-1.f, -1.f), x);
#if ROTATTN_POLY_DEG == 4
  float2 p = ffma2(make_float2(9.570101276e-03f, 9.570101276e-03f), fr, make_float2(5.591785908e-02f, 5.591785908e-02f));
  p = ffma2(p, fr, make_float2(2.402474433e-01f, 2.402474433e-01f));
  p = ffma2(p, fr, make_float2(6.931217909e-01f, 6.931217909e-01f));
  p = ffma2(p, fr, make_float2(9.999992847e-01f, 9.999992847e-01f));
#else
  float2 p = ffma2(make_float2(5.517166480e-02f, 5.517166480e-02f), fr, make_float2(2.426111251e-01f, 2.426111251e-01f));
  p = ffma2(p, fr, make_float2(6.932609677e-01f, 6.932609677e-01f));
  p = ffma2(p, fr, make_float2(9.999280572e-01f, 9.999280572e-01f));
#endif
  return make_float2(__uint_as_float(__float_as_uint(p.x) + (__float_as_uint(t.x) << 23)),
                     __uint_as_float(__float_as_uint(p.y) + (__float_as_uint(t.y) << 23)));
}
// Pairs per 16 keys (of 8) that take the FMA-pipe route.  Measured on cfg 2 (B200, round 3, ms per call):
//   qk_group = 128 + v_scale = GROUP (the only variant the exp2 unit limits):
//     0: 4.276   1 (deg 3): 4.159   2 (deg 3): 4.145 <- shipped   3 (deg 3): 4.430   4 (deg 3): 4.698   1 (deg 4): 4.171   2 (deg 4): 4.347
//   qk_group = 128, per-channel V scales: 0: 4.514   1 (deg 4): 4.782   2 (deg 4): 4.989     (the drain's V-scale arithmetic already loads the FMA pipe)
//   per-token Q/K scales: 0: 4.986 / 4.741 (v_scale = GROUP)   1 (deg 4): 5.015 / 4.703
// so only the first gets it.  Degree 3 moves a P code by +-1 where LEVELS * P^ lies within ~1e-3 of a rounding boundary; the
// parity tests hold the per-tile mismatch rate of this variant to the same 0.1 % as every other.
#ifndef ROTATTN_POLY_BLOCK
#define ROTATTN_POLY_BLOCK 2
#endif
#ifndef ROTATTN_POLY_BLOCK_VCH
#define ROTATTN_POLY_BLOCK_VCH 0
#endif
#ifndef ROTATTN_POLY_TOKEN
#define ROTATTN_POLY_TOKEN 0
#endif

template <int D, int P_MODE, int QKG, int VSC, int SM, int PN, bool DEBUG>
__global__ void __launch_bounds__(kFwdThreads, 1)
fwd_int4_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                const __grid_constant__ CUtensorMap tmV, const FwdInt4Args a) {
  using L = SmemInt4<D>;
  // Per-token variants: the softmax warps of a sub-partition alternate in the exp2 phase (token; measured on cfg 2:
  // 5.15 -> 4.98 ms; the per-block variants are faster without it).
  constexpr bool TOKEN = QKG == 1;
  constexpr int kRegSoftmax = 152, kRegDrain = (65536 - 128 * 24 - 256 * kRegSoftmax) / 128;
  extern __shared__ __align__(1024) uint8_t smem[];      // no static shared memory in this kernel: base is 1024-aligned
  uint8_t* sQ = smem + L::OFF_Q;
  uint8_t* sK = smem + L::OFF_K;
  uint8_t* sV = smem + L::OFF_V;
  uint8_t* sP = smem + L::OFF_P;
  float* sKs = (float*)(smem + L::OFF_KS);
  float* sKc = (float*)(smem + L::OFF_KC);
  float* sVs = (float*)(smem + L::OFF_VS);
  float* sAB = (float*)(smem + L::OFF_AB);
  float* sRun = (float*)(smem + L::OFF_RUN);
  uint64_t* bars = (uint64_t*)(smem + L::OFF_BAR);
  uint64_t* q_full = bars;
  uint64_t* k_full = q_full + 1;              // [K_STAGES] TMA -> MMA
  uint64_t* v_full = k_full + K_STAGES;       // [V_STAGES] TMA -> MMA
  uint64_t* s_done = v_full + V_STAGES;       // [K_STAGES] S(m) complete: -> softmax group m & 1 (S ready), -> TMA (K stage free)
  uint64_t* s_empty = s_done + K_STAGES;      // [2] softmax group -> MMA (count 128): S buffer is in registers
  uint64_t* p_full = s_empty + 2;             // [P_SLOTS] softmax group -> MMA (count 128)
  uint64_t* pv_done = p_full + P_SLOTS;       // [P_SLOTS] both halves of P~V(j) complete: -> softmax (P slot free), TMA (V stage free)
  uint64_t* pvh_done = pv_done + P_SLOTS;     // [PV_BUFS] half k = 2j+h of P~V complete -> drain
  uint64_t* pvh_empty = pvh_done + PV_BUFS;   // [PV_BUFS] drain -> MMA (count 128): half buffer is in registers
  uint64_t* ab_full = pvh_empty + PV_BUFS;    // [AB_RING] softmax -> drain (count 128)
  uint64_t* ks_full = ab_full + AB_RING;      // [KS_RING] bulk copy of the key scales of a block -> softmax
  uint64_t* ks_empty = ks_full + KS_RING;     // [KS_RING] softmax -> TMA producer (count 128)
  uint64_t* vs_full = ks_empty + KS_RING;     // [VS_RING] bulk copy of Vs[g][:] -> drain
  uint64_t* vs_empty = vs_full + VS_RING;     // [VS_RING] drain -> TMA producer (count 128)
  uint64_t* run_full = vs_empty + VS_RING;    // [RUN_RING] softmax(j) -> softmax(j + 1) (count 128): running max after block j
  uint32_t* tmem_slot = (uint32_t*)(smem + L::OFF_TMEM);

  // Role of a warp.  Within an SM sub-partition the scheduler favours the highest warp id among the eligible warps.  The
  // per-token variants keep the service warps on the highest ids (with them on the lowest the kernel is 22 % slower: the
  // latency from an arrival to the MMA issue is on its critical path); the per-block variants, whose softmax warps wait
  // less, are 2-3 % faster with the softmax warps on top (physical warps 0-3 service, 4-7 drain, 8-15 softmax).  Roles
  // move in whole warp quads, so the TMEM lane quarter of a warp (warp % 4) is the same in both maps.
  const int pwarp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);  // warp-uniform (kept in a uniform register)
  const int warp = QKG == 1 ? pwarp : (pwarp < 4 ? pwarp + 12 : (pwarp < 8 ? pwarp + 4 : pwarp - 8));
  const int lane = threadIdx.x & 31;
  const int qtile = DEBUG ? a.dbg_qtile : blockIdx.x;
  const int bh = DEBUG ? a.dbg_bh : (a.head_sel ? a.head_sel[blockIdx.y] : (int)blockIdx.y);
  const int q0 = qtile * kTile;
  const int nblk = a.nblk;

  if (threadIdx.x == 0) {
    if (smem_u32(smem) & 1023u) __trap();     // SWIZZLE_128B operand tiles need 1024-byte alignment
    mbar_init(q_full, 1);
    for (int i = 0; i < K_STAGES; ++i) { mbar_init(&k_full[i], 1); mbar_init(&s_done[i], 1); }
    for (int i = 0; i < V_STAGES; ++i) mbar_init(&v_full[i], 1);
    for (int i = 0; i < 2; ++i) mbar_init(&s_empty[i], 128);
    for (int i = 0; i < P_SLOTS; ++i) mbar_init(&p_full[i], 128);
    for (int i = 0; i < P_SLOTS; ++i) mbar_init(&pv_done[i], 1);
    for (int i = 0; i < PV_BUFS; ++i) { mbar_init(&pvh_done[i], 1); mbar_init(&pvh_empty[i], 128); }
    for (int i = 0; i < AB_RING; ++i) mbar_init(&ab_full[i], 128);
    for (int i = 0; i < KS_RING; ++i) { mbar_init(&ks_full[i], 1); mbar_init(&ks_empty[i], 128); }
    for (int i = 0; i < VS_RING; ++i) { mbar_init(&vs_full[i], 1); mbar_init(&vs_empty[i], 128); }
    for (int i = 0; i < RUN_RING; ++i) mbar_init(&run_full[i], 128);
    fence_mbar_init();
  }
  if (warp == kWarpAlloc) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  constexpr uint32_t TM_S = 0, TM_PV = 256;                 // S[2] x 128 | PV half buffers [4] x 64

  // register pool of the CTA = 512 x 128; after redistribution 128 x 24 + 256 x kRegSoftmax + 128 x kRegDrain = 65536
  if (warp >= kWarpAlloc) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
    // The single-thread roles keep warp-uniform control flow (every lane waits; one elected lane issues), so that the
    // TMA / MMA operands stay in uniform registers.
    if (warp == kWarpTma) {
      // ---------------------------------------------------------------- TMA producer
      if (elect_one()) {
        tma_prefetch_desc(&tmQ); tma_prefetch_desc(&tmK); tma_prefetch_desc(&tmV);
        mbar_arrive_expect_tx(q_full, L::Q_BYTES);
        tma_load_3d(sQ, &tmQ, q_full, 0, q0, bh);
      }
      __syncwarp();
      for (int i = 0; i < nblk + 2; ++i) {
        const int m = i, j = i - 2;                                      // K runs two blocks ahead of V
        if (m < nblk) {
          const int s = m % K_STAGES;
          mbar_wait_hint(&s_done[s], ((m / K_STAGES) & 1) ^ 1);               // S(m-4) has consumed this K stage
          if (elect_one()) {
            mbar_arrive_expect_tx(&k_full[s], L::K_BYTES);
            tma_load_3d(sK + s * L::K_BYTES, &tmK, &k_full[s], 0, m * kTile, bh);
          }
          __syncwarp();
          if (QKG == 1) {                                                     // key scales of block m (and the smoothing correction)
            const int rg = m % KS_RING;
            mbar_wait_hint(&ks_empty[rg], ((m / KS_RING) & 1) ^ 1);
            if (elect_one()) {
              mbar_arrive_expect_tx(&ks_full[rg], SM ? 1024 : 512);
              bulk_load(smem_u32(sKs + rg * 128), a.KsP + (size_t)bh * a.npad + m * kTile, 512, smem_u32(&ks_full[rg]));
              if (SM) bulk_load(smem_u32(sKc + rg * 128), a.KcP + (size_t)bh * a.npad + m * kTile, 512, smem_u32(&ks_full[rg]));
            }
            __syncwarp();
          }
        }
        if (j >= 0) {
          const int s = j % V_STAGES;
          if (j >= V_STAGES) mbar_wait_hint(&pv_done[(j - V_STAGES) % P_SLOTS], ((j - V_STAGES) / P_SLOTS) & 1);   // P~V(j-3) has consumed this V stage
          if (elect_one()) {
            mbar_arrive_expect_tx(&v_full[s], L::V_BYTES);
            tma_load_3d(sV + s * L::V_BYTES, &tmV, &v_full[s], j * kTile, 0, bh);
          }
          __syncwarp();
          if (VSC == 0) {                                                     // V scales of group j
            const int rg = j % VS_RING;
            mbar_wait_hint(&vs_empty[rg], ((j / VS_RING) & 1) ^ 1);
            if (elect_one()) {
              mbar_arrive_expect_tx(&vs_full[rg], D * 4);
              bulk_load(smem_u32(sVs + rg * D), a.Vs + ((size_t)bh * nblk + j) * D, D * 4, smem_u32(&vs_full[rg]));
            }
            __syncwarp();
          }
        }
      }
    } else if (warp == kWarpMmaS) {
      // ---------------------------------------------------------------- MMA issuer 1: S(m) = Q K(m)^T -> buffer m & 1
      constexpr uint32_t idesc_s = umma_idesc(1, 0, 0, 128, 128);        // f32 <- e4m3 x e4m3 (integer codes * 2^-9)
      constexpr int KSTEPS_S = D / 32;                                   // D=64 rows are zero-padded to 128 B
      const uint64_t qd = umma_desc_k128(smem_u32(sQ));
      mbar_wait_hint(q_full, 0);
      for (int m = 0; m < nblk; ++m) {
        const int st = m % K_STAGES, b = m & 1;
        mbar_wait_hint(&k_full[st], (m / K_STAGES) & 1);
        if (m >= 2) mbar_wait_hint(&s_empty[b], ((m >> 1) - 1) & 1);          // softmax has read S(m-2) out of this buffer
        tc_fence_after();
        if (elect_one()) {
          const uint64_t kd = umma_desc_k128(smem_u32(sK + st * L::K_BYTES));
#pragma unroll
          for (int k = 0; k < KSTEPS_S; ++k)
            mma_ss<MmaKind::F8F6F4>(tmem_base + TM_S + b * 128, qd + 2 * k, kd + 2 * k, idesc_s, k != 0);
          tc_commit(&s_done[st]);                                        // -> softmax group (S ready) and TMA (K stage free)
        }
        __syncwarp();
      }
    } else if (warp == kWarpMmaPV) {
      // ---------------------------------------------------------------- MMA issuer 2: PV = P~(j) V(j)
      constexpr uint32_t idesc_pv = umma_idesc(1, 0, 0, 128, D / 2);
      for (int j = 0; j < nblk; ++j) {
        const int slot = j % P_SLOTS, vst = j % V_STAGES;
        mbar_wait_hint(&v_full[vst], (j / V_STAGES) & 1);
        mbar_wait_hint(&p_full[slot], (j / P_SLOTS) & 1);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int buf = 2 * (j & 1) + h;
          mbar_wait_hint(&pvh_empty[buf], ((j >> 1) & 1) ^ 1);                // drain has read half (j-2, h) out of this buffer
          tc_fence_after();
          if (elect_one()) {
            // V^T tile: channel half h starts D/2 rows (= D/2 * 128 B, whole 1024-byte swizzle atoms) into the tile
            const uint64_t pd = umma_desc_k128(smem_u32(sP + slot * L::P_BYTES));
            const uint64_t vd = umma_desc_k128(smem_u32(sV + vst * L::V_BYTES + h * (D / 2) * 128));
#pragma unroll
            for (int k = 0; k < 4; ++k)
              mma_ss<MmaKind::F8F6F4>(tmem_base + TM_PV + buf * 64, pd + 2 * k, vd + 2 * k, idesc_pv, k != 0);
            tc_commit(&pvh_done[buf]);                                   // -> drain
            if (h == 1) tc_commit(&pv_done[slot]);                        // -> softmax (P slot free), TMA (V stage free)
          }
          __syncwarp();
        }
      }
    }
  } else if (warp < kWarpDrain) {
    // ------------------------------------------------------------------ softmax groups: 0 = even blocks, 1 = odd blocks
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegSoftmax));
    constexpr float LOG2_LEVELS = P_MODE == ROTATTN_P_ASYM15 ? 3.9068905956085187f : 2.8073549220576042f;
    const int g = warp >> 2;                         // group index = S buffer index
    const int r = (warp & 3) * 32 + lane;
    const int row = q0 + r;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    // Per-token: f = Qs_i * 2^18 log2e/sqrt(D); f >= 1e-30 keeps (-inf) * f well defined for masked keys; an all-zero
    // query row still gives s == 0 everywhere.  QKG = 128: f = max(Qs_tile * Ks_block * 2^18 log2e/sqrt(D), 1e-30), same reason.
    float fq;
    if (QKG == 1) fq = (row < a.N) ? fmaxf(a.Qs[(size_t)bh * a.N + row] * a.scale_log2, 1e-30f) : 1e-30f;
    else fq = a.Qs[(size_t)bh * nblk + qtile] * a.scale_log2;
    const float* ksg = a.Ks + (size_t)bh * nblk;           // QKG = 128 only
    const uint32_t s_addr = tmem_base + lane_off + TM_S + g * 128;
    const uint32_t p_row0 = smem_u32(sP) + r * 128;        // 16-byte chunk q of row r lives at chunk q ^ (r & 7)
    const uint32_t swz = (uint32_t)(r & 7) << 4;
    const int tok_mine = 1 + 4 * g + (warp & 3), tok_other = 1 + 4 * (g ^ 1) + (warp & 3);
    if (TOKEN && g == 1) bar_arrive(tok_other, 64);        // group 0 takes the first turn
    for (int j = g; j < nblk; j += 2) {
      const int ring = j % KS_RING, slot = j % P_SLOTS, abslot = j % AB_RING;
      const int nvalid = a.N - j * kTile;                  // < 128 only on the ragged last block
      float qs = fq;
      if (QKG != 1) qs = fmaxf(qs * ksg[j], 1e-30f);       // a zero block scale (all-zero Q tile / K block) must not meet the -inf of masked keys
      const float2 qs2 = make_float2(qs, qs);
      if (QKG == 1) mbar_wait(&ks_full[ring], (j / KS_RING) & 1);
      mbar_wait(&s_done[j % K_STAGES], (j / K_STAGES) & 1);
      tc_fence_after();
      if (nvalid < kTile) {                                // keys >= N: -inf over their accumulators (once per CTA)
#pragma unroll 1
        for (int c = nvalid >> 4; c < 8; ++c) {
          uint32_t v[16];
          tmem_ld16(s_addr + c * 16, v);
          tmem_wait_ld();
#pragma unroll
          for (int i = 0; i < 16; ++i) v[i] = (c * 16 + i >= nvalid) ? 0xff800000u : v[i];
          tmem_st16(s_addr + c * 16, v);
        }
        tmem_wait_st();
      }
      uint32_t u[4][32];                                   // the row of S: accumulator * 2^-18 as fp32
#pragma unroll
      for (int c = 0; c < 4; ++c) tmem_ld32(s_addr + c * 32, u[c]);
      tmem_wait_ld();
      tc_fence_before();
      mbar_arrive(&s_empty[g]);                            // S(j+2) may be issued: this thread works from registers now
      if (DEBUG) {
#pragma unroll
        for (int i = 0; i < 128; ++i)
          a.S_dump[(size_t)r * a.npad + j * kTile + i] = (int32_t)(__uint_as_float(u[i >> 5][i & 31]) * kAccScale);
      }
      // ---- t = S * ks (per-token), block row max
      float mx0 = -INFINITY, mx1 = -INFINITY;
      {
        const float4* ks4 = reinterpret_cast<const float4*>(sKs + ring * 128);
        const float4* kc4 = reinterpret_cast<const float4*>(sKc + ring * 128);
#pragma unroll
        for (int c = 0; c < 32; ++c) {
          uint32_t* w = &u[c >> 3][(c & 7) * 4];
          float2 t0 = make_float2(__uint_as_float(w[0]), __uint_as_float(w[1]));
          float2 t1 = make_float2(__uint_as_float(w[2]), __uint_as_float(w[3]));
          if (QKG == 1) {
            const float4 k = ks4[c];
            t0 = fmul2(t0, make_float2(k.x, k.y));
            t1 = fmul2(t1, make_float2(k.z, k.w));
          }
          if (SM) {
            const float4 k = kc4[c];
            t0 = ffma2(t0, qs2, make_float2(k.x, k.y));
            t1 = ffma2(t1, qs2, make_float2(k.z, k.w));
          }
          mx0 = fmax3(mx0, t0.x, t0.y);
          mx1 = fmax3(mx1, t1.x, t1.y);
          if (QKG == 1 || SM) {
            w[0] = __float_as_uint(t0.x); w[1] = __float_as_uint(t0.y);
            w[2] = __float_as_uint(t1.x); w[3] = __float_as_uint(t1.y);
          }
        }
      }
      if (QKG == 1) mbar_arrive(&ks_empty[ring]);
      const float tmax = fmaxf(mx0, mx1);
      float mt = SM ? tmax : qs * tmax;                    // block row max of s * log2e (smoothing: Qs_i is already in t)
      if (PN == ROTATTN_NORM_RUNNING) {
        // Codes relative to the running max (SURVEY 8c reading 13, alternative): block j needs the maximum over blocks
        // <= j.  Block j - 1 belongs to the other softmax group, whose thread of the same row publishes its running max
        // right after its own max pass, so only the max passes are serialised, not the exp2 phases.  The drain needs no
        // change: it receives the normaliser of the block, whatever its definition.
        if (j > 0) {
          mbar_wait(&run_full[(j - 1) % RUN_RING], ((j - 1) / RUN_RING) & 1);
          mt = fmaxf(mt, sRun[((j - 1) % RUN_RING) * 128 + r]);
        }
        sRun[(j % RUN_RING) * 128 + r] = mt;               // slot reuse: block j + 4 starts after block j + 3, which read block j + 2, ...
        mbar_arrive(&run_full[j % RUN_RING]);
      }
      const float nref = LOG2_LEVELS - mt;
      const float2 nref2 = make_float2(nref, nref);
      const float2 es2 = SM ? make_float2(1.f, 1.f) : qs2;
      mbar_wait(&pv_done[slot], ((j / P_SLOTS) & 1) ^ 1);            // P~V(j-4) has consumed this P slot
      // The two softmax warps of an SM sub-partition (one of each group) take turns in the exp2 phase (a token passed
      // through two named barriers): one of them feeds the exp2 unit while the other is in its load / scale / max phase,
      // instead of both running the same phase side by side and leaving the unit idle in between.  bar.sync orders memory
      // operations only: ptxas schedules the 64 exponent FFMA2 and the first ~19 MUFU.EX2 of the block before it, which is
      // the best split measured (everything behind the token: +6 %).
      if (TOKEN) bar_sync(tok_mine, 64);
      // ---- LEVELS * P^ = exp2(t * f - mt + log2(LEVELS)); codes u = rne(LEVELS * P^) taken from the low byte of
      // (LEVELS * P^) + 1.5 * 2^23 (Eq.12 L166-168 with the fixed scale 15 / Eq.11 L161 with 7); four codes per 32-bit word
      float2 ls0 = make_float2(0.f, 0.f), ls1 = make_float2(0.f, 0.f);
      const float2 magic2 = make_float2(12582912.f, 12582912.f);
      const uint32_t p_row = p_row0 + slot * L::P_BYTES;
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        uint32_t pw[4];
#pragma unroll
        for (int x = 0; x < 4; ++x) {
          const uint32_t* w = &u[q >> 1][(q & 1) * 16 + x * 4];
          const float2 e0 = ffma2(make_float2(__uint_as_float(w[0]), __uint_as_float(w[1])), es2, nref2);
          const float2 e1 = ffma2(make_float2(__uint_as_float(w[2]), __uint_as_float(w[3])), es2, nref2);
          constexpr int POLY = (QKG != 1 && VSC != 0) ? ROTATTN_POLY_BLOCK : (QKG != 1 ? ROTATTN_POLY_BLOCK_VCH : ROTATTN_POLY_TOKEN);
          const bool poly = (POLY >= 1 && x == 3) || (POLY >= 2 && x == 1) || (POLY >= 3 && x == 2) || (POLY >= 4 && x == 0);   // compile-time after unrolling
          const float2 p0 = make_float2(ex2_approx(e0.x), ex2_approx(e0.y));
          const float2 p1 = poly ? ex2_fma_pipe2(e1) : make_float2(ex2_approx(e1.x), ex2_approx(e1.y));
          ls0 = fadd2(ls0, p0);
          ls1 = fadd2(ls1, p1);
          const float2 f0 = fadd2(p0, magic2), f1 = fadd2(p1, magic2);
          const uint32_t lo = __byte_perm(__float_as_uint(f0.x), __float_as_uint(f0.y), 0x0040);
          const uint32_t hi = __byte_perm(__float_as_uint(f1.x), __float_as_uint(f1.y), 0x0040);
          pw[x] = __byte_perm(lo, hi, 0x5410);
        }
        if (DEBUG) {
#pragma unroll
          for (int x = 0; x < 4; ++x) *reinterpret_cast<uint32_t*>(a.P_dump + (size_t)r * a.npad + j * kTile + q * 16 + x * 4) = pw[x];
        }
        sts_u32x4(p_row + (((uint32_t)q << 4) ^ swz), pw[0], pw[1], pw[2], pw[3]);
      }
      if (TOKEN) bar_arrive(tok_other, 64);
      sAB[(abslot * 2) * 128 + r] = mt;
      sAB[(abslot * 2 + 1) * 128 + r] = (ls0.x + ls0.y) + (ls1.x + ls1.y);
      fence_proxy_async_smem();                          // P codes (generic-proxy stores) -> visible to the MMA (async proxy)
      mbar_arrive(&p_full[slot]);
      mbar_arrive(&ab_full[abslot]);
    }
  } else {
    // ------------------------------------------------------------------ drain: one thread per query row of O
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegDrain));
    constexpr int DH = D / 2;                      // channels per P~V half buffer
    const int r = (warp & 3) * 32 + lane;
    const int row = q0 + r;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    float2 o2[D / 2];
#pragma unroll
    for (int d = 0; d < D / 2; ++d) o2[d] = make_float2(0.f, 0.f);
    // Online softmax bookkeeping (L157) with a lazily updated reference max: O and l are kept relative to m_ref, which
    // only moves when a block max exceeds it by more than 2^8 (fp32 has the headroom), so the common path is
    // O += beta * pv * Vs with beta = exp2(mt - m_ref) and no rescale of the accumulators.
    constexpr float kLazy = 8.f;
    float m_ref = -INFINITY, l_run = 0.f;
    const float* vsg = a.Vs + (size_t)bh * nblk;             // VSC = 1 only
    for (int j = 0; j < nblk; ++j) {
      const int abslot = j % AB_RING;
      mbar_wait(&ab_full[abslot], (j / AB_RING) & 1);
      const float mt = sAB[(abslot * 2) * 128 + r];
      const float bsum = sAB[(abslot * 2 + 1) * 128 + r];
      const int vring = j % VS_RING;
      if (__any_sync(0xffffffffu, mt > m_ref + kLazy)) {               // rare after the first blocks (warp-uniform branch)
        const float m_new = (mt > m_ref + kLazy) ? mt : m_ref;
        const float alpha = ex2_approx(m_ref - m_new);                 // first block: exp2(-inf) = 0; unchanged rows: 1
        const float2 a2 = make_float2(alpha, alpha);
#pragma unroll
        for (int d = 0; d < D / 2; ++d) o2[d] = fmul2(o2[d], a2);
        l_run *= alpha;
        m_ref = m_new;
      }
      const float beta = ex2_approx(mt - m_ref);                       // <= 2^8
      l_run = fmaf(beta, bsum, l_run);                                 // in units of LEVELS (cancels in O/l)
      float cf = beta * kAccScale;                                     // undoes the 2^-18 of the E4M3 code products
      if (VSC != 0) cf *= vsg[j];
      const float2 c2 = make_float2(cf, cf);
      if (VSC == 0) mbar_wait(&vs_full[vring], (j / VS_RING) & 1);
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int buf = 2 * (j & 1) + h;
        const uint32_t pv_addr = tmem_base + lane_off + TM_PV + buf * 64;
        const float4* vsb4 = reinterpret_cast<const float4*>(sVs + vring * D + h * DH);
        mbar_wait(&pvh_done[buf], (j >> 1) & 1);
        tc_fence_after();
        uint32_t va[16], vb[16];
        tmem_ld16(pv_addr, va);
#pragma unroll
        for (int cc = 0; cc < DH / 16; ++cc) {
          tmem_wait_ld();
          uint32_t(&cur)[16] = (cc & 1) ? vb : va;
          uint32_t(&nxt)[16] = (cc & 1) ? va : vb;
          if (cc + 1 < DH / 16) tmem_ld16(pv_addr + (cc + 1) * 16, nxt);
          else { tc_fence_before(); mbar_arrive(&pvh_empty[buf]); }      // this half-width accumulator is in registers now
          if (DEBUG) {
            if (a.PV_dump) {
#pragma unroll
              for (int i = 0; i < 16; ++i)
                a.PV_dump[((size_t)j * kTile + r) * D + h * DH + cc * 16 + i] = (int32_t)(__uint_as_float(cur[i]) * kAccScale);
            }
          }
#pragma unroll
          for (int d = 0; d < 4; ++d) {
            float2 y0 = make_float2(__uint_as_float(cur[4 * d]), __uint_as_float(cur[4 * d + 1]));
            float2 y1 = make_float2(__uint_as_float(cur[4 * d + 2]), __uint_as_float(cur[4 * d + 3]));
            if (VSC == 0) {
              const float4 s = vsb4[cc * 4 + d];
              y0 = fmul2(y0, make_float2(s.x, s.y));
              y1 = fmul2(y1, make_float2(s.z, s.w));
            }
            float2& oa = o2[h * (DH / 2) + cc * 8 + 2 * d];
            float2& ob = o2[h * (DH / 2) + cc * 8 + 2 * d + 1];
            oa = ffma2(y0, c2, oa);                                      // O += beta * pv * Vs[g][d]
            ob = ffma2(y1, c2, ob);
          }
        }
      }
      if (VSC == 0) mbar_arrive(&vs_empty[vring]);
    }
    const float inv_l = 1.f / l_run;
    if (row < a.N) {
      __half* dst = DEBUG ? a.O + (size_t)r * D : a.O + ((size_t)bh * a.N + row) * D;
      const float2* mv2 = reinterpret_cast<const float2*>(a.means + ((size_t)bh * 3 + 2) * D);   // smoothing: mean of V
#pragma unroll
      for (int d = 0; d < D; d += 8) {
        __half2 hh[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          float2 o = make_float2(o2[d / 2 + i].x * inv_l, o2[d / 2 + i].y * inv_l);
          if (SM) { const float2 m = mv2[d / 2 + i]; o.x += m.x; o.y += m.y; }       // softmax(.)(V - mean) + mean
          hh[i] = __floats2half2_rn(o.x, o.y);
        }
        *reinterpret_cast<uint4*>(dst + d) = *reinterpret_cast<uint4*>(hh);
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kWarpAlloc) tmem_dealloc(tmem_base, 512);
}


// ---- host side: variant dispatch for one (D, DEBUG) flavour -------------------------------------------------------
template <int D, int P_MODE, int QKG, int VSC, int SM, int PN, bool DEBUG>
int launch_one(const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv, const FwdInt4Args& a, dim3 grid,
               cudaStream_t cs) {
  constexpr int smem = SmemInt4<D>::TOTAL;
  auto kern = fwd_int4_kernel<D, P_MODE, QKG, VSC, SM, PN, DEBUG>;
  static PerDeviceOnce once;    // per variant and device: ptxas must have allocated exactly the register pool setmaxnreg assumes,
  int dev = 0;                  // and the dynamic shared-memory opt-in is a per-device attribute
  ROTATTN_CUDA_TRY(cudaGetDevice(&dev));
  if (!once.done(dev)) {
    cudaFuncAttributes fa;
    ROTATTN_CUDA_TRY(cudaFuncGetAttributes(&fa, kern));
    if (fa.numRegs != 128) {
      set_error_text("fwd_int4_kernel: unexpected register allocation (setmaxnreg pool assumes 128 registers per thread)");
      return ROTATTN_ERR_UNSUPPORTED;
    }
    ROTATTN_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    once.mark(dev);
  }
  kern<<<grid, kFwdThreads, smem, cs>>>(tq, tk, tv, a);
  ROTATTN_CUDA_TRY(cudaGetLastError());
  return ROTATTN_OK;
}

template <int D, bool DEBUG>
int launch_variants(const rotattn_params& p, const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv,
                    const FwdInt4Args& a, dim3 grid, cudaStream_t cs) {
  const int sel = (p.p_mode == ROTATTN_P_SYM7 ? 4 : 0) | (p.qk_group == 128 ? 2 : 0) | (p.v_scale == ROTATTN_VSCALE_GROUP ? 1 : 0);
  if (p.p_norm == ROTATTN_NORM_RUNNING)   // validated: the running normaliser comes with the paper's granularity only, without smoothing
    return sel & 4 ? launch_one<D, ROTATTN_P_SYM7, 1, 0, 0, ROTATTN_NORM_RUNNING, DEBUG>(tq, tk, tv, a, grid, cs)
                   : launch_one<D, ROTATTN_P_ASYM15, 1, 0, 0, ROTATTN_NORM_RUNNING, DEBUG>(tq, tk, tv, a, grid, cs);
  if (p.smooth)        // validated: smoothing comes with the paper's granularity only
    return sel & 4 ? launch_one<D, ROTATTN_P_SYM7, 1, 0, 1, ROTATTN_NORM_ROWBLOCK, DEBUG>(tq, tk, tv, a, grid, cs)
                   : launch_one<D, ROTATTN_P_ASYM15, 1, 0, 1, ROTATTN_NORM_ROWBLOCK, DEBUG>(tq, tk, tv, a, grid, cs);
  switch (sel) {
    case 0: return launch_one<D, ROTATTN_P_ASYM15, 1, 0, 0, ROTATTN_NORM_ROWBLOCK, DEBUG>(tq, tk, tv, a, grid, cs);
    case 1: return launch_one<D, ROTATTN_P_ASYM15, 1, 1, 0, ROTATTN_NORM_ROWBLOCK, DEBUG>(tq, tk, tv, a, grid, cs);
    case 2: return launch_one<D, ROTATTN_P_ASYM15, 128, 0, 0, ROTATTN_NORM_ROWBLOCK, DEBUG>(tq, tk, tv, a, grid, cs);
    case 3: return launch_one<D, ROTATTN_P_ASYM15, 128, 1, 0, ROTATTN_NORM_ROWBLOCK, DEBUG>(tq, tk, tv, a, grid, cs);
    case 4: return launch_one<D, ROTATTN_P_SYM7, 1, 0, 0, ROTATTN_NORM_ROWBLOCK, DEBUG>(tq, tk, tv, a, grid, cs);
    case 5: return launch_one<D, ROTATTN_P_SYM7, 1, 1, 0, ROTATTN_NORM_ROWBLOCK, DEBUG>(tq, tk, tv, a, grid, cs);
    case 6: return launch_one<D, ROTATTN_P_SYM7, 128, 0, 0, ROTATTN_NORM_ROWBLOCK, DEBUG>(tq, tk, tv, a, grid, cs);
    default: return launch_one<D, ROTATTN_P_SYM7, 128, 1, 0, ROTATTN_NORM_ROWBLOCK, DEBUG>(tq, tk, tv, a, grid, cs);
  }
}

}  // namespace rotattn
