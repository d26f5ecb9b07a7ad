// Shared declarations of the two INT4 attention kernels (fwd_int4.cu: ROWBLOCK normaliser, block-independent
// softmax; fwd_int4_sync.cu: RUNNING normaliser, softmax serialised over KV blocks).
#pragma once
#include "tc_common.cuh"

namespace rotattn {

constexpr int kInt4Threads = 640;
// The widened operands are E4M3 bytes that encode code * 2^-9 (see prologue.cu: code_byte), so both tensor products
// arrive in tensor memory as fp32 values  integer_accumulator * 2^-18  (exact: |acc| <= 13440 < 2^24).
constexpr float kAccScale = 262144.f;

struct FwdInt4Args {
  const float* Qs;        // [BH, N]
  const float* Ks;        // [BH, N]
  const float* Vs;        // [BH, nG, D]
  __half* O;              // [BH, N, D]  (debug: [128, D] tile)
  const int32_t* head_sel;
  int32_t* S_dump;        // debug only
  uint8_t* P_dump;        // debug only
  int N, nblk, npad;
  int dbg_bh, dbg_qtile;  // debug only
  float scale_log2;       // 2^18 * log2(e) / sqrt(D)
#ifdef ROTATTN_TRACE
  long long* trace;       // development builds only: [32 warps][64 blocks][16 events] clock stamps of CTA (0,0)
#endif
};

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
#if defined(ROTATTN_ABL) && ROTATTN_ABL == 1      // development ablation: no MUFU
  y = x * 0.0001f + 1.0f;
#else
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
#endif
  return y;
}

#ifdef ROTATTN_TRACE
#define ROTATTN_STAMP(j, e)                                                                                     \
  do {                                                                                                          \
    if (a.trace && blockIdx.x == 0 && blockIdx.y == 0 && (threadIdx.x & 31) == 0 && (j) < 64)                   \
      a.trace[(((threadIdx.x >> 5) * 64) + (j)) * 16 + (e)] = clock64();                                         \
  } while (0)
#else
#define ROTATTN_STAMP(j, e) do {} while (0)
#endif

// RUNNING-normaliser kernel (fwd_int4_sync.cu)
int launch_fwd_int4_sync(const rotattn_params& p, const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv,
                         const FwdInt4Args& a, dim3 grid, bool debug, cudaStream_t cs);

}  // namespace rotattn
