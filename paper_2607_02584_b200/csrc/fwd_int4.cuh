// Shared declarations of the INT4 attention kernel (fwd_int4_kernel.cuh: ROWBLOCK and RUNNING normalisers).
#pragma once
#include "tc_common.cuh"

namespace rotattn {

constexpr int kFwdThreads = 512;       // fwd_int4_kernel
// The widened operands are E4M3 bytes that encode code * 2^-9 (see prologue.cu: code_byte), so both tensor products
// arrive in tensor memory as fp32 values  integer_accumulator * 2^-18  (exact: |acc| <= 13440 < 2^24;
// tests/test_gpu_probe.py holds the adversarial exactness cases).
constexpr float kAccScale = 262144.f;

struct FwdInt4Args {
  const float* Qs;        // [BH, N]   (qk_group = 128: [BH, nblk])
  const float* Ks;        // [BH, N]   (qk_group = 128: [BH, nblk])
  const float* KsP;       // workspace copy of Ks padded to [BH, npad] (per-token mode; bulk-copied next to the K tiles)
  const float* KcP;       // smoothing: per-key correction (log2 domain), padded [BH, npad]
  const float* means;     // smoothing: column means [BH, 3, D] (Q, K, V)
  const float* Vs;        // [BH, nblk, D]   (v_scale = GROUP: [BH, nblk])
  __half* O;              // [BH, N, D]  (debug: [128, D] tile)
  const int32_t* head_sel;
  int32_t* S_dump;        // debug only: [128, npad]
  uint8_t* P_dump;        // debug only: [128, npad]
  int32_t* PV_dump;       // debug only, may be NULL: [nblk, 128, D]
  int N, nblk, npad;
  int dbg_bh, dbg_qtile;  // debug only
  float scale_log2;       // 2^18 * log2(e) / sqrt(D)
};

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// one translation unit per head dimension / debug flavour (parallel compilation)
int launch_fwd_int4_d128(const rotattn_params& p, const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv,
                         const FwdInt4Args& a, dim3 grid, cudaStream_t cs);
int launch_fwd_int4_d64(const rotattn_params& p, const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv,
                        const FwdInt4Args& a, dim3 grid, cudaStream_t cs);
int launch_fwd_int4_debug(const rotattn_params& p, const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv,
                          const FwdInt4Args& a, dim3 grid, cudaStream_t cs);
}  // namespace rotattn
