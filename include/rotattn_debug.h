/* rotattn_debug.h - test and measurement aids of librotattn.so.  NOT part of the product ABI (include/rotattn.h) and
 * never on the timed path: parity tests use the dumps, bench.py uses the GEMM probe to MEASURE the dense 8-bit tensor
 * peak that the roofline of fwd_int4 is quoted against. */
#ifndef ROTATTN_DEBUG_H_
#define ROTATTN_DEBUG_H_

#include "rotattn.h"

#ifdef __cplusplus
extern "C" {
#endif

/* rotattn_fwd_int4 for ONE (bh, query tile of 128 rows), additionally dumping the integer S accumulators (step 7),
 * the P codes (step 9) and the integer P~V accumulators of every KV block (step 10).
 * S_dump: int32 [128, ceil128(N)], P_dump: uint8 [128, ceil128(N)], PV_dump: int32 [ceil(N/128), 128, D] or NULL,
 * O_tile: fp16 [128, D] (rows >= N untouched). */
int rotattn_fwd_int4_debug(const rotattn_params* p,
                           const uint8_t* Q4, const float* Qs, const uint8_t* K4, const float* Ks,
                           const uint8_t* V4, const float* Vs,
                           int32_t bh, int32_t q_tile, int32_t* S_dump, uint8_t* P_dump, int32_t* PV_dump, void* O_tile,
                           void* workspace, size_t ws_bytes, int32_t ws_state, void* stream);

/* rotattn_fwd_fp16 with the epilogue's quotient O/l stored as fp32 instead of being rounded to fp16 (same kernel, one
 * compile-time switch in the last store).  It exists so that the kernel's ARITHMETIC can be held to north_star's strict
 * "within 2e-3 max-abs of FP64 attention" (PAPER.md:L157 exact attention, L192 fallback precision): on the fp16 output half
 * an ulp of |O| in [4, 16) is itself 2e-3 .. 3.9e-3, which is rounding of the result, not kernel error (reading 25).
 * O32: out, fp32 [B,H,N,D], 16-byte aligned.  Other arguments as for rotattn_fwd_fp16. */
int rotattn_fwd_fp16_debug_f32(const rotattn_params* p, const void* Q16, const void* K16, const void* V16, float* O32,
                               const int32_t* head_sel, int32_t n_sel, void* workspace, size_t ws_bytes, void* stream);

/* Dense 8-bit GEMM C[M,N] = A[M,K] * B[N,K]^T on the same tcgen05 path the attention kernel uses.
 * M multiple of 128, N multiple of 256, K multiple of 128.  A,B: device, row-major, 1 byte per element.
 *   mode 0: kind::i8, A and B signed int8, C int32.
 *   mode 1: kind::f8f6f4, A and B E4M3 bit patterns, C float (fp32 accumulators) - the attention kernels' path.
 *   mode 2: kind::i8 with A (UNSIGNED u8) staged through tensor memory, B signed; M=N=K=128 only, C int32. */
int rotattn_probe_gemm8(int32_t M, int32_t N, int32_t K, const void* A, const void* B, void* C,
                        int32_t mode, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* ROTATTN_DEBUG_H_ */
