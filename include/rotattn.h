/* rotattn.h — C-ABI of the B200-native RotateAttention hot path (arxiv/paper_2607_02584).
 *
 * One shared object, librotattn.so, hand-written CUDA for sm_100a.  There is NO CPU fallback and
 * no other backend: on a machine without an sm_100 device every compute entry point returns
 * ROTATTN_ERR_UNSUPPORTED / ROTATTN_ERR_CUDA.  Citations "PAPER.md:Lnnn" are lines of the paper
 * text; "reading n" refers to the table of readings in DESIGN.md.
 *
 * Conventions (all entry points)
 *  - Tensor pointers are CALLER-OWNED DEVICE pointers unless the argument says "host".
 *    The library never allocates, frees or synchronises; all work is enqueued on `stream`
 *    (a cudaStream_t passed as void*; NULL = legacy default stream).  Inputs are never modified.
 *  - Layout: Q,K,V,O are [B,H,N,D] row-major (D contiguous), fp16 (IEEE binary16).
 *    N = N_rope + N_text; token n < N_rope = grid_t*grid_h*grid_w sits at video position
 *    (t,h,w) with n = (t*grid_h + h)*grid_w + w; tokens n >= N_rope carry no RoPE (reading 7).
 *  - Return value: 0 on success, a negative rotattn_status otherwise.  Never aborts or throws.
 */
#ifndef ROTATTN_H_
#define ROTATTN_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum rotattn_status {
  ROTATTN_OK = 0,
  ROTATTN_ERR_INVALID_ARG = -1,         /* NULL pointer, sum(pairs) != D/2, t*h*w > N, n_sel out of range */
  ROTATTN_ERR_UNSUPPORTED = -2,         /* D not in {64,128}, kv_block != 128, v_group != 128, qk_group != 1,
                                           device is not sm_100 */
  ROTATTN_ERR_NOT_ORTHOGONAL = -3,      /* max|R_i^T R_i - I| > 1e-5 */
  ROTATTN_ERR_WORKSPACE_TOO_SMALL = -4,
  ROTATTN_ERR_CUDA = -5                 /* a CUDA runtime/driver call failed; see rotattn_last_cuda_error() */
} rotattn_status;

enum { ROTATTN_ROT_NONE = 0, ROTATTN_ROT_INTERLEAVED = 1, ROTATTN_ROT_HALF = 2 };
enum { ROTATTN_P_ASYM15 = 0, ROTATTN_P_SYM7 = 1 };
enum { ROTATTN_NORM_ROWBLOCK = 0, ROTATTN_NORM_RUNNING = 1 };
/* ws_state bits for rotattn_fwd_int4 */
enum { ROTATTN_WS_HAS_QK = 1, ROTATTN_WS_HAS_V = 2 };

/* Problem statement: Q,K,V in R^{N x D} per head; D = D_f + D_h + D_w (L58);
 * block-diagonal rotation R of D/2 O(2) blocks (Eq.3); per-token Q/K and per-group V scales
 * (L190); KV block of the FlashAttention loop (L157). */
typedef struct rotattn_params {
  int32_t B, H, N, D;                 /* D in {64,128} */
  int32_t grid_t, grid_h, grid_w;     /* N_rope = t*h*w <= N */
  int32_t pairs_t, pairs_h, pairs_w;  /* RoPE pairs per section, sum == D/2, channel order [t|h|w] */
  float   rope_base;                  /* 10000 */
  int32_t rot_mode;                   /* ROTATTN_ROT_* : NONE, INTERLEAVED (merged into the table, Eq.7),
                                         HALF (Eq.8, same register pass) */
  int32_t p_mode;                     /* ROTATTN_P_ASYM15 (Eq.12) | ROTATTN_P_SYM7 (Eq.11) */
  int32_t p_norm;                     /* ROTATTN_NORM_ROWBLOCK (reading 13, default) | ROTATTN_NORM_RUNNING */
  int32_t qk_group;                   /* tokens per Q/K scale; 1 = per-token (L190).  Only 1 is built. */
  int32_t v_group;                    /* tokens per V scale group (L190, reading 11).  Only 128 is built. */
  int32_t kv_block;                   /* P-normalisation block (L157, reading 18).  Only 128 is built. */
} rotattn_params;

/* ---- host-side helpers (no GPU needed) ------------------------------------------------------- */

/* Validate a parameter block.  Returns ROTATTN_OK / INVALID_ARG / UNSUPPORTED. */
int rotattn_validate(const rotattn_params* p);

/* Number of floats of the coefficient table: 4 * ((t+1)*P_t + (h+1)*P_h + (w+1)*P_w). */
size_t rotattn_table_floats(const rotattn_params* p);

/* Build the per-axis RoPE coefficient table offline ("pre-fusing R into the RoPE
 * weights").  For axis a in (t,h,w), position pos = 0..L_a (row L_a = no-RoPE row for text tokens),
 * pair k = 0..P_a-1: 2x2 block A = [a00,a01,a10,a11], theta = pos * base^(-k/P_a):
 *   NONE/HALF: A = M(theta) = [[cos,sin],[-sin,cos]]  (row-vector convention, y = x A, L60, Eq.7)
 *   INTERLEAVED: A = M(theta) * R_k'                  (Eq.7), product in fp64, rounded to fp32.
 * rot_host: host float [D/2][4] = (r00,r01,r10,r11) per pair, or NULL for R_i = H_2 (Eq.4).
 * coef_host: host output, rotattn_table_floats(p) floats.  The caller copies it to the device.
 * Errors: INVALID_ARG, UNSUPPORTED, NOT_ORTHOGONAL. */
int rotattn_build_tables(const rotattn_params* p, const float* rot_host, float* coef_host);

/* Bytes of scratch the device entry points need.  which = 0: INT4 path (shared by prepare_qk,
 * quant_v and fwd_int4: widened int8 copies of the Q/K codes [B,H,N,D] and of the V codes
 * transposed [B,H,D,ceil128(N)]); which = 1: FP16 path (transposed V copy). */
size_t rotattn_workspace_bytes(const rotattn_params* p, int which);

/* Mixed-precision fallback policy: FP16 on the first/last sampling steps and the
 * first/last DiT blocks (and on heads flagged in fp16_head_mask), INT4 elsewhere.  Pure host logic. */
typedef struct rotattn_policy {
  int32_t n_steps, n_blocks, first_steps, last_steps, first_blocks, last_blocks;
  const uint8_t* fp16_head_mask;      /* host [H] or NULL */
} rotattn_policy;
/* 0 = INT4, 1 = FP16, negative = error. */
int rotattn_policy_select(const rotattn_policy* pol, int32_t step, int32_t block, int32_t head);
/* Fill sel_int4 / sel_fp16 (host int32, capacity B*H each) with the b*H+h indices each kernel must run
 * for this (step, block); counts are returned through n_int4 / n_fp16. */
int rotattn_policy_split_heads(const rotattn_policy* pol, int32_t step, int32_t block, int32_t B, int32_t H,
                               int32_t* sel_int4, int32_t* n_int4, int32_t* sel_fp16, int32_t* n_fp16);

const char* rotattn_strerror(int status);
/* Text of the last CUDA error seen by this thread's calls (empty string if none). */
const char* rotattn_last_cuda_error(void);

/* ---- device entry points ---------------------------------------------------------------------- */

/* Prologue, steps a1+a2: y = x (M R) — 3D RoPE (L58-62) together with the 2x2 block rotation
 * (INTERLEAVED: merged table, Eq.7; HALF: second stage in the same register pass, Eq.8) in fp32 with
 * one rounding per operation (no FMA contraction), then per-token symmetric INT4 (L190, reading 10):
 *   amax = max_d |y_d|; scale = amax/7; code_d = clamp(rne(y_d * (7/amax)), -7, 7); amax = 0 -> zeros.
 * coef_dev: device copy of the table from rotattn_build_tables.
 * rot_dev : device float [D/2][4] blocks used by HALF mode, or NULL for H_2.  Ignored otherwise.
 * Q,K     : fp16 [B,H,N,D].
 * Q4,K4   : out, packed codes [B,H,N,D/2] uint8: byte i = (code_{2i} & 0xF) | (code_{2i+1} & 0xF) << 4.
 * Qs,Ks   : out, fp32 scales [B,H,N].
 * Qrope16,Krope16 : optional out (may be NULL), y rounded once to fp16 [B,H,N,D] (input of fwd_fp16).
 * workspace: optional (may be NULL): if given (>= rotattn_workspace_bytes(p,0)) the widened int8
 *           copies used by fwd_int4 are also written (then pass ROTATTN_WS_HAS_QK to fwd_int4). */
int rotattn_prepare_qk(const rotattn_params* p, const float* coef_dev, const float* rot_dev,
                       const void* Q, const void* K,
                       uint8_t* Q4, float* Qs, uint8_t* K4, float* Ks,
                       void* Qrope16, void* Krope16,
                       void* workspace, size_t ws_bytes, void* stream);

/* Step a3: per-group symmetric INT4 of Hadamard-domain V (L190; Eq.14: H is folded into
 * W_v offline, so V arrives transformed).  One scale per (128 consecutive tokens, channel); the ragged
 * last group uses the tokens that exist.
 * V : fp16 [B,H,N,D].  V4: out packed [B,H,N,D/2].  Vs: out fp32 [B,H,ceil(N/128),D].
 * workspace as for prepare_qk (then pass ROTATTN_WS_HAS_V to fwd_int4). */
int rotattn_quant_v(const rotattn_params* p, const void* V, uint8_t* V4, float* Vs,
                    void* workspace, size_t ws_bytes, void* stream);

/* Steps a4-a9: INT4 FlashAttention forward (§4.2).
 *   S = Q4 K4^T as an integer tensor-core MMA with int32 accumulation (L157);
 *   s_ij = acc * Qs_i * Ks_j / sqrt(D); per KV block of 128 keys: block row max, P^ = exp(s - max),
 *   u = rne(15 P^) in {0..15} (Eq.12: scale 15, zero-point -8, stored unsigned u = c + 8; SYM7: rne(7 P^));
 *   integer P~V with int32 accumulation; O <- alpha O + beta (Vs/15) pv in fp32; epilogue O/l -> fp16.
 * Q4..Vs: the outputs of prepare_qk / quant_v.   O: out fp16 [B,H,N,D] (only selected heads written).
 * head_sel: device int32 [n_sel] of b*H+h indices to process, or NULL (all B*H heads, n_sel ignored).
 * workspace: required, >= rotattn_workspace_bytes(p,0).  ws_state: ROTATTN_WS_HAS_QK|ROTATTN_WS_HAS_V
 *   if this workspace was passed to prepare_qk / quant_v with the same params; missing copies are rebuilt
 *   from the packed buffers by an unpack kernel first. */
int rotattn_fwd_int4(const rotattn_params* p,
                     const uint8_t* Q4, const float* Qs, const uint8_t* K4, const float* Ks,
                     const uint8_t* V4, const float* Vs, void* O,
                     const int32_t* head_sel, int32_t n_sel,
                     void* workspace, size_t ws_bytes, int32_t ws_state, void* stream);

/* Same computation for ONE (bh, query tile of 128 rows), additionally dumping the int32 S accumulators
 * and the P codes (parity tests only; not on the timed path).
 * S_dump: int32 [128, ceil128(N)], P_dump: uint8 [128, ceil128(N)], O_tile: fp16 [128, D] (rows >= N untouched). */
int rotattn_fwd_int4_debug(const rotattn_params* p,
                           const uint8_t* Q4, const float* Qs, const uint8_t* K4, const float* Ks,
                           const uint8_t* V4, const float* Vs,
                           int32_t bh, int32_t q_tile, int32_t* S_dump, uint8_t* P_dump, void* O_tile,
                           void* workspace, size_t ws_bytes, int32_t ws_state, void* stream);

/* Step a10: FP16 FlashAttention forward, the fallback precision and the speed baseline (L21, L192, L267).
 * Q16,K16: fp16 RoPE'd Q,K [B,H,N,D] (Qrope16/Krope16 of prepare_qk); V16: fp16 V [B,H,N,D]; fp32 accumulate.
 * workspace: required, >= rotattn_workspace_bytes(p,1). */
int rotattn_fwd_fp16(const rotattn_params* p, const void* Q16, const void* K16, const void* V16, void* O,
                     const int32_t* head_sel, int32_t n_sel,
                     void* workspace, size_t ws_bytes, void* stream);

/* Measurement aid: dense 8-bit GEMM C[M,N] = A[M,K] * B[N,K]^T on the same tcgen05 path the attention
 * kernel uses; used to MEASURE the dense INT8 tensor peak that the roofline of fwd_int4 is quoted against.
 * M multiple of 128, N multiple of 256, K multiple of 128.  A,B: device, row-major, 1 byte per element.
 *   mode 0: kind::i8, A and B signed int8, C int32.
 *   mode 1: kind::f8f6f4, A and B E4M3 bit patterns, C float (fp32 accumulators).
 *   mode 2: kind::i8 with A (UNSIGNED u8) staged through tensor memory, B signed; M=N=K=128 only
 *           (checks the TMEM A-operand layout used for the P~V product), C int32. */
int rotattn_probe_gemm8(int32_t M, int32_t N, int32_t K, const void* A, const void* B, void* C,
                        int32_t mode, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* ROTATTN_H_ */
