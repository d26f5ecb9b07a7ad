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

/* Version of this binary interface.  It changes whenever a struct below gains, loses or moves a field or an enum value is
 * renumbered (version 2 appended v_scale / smooth to rotattn_params, inserted n_heads into rotattn_policy and renumbered
 * the `which` of rotattn_workspace_bytes; version 3 adds rotattn_fwd_int4_static, ROTATTN_WS_HAS_STATS and this query).  The structs carry no
 * size field, so a caller built against another version would be read wrongly without any error: compare
 * rotattn_abi_version() with the ROTATTN_ABI_VERSION you compiled against once, before the first other call. */
#define ROTATTN_ABI_VERSION 3
int rotattn_abi_version(void);

typedef enum rotattn_status {
  ROTATTN_OK = 0,
  ROTATTN_ERR_INVALID_ARG = -1,         /* NULL pointer, sum(pairs) != D/2, t*h*w > N, n_sel out of range */
  ROTATTN_ERR_UNSUPPORTED = -2,         /* D not in {64,128}, kv_block != 128, v_group != 128, qk_group not in {1,128},
                                           p_norm = RUNNING or smooth with a non-default granularity, device is not sm_100 */
  ROTATTN_ERR_NOT_ORTHOGONAL = -3,      /* max|R_i^T R_i - I| > 1e-5 */
  ROTATTN_ERR_WORKSPACE_TOO_SMALL = -4,
  ROTATTN_ERR_CUDA = -5                 /* a CUDA runtime/driver call failed; see rotattn_last_cuda_error() */
} rotattn_status;

enum { ROTATTN_ROT_NONE = 0, ROTATTN_ROT_INTERLEAVED = 1, ROTATTN_ROT_HALF = 2,
       ROTATTN_ROT_FULL = 3 /* the paper's "Full" ablation baseline: dense D x D Hadamard after RoPE */ };
enum { ROTATTN_P_ASYM15 = 0, ROTATTN_P_SYM7 = 1 };
enum { ROTATTN_NORM_ROWBLOCK = 0, ROTATTN_NORM_RUNNING = 1 };
enum { ROTATTN_VSCALE_CHANNEL = 0 /* one V scale per (128-token group, channel): DESIGN.md reading 11 */,
       ROTATTN_VSCALE_GROUP = 1   /* one V scale per 128-token group */ };
/* ws_state bits for rotattn_fwd_int4 */
enum { ROTATTN_WS_HAS_QK = 1, ROTATTN_WS_HAS_V = 2,
       ROTATTN_WS_HAS_STATS = 4 /* smooth = 1 only: the caller states that rotattn_smooth_stats ran on THIS workspace for THESE
                                   Q, K, V before prepare_qk / quant_v.  The library cannot see it (it never reads device memory
                                   on the host), and stale or missing means give a silently wrong O - so fwd_int4 refuses
                                   smooth = 1 unless the caller has said so. */ };

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
  int32_t qk_group;                   /* tokens per Q/K scale: 1 = per-token (L190, the paper's setting) or 128 = one scale
                                         per 128-token block (north_star "per-block scales") */
  int32_t v_group;                    /* tokens per V scale group (L190, reading 11).  Only 128 is built. */
  int32_t kv_block;                   /* P-normalisation block (L157, reading 18).  Only 128 is built. */
  int32_t v_scale;                    /* ROTATTN_VSCALE_CHANNEL (default) | ROTATTN_VSCALE_GROUP */
  int32_t smooth;                     /* 0 | 1: subtract the token mean of Q, K, V before quantisation ("we first
                                         perform smoothing on Q, K, V"; L40, L52), see rotattn_smooth_* below */
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

/* Bytes of scratch the device entry points need.  which = 0 (prepare_qk / quant_v / smooth_stats) and which = 1
 * (fwd_int4) are one and the same INT4-path workspace: sign-magnitude operand bytes of the Q/K codes [B,H,N,128] and
 * of the V codes transposed [B,H,D,ceil128(N)] (one byte per code = the E4M3 bit pattern of code * 2^-9), the key
 * scales padded to whole blocks, and the smoothing state.  which = 2: FP16 path - 0 since ABI version 3 (V is read in place). */
size_t rotattn_workspace_bytes(const rotattn_params* p, int which);

/* Mixed-precision fallback policy: FP16 on the first/last sampling steps and the
 * first/last DiT blocks (and on heads flagged in fp16_head_mask), INT4 elsewhere.  Pure host logic. */
typedef struct rotattn_policy {
  int32_t n_steps, n_blocks, first_steps, last_steps, first_blocks, last_blocks;
  int32_t n_heads;                    /* entries of fp16_head_mask (ignored when the mask is NULL) */
  const uint8_t* fp16_head_mask;      /* host [n_heads] or NULL */
} rotattn_policy;
/* 0 = INT4, 1 = FP16, negative = error (INVALID_ARG also for head >= n_heads when a mask is given). */
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
 * Qs,Ks   : out, fp32 scales [B,H,N]  (qk_group = 128: one scale per 128-token block, [B,H,ceil(N/128)], amax over
 *           the block's tokens and channels).
 * Qrope16,Krope16 : optional out (may be NULL), y rounded once to fp16 [B,H,N,D] (input of fwd_fp16; never smoothed).
 * rot_mode = FULL (the paper's "Full" baseline, L208): after RoPE, y <- y H_D / sqrt(D) as a Sylvester butterfly
 *           (strides 1, 2, .., D/2; (a,b) -> (a+b, a-b); one multiplication by fl(1/sqrt(D)) at the end).
 * smooth = 1: rotattn_smooth_stats must have run on this workspace first; y - mean_n(y) is quantised instead of y, and
 *           the per-key correction mean(y_Q) . (y_K - mean(y_K)) is stored in the workspace for fwd_int4.
 * workspace: optional (may be NULL, required for smooth): if given (>= rotattn_workspace_bytes(p,0)) the operand
 *           bytes and padded key scales used by fwd_int4 are also written (then pass ROTATTN_WS_HAS_QK to fwd_int4). */
int rotattn_prepare_qk(const rotattn_params* p, const float* coef_dev, const float* rot_dev,
                       const void* Q, const void* K,
                       uint8_t* Q4, float* Qs, uint8_t* K4, float* Ks,
                       void* Qrope16, void* Krope16,
                       void* workspace, size_t ws_bytes, void* stream);

/* Step a3: per-group symmetric INT4 of Hadamard-domain V (L190; Eq.14: H is folded into
 * W_v offline, so V arrives transformed).  One scale per (128 consecutive tokens, channel); the ragged
 * last group uses the tokens that exist.
 * V : fp16 [B,H,N,D].  V4: out packed [B,H,N,D/2].  Vs: out fp32 [B,H,ceil(N/128),D], 16-byte aligned
 *   (v_scale = GROUP: one scale per group, [B,H,ceil(N/128)], amax over the group's tokens and channels).
 * smooth = 1: v - mean_n(v) is quantised (the mean is added back to O by fwd_int4).
 * workspace as for prepare_qk (then pass ROTATTN_WS_HAS_V to fwd_int4). */
int rotattn_quant_v(const rotattn_params* p, const void* V, uint8_t* V4, float* Vs,
                    void* workspace, size_t ws_bytes, void* stream);

/* Smoothing pre-pass ("we first perform smoothing on Q, K, V", L40, L52): column means
 * over the N tokens of y_Q, y_K (after RoPE and rotation) and of V, per (b,h), kept in the workspace.  Needed once
 * before rotattn_prepare_qk / rotattn_quant_v when p->smooth = 1.  The sums are taken in fixed point (units of 2^-20
 * for y, 2^-24 for the fp16 V) so that they do not depend on the order of summation:
 *   mean = fl32( fp64(sum_n rne(y_n * 2^20)) / (N * 2^20) ).
 * Exactness of the shifts: K - mean(K) leaves softmax(QK^T) unchanged; (Q - mean Q) K'^T + mean(Q) K'^T = Q K'^T, the
 * rank-1 term is added to S in fp32; softmax(.)(V - mean V) + mean V = softmax(.) V. */
int rotattn_smooth_stats(const rotattn_params* p, const float* coef_dev, const float* rot_dev,
                         const void* Q, const void* K, const void* V,
                         void* workspace, size_t ws_bytes, void* stream);
/* Copies the smoothing state out of the workspace (either pointer may be NULL):
 * means_out fp32 [B,H,3,D] (y_Q, y_K, V); kcorr_out fp32 [B,H,N] = mean(y_Q) . (y_K - mean y_K) * log2(e)/sqrt(D). */
int rotattn_smooth_read(const rotattn_params* p, const void* workspace, size_t ws_bytes,
                        float* means_out, float* kcorr_out, void* stream);

/* Steps a4-a9: INT4 FlashAttention forward (PAPER.md 4.2 L155-170).
 *   S = Q4 K4^T on the tensor cores with exact integer accumulation (L157): sm_100a has no 4-bit integer MMA and its
 *   8-bit integer kind returns int32 that would have to be converted three times per element, so the codes travel as
 *   the E4M3 bit patterns of code * 2^-9 through tcgen05 kind::f8f6f4 and the fp32 accumulators hold acc * 2^-18
 *   exactly (|acc| <= 13440 < 2^24; adversarial tests in tests/test_gpu_probe.py).
 *   s_ij = acc * Qs_i * Ks_j / sqrt(D); per KV block of 128 keys: block row max, P^ = exp(s - max),
 *   u = rne(15 P^) in {0..15} (Eq.12: scale 15, zero-point -8, stored unsigned u = c + 8; SYM7: rne(7 P^));
 *   integer P~V, same exact path; O <- alpha O + beta (Vs/15) pv in fp32; epilogue O/l -> fp16.
 * Q4..Vs: the outputs of prepare_qk / quant_v (shapes follow qk_group / v_scale).
 * O: out fp16 [B,H,N,D], 16-byte aligned (only selected heads written).
 * head_sel: device int32 [n_sel] of b*H+h indices to process, or NULL (all B*H heads, n_sel ignored).
 * workspace: required, >= rotattn_workspace_bytes(p,1).  ws_state: ROTATTN_WS_HAS_QK|ROTATTN_WS_HAS_V
 *   if this workspace was passed to prepare_qk / quant_v with the same params; missing copies are rebuilt
 *   from the packed buffers by an unpack kernel first (smooth = 1 needs both bits and ROTATTN_WS_HAS_STATS: its state
 *   exists only there; anything less returns ROTATTN_ERR_INVALID_ARG). */
int rotattn_fwd_int4(const rotattn_params* p,
                     const uint8_t* Q4, const float* Qs, const uint8_t* K4, const float* Ks,
                     const uint8_t* V4, const float* Vs, void* O,
                     const int32_t* head_sel, int32_t n_sel,
                     void* workspace, size_t ws_bytes, int32_t ws_state, void* stream);

/* rotattn_fwd_int4 for callers that cannot supply a workspace and must not allocate one.
 *
 * Typical callers: a DiT serving process whose own arena took all of HBM at start-up and which forbids cudaMalloc on the
 * request path (an allocation there synchronises the device, stalls the other streams and may fail outright), or an
 * operator plugged into a foreign runtime through an "inputs, outputs" signature with no workspace slot.
 *
 * Same computation and same kernels as rotattn_fwd_int4 with ws_state = 0 (steps a4-a9, PAPER.md 4.2 L155-170): the
 * operand copies are rebuilt from the packed Q4/K4/V4 on every call.  The workspace is a device array of
 * ROTATTN_STATIC_WS_BYTES built into librotattn.so; every GPU that loads the library carries it until the process ends.
 *  - Limit: rotattn_workspace_bytes(p, 1) <= ROTATTN_STATIC_WS_BYTES (roughly B*H*N <= 21 000 tokens at D = 128, e.g. one
 *    head of a 480p video or all 12 heads of a 1 700-token clip).  Larger shapes return ROTATTN_ERR_WORKSPACE_TOO_SMALL
 *    (text in rotattn_last_cuda_error()); split them over heads with separate per-head calls.
 *  - smooth = 1 returns ROTATTN_ERR_UNSUPPORTED (its state lives in the prologue's workspace).
 *  - This call allocates nothing and frees nothing: no cudaMalloc / cudaFree / allocating library routine, here or below.
 *  - The first call on each device looks up the array's device address (cudaGetSymbolAddress, that device current) and
 *    remembers it; make that first call during start-up, before any stream capture begins on that device.
 *  - ALL calls on a device share the one array, and it keeps what the previous call left.  Each call rewrites every byte
 *    it later reads, so stale contents are harmless and nothing needs clearing - but two calls that overlap on the GPU
 *    (different streams, no ordering between them) race on it and corrupt each other.  Calls on one stream are safe.
 * Arguments as for rotattn_fwd_int4 (caller-owned device pointers; O 16-byte aligned; head_sel may be NULL). */
#define ROTATTN_STATIC_WS_BYTES (8u << 20)
int rotattn_fwd_int4_static(const rotattn_params* p,
                            const uint8_t* Q4, const float* Qs, const uint8_t* K4, const float* Ks,
                            const uint8_t* V4, const float* Vs, void* O,
                            const int32_t* head_sel, int32_t n_sel, void* stream);

/* Step a10: FP16 FlashAttention forward, the fallback precision and the speed baseline (L21, L192, L267).
 * Q16,K16: fp16 RoPE'd Q,K [B,H,N,D] (Qrope16/Krope16 of prepare_qk); V16: fp16 V [B,H,N,D]; fp32 accumulate.
 * Q16, K16, V16, O: 16-byte aligned.  workspace / ws_bytes: ignored (kept for the ABI; the kernel needs no scratch: V is fed to the
 * tensor cores as it lies in memory, as an MN-major operand); may be NULL / 0. */
int rotattn_fwd_fp16(const rotattn_params* p, const void* Q16, const void* K16, const void* V16, void* O,
                     const int32_t* head_sel, int32_t n_sel,
                     void* workspace, size_t ws_bytes, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* ROTATTN_H_ */
