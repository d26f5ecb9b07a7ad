// Host-side logic of librotattn: validation, coefficient tables (a0), workspace sizing,
// fallback policy (a11), error text.  No device code here.
#include <cmath>
#include <cstdio>
#include <cstring>
#include "common.cuh"

namespace rotattn {

static thread_local char g_err[512] = "";

void set_cuda_error(cudaError_t e, const char* where) {
  snprintf(g_err, sizeof(g_err), "%s: %s (%s)", where, cudaGetErrorString(e), cudaGetErrorName(e));
}
void set_error_text(const char* text) { snprintf(g_err, sizeof(g_err), "%s", text); }

int check_device_sm100() {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { set_cuda_error(e, "cudaGetDevice"); return ROTATTN_ERR_CUDA; }
  int major = 0;
  e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  if (e != cudaSuccess) { set_cuda_error(e, "cudaDeviceGetAttribute"); return ROTATTN_ERR_CUDA; }
  if (major != 10) { set_error_text("device is not sm_100; there is no other backend"); return ROTATTN_ERR_UNSUPPORTED; }
  return ROTATTN_OK;
}

}  // namespace rotattn

using namespace rotattn;

extern "C" {

int rotattn_abi_version(void) { return ROTATTN_ABI_VERSION; }

int rotattn_validate(const rotattn_params* p) {
  if (!p) return ROTATTN_ERR_INVALID_ARG;
  if (p->B < 1 || p->H < 1 || p->N < 1) return ROTATTN_ERR_INVALID_ARG;
  if (p->grid_t < 1 || p->grid_h < 1 || p->grid_w < 1) return ROTATTN_ERR_INVALID_ARG;
  if ((int64_t)p->grid_t * p->grid_h * p->grid_w > (int64_t)p->N) return ROTATTN_ERR_INVALID_ARG;
  if (p->pairs_t < 1 || p->pairs_h < 1 || p->pairs_w < 1) return ROTATTN_ERR_INVALID_ARG;
  if (p->D != 64 && p->D != 128) return ROTATTN_ERR_UNSUPPORTED;
  if (p->pairs_t + p->pairs_h + p->pairs_w != p->D / 2) return ROTATTN_ERR_INVALID_ARG;
  if (!(p->rope_base > 1.0f)) return ROTATTN_ERR_INVALID_ARG;
  if (p->rot_mode < 0 || p->rot_mode > 3) return ROTATTN_ERR_INVALID_ARG;
  if (p->p_mode < 0 || p->p_mode > 1) return ROTATTN_ERR_INVALID_ARG;
  if (p->p_norm < 0 || p->p_norm > 1) return ROTATTN_ERR_INVALID_ARG;
  if (p->v_scale < 0 || p->v_scale > 1 || p->smooth < 0 || p->smooth > 1 || p->qk_group < 1) return ROTATTN_ERR_INVALID_ARG;
  if (p->qk_group != 1 && p->qk_group != kTile) return ROTATTN_ERR_UNSUPPORTED;
  if (p->v_group != kTile || p->kv_block != kTile) return ROTATTN_ERR_UNSUPPORTED;
  // the RUNNING normaliser and smoothing are built for the paper's granularity only (per-token Q/K, per-channel V scales)
  const bool f1 = p->qk_group != 1 || p->v_scale != ROTATTN_VSCALE_CHANNEL;
  if (f1 && (p->p_norm == ROTATTN_NORM_RUNNING || p->smooth)) return ROTATTN_ERR_UNSUPPORTED;
  if (p->smooth && p->p_norm == ROTATTN_NORM_RUNNING) return ROTATTN_ERR_UNSUPPORTED;
  return ROTATTN_OK;
}

size_t rotattn_table_floats(const rotattn_params* p) {
  if (rotattn_validate(p) != ROTATTN_OK) return 0;
  return 4 * ((size_t)(p->grid_t + 1) * p->pairs_t + (size_t)(p->grid_h + 1) * p->pairs_h +
              (size_t)(p->grid_w + 1) * p->pairs_w);
}

int rotattn_build_tables(const rotattn_params* p, const float* rot_host, float* coef_host) {
  int st = rotattn_validate(p);
  if (st != ROTATTN_OK) return st;
  if (!coef_host) return ROTATTN_ERR_INVALID_ARG;
  const int npairs = p->D / 2;
  // R_i in O(2) (Eq.3); default H_2 (Eq.4)
  double rot[64][4];
  const double h = 1.0 / std::sqrt(2.0);
  for (int k = 0; k < npairs; ++k) {
    if (rot_host) {
      for (int e = 0; e < 4; ++e) rot[k][e] = (double)rot_host[4 * k + e];
    } else {
      rot[k][0] = h; rot[k][1] = h; rot[k][2] = h; rot[k][3] = -h;
    }
    const double a = rot[k][0], b = rot[k][1], c = rot[k][2], d = rot[k][3];
    const double e00 = a * a + c * c - 1.0, e01 = a * b + c * d, e11 = b * b + d * d - 1.0;
    if (std::fabs(e00) > 1e-5 || std::fabs(e01) > 1e-5 || std::fabs(e11) > 1e-5) return ROTATTN_ERR_NOT_ORTHOGONAL;
  }
  const int len[3] = {p->grid_t, p->grid_h, p->grid_w};
  const int P[3] = {p->pairs_t, p->pairs_h, p->pairs_w};
  size_t row = 0;
  int gpair = 0;
  for (int a = 0; a < 3; ++a) {
    for (int pos = 0; pos <= len[a]; ++pos) {
      for (int k = 0; k < P[a]; ++k) {
        double m00 = 1.0, m01 = 0.0, m10 = 0.0, m11 = 1.0;
        if (pos < len[a]) {
          // f = base^(-k/P_a) (reading 2); M = [[c, s], [-s, c]] (reading 1, row-vector convention)
          const double f = std::pow((double)p->rope_base, -(double)k / (double)P[a]);
          const double th = (double)pos * f;
          const double c = std::cos(th), s = std::sin(th);
          m00 = c; m01 = s; m10 = -s; m11 = c;
        }
        double o00 = m00, o01 = m01, o10 = m10, o11 = m11;
        if (p->rot_mode == ROTATTN_ROT_INTERLEAVED) {     // A = M R (Eq.7)
          const double* r = rot[gpair + k];
          o00 = m00 * r[0] + m01 * r[2];
          o01 = m00 * r[1] + m01 * r[3];
          o10 = m10 * r[0] + m11 * r[2];
          o11 = m10 * r[1] + m11 * r[3];
        }
        coef_host[4 * row + 0] = (float)o00;
        coef_host[4 * row + 1] = (float)o01;
        coef_host[4 * row + 2] = (float)o10;
        coef_host[4 * row + 3] = (float)o11;
        ++row;
      }
    }
    gpair += P[a];
  }
  return ROTATTN_OK;
}

size_t rotattn_workspace_bytes(const rotattn_params* p, int which) {
  if (rotattn_validate(p) != ROTATTN_OK) return 0;
  if (which == 0 || which == 1) return WsInt4(*p).total;      // prepare_qk / quant_v and fwd_int4 share one workspace
  if (which == 2) return 0;                                     // fwd_fp16 reads V in place (MN-major B operand): no scratch
  return 0;
}

int rotattn_policy_select(const rotattn_policy* pol, int32_t step, int32_t block, int32_t head) {
  if (!pol || pol->n_steps < 1 || pol->n_blocks < 1) return ROTATTN_ERR_INVALID_ARG;
  if (step < 0 || step >= pol->n_steps || block < 0 || block >= pol->n_blocks || head < 0) return ROTATTN_ERR_INVALID_ARG;
  if (pol->first_steps < 0 || pol->last_steps < 0 || pol->first_blocks < 0 || pol->last_blocks < 0) return ROTATTN_ERR_INVALID_ARG;
  if (step < pol->first_steps || step >= pol->n_steps - pol->last_steps) return 1;
  if (block < pol->first_blocks || block >= pol->n_blocks - pol->last_blocks) return 1;
  if (pol->fp16_head_mask) {
    if (head >= pol->n_heads) return ROTATTN_ERR_INVALID_ARG;      // the mask holds n_heads entries
    if (pol->fp16_head_mask[head]) return 1;
  }
  return 0;
}

int rotattn_policy_split_heads(const rotattn_policy* pol, int32_t step, int32_t block, int32_t B, int32_t H,
                               int32_t* sel_int4, int32_t* n_int4, int32_t* sel_fp16, int32_t* n_fp16) {
  if (!pol || !sel_int4 || !n_int4 || !sel_fp16 || !n_fp16 || B < 1 || H < 1) return ROTATTN_ERR_INVALID_ARG;
  if (pol->fp16_head_mask && H > pol->n_heads) return ROTATTN_ERR_INVALID_ARG;
  int a = 0, b = 0;
  for (int bi = 0; bi < B; ++bi)
    for (int h = 0; h < H; ++h) {
      int r = rotattn_policy_select(pol, step, block, h);
      if (r < 0) return r;
      if (r == 0) sel_int4[a++] = bi * H + h; else sel_fp16[b++] = bi * H + h;
    }
  *n_int4 = a;
  *n_fp16 = b;
  return ROTATTN_OK;
}

const char* rotattn_strerror(int status) {
  switch (status) {
    case ROTATTN_OK: return "ok";
    case ROTATTN_ERR_INVALID_ARG: return "invalid argument";
    case ROTATTN_ERR_UNSUPPORTED: return "unsupported configuration or device (sm_100a only, no fallback)";
    case ROTATTN_ERR_NOT_ORTHOGONAL: return "rotation blocks are not orthogonal";
    case ROTATTN_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
    case ROTATTN_ERR_CUDA: return "CUDA error";
    default: return "unknown status";
  }
}

const char* rotattn_last_cuda_error(void) { return g_err; }

}  // extern "C"
