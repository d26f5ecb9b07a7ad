// rotattn_fwd_int4 / rotattn_fwd_int4_debug: host side of the INT4 attention kernels (argument checks, workspace
// copies, tensor maps, variant dispatch).  The kernel is in fwd_int4_kernel.cuh (ROWBLOCK and RUNNING normalisers).
#include <cmath>
#include <cstdio>
#include "fwd_int4.cuh"

using namespace rotattn;

namespace {

int fwd_int4_common(const rotattn_params* p, const uint8_t* Q4, const float* Qs, const uint8_t* K4, const float* Ks,
                    const uint8_t* V4, const float* Vs, void* O, const int32_t* head_sel, int32_t n_sel,
                    void* workspace, size_t ws_bytes, int32_t ws_state, void* stream,
                    bool debug, int32_t bh, int32_t q_tile, int32_t* S_dump, uint8_t* P_dump, int32_t* PV_dump) {
  int st = rotattn_validate(p);
  if (st != ROTATTN_OK) return st;
  if (!Q4 || !Qs || !K4 || !Ks || !V4 || !Vs || !O || !workspace) return ROTATTN_ERR_INVALID_ARG;
  if (((uintptr_t)Vs & 15) || ((uintptr_t)O & 15)) return ROTATTN_ERR_INVALID_ARG;      // bulk copies / 16-byte stores
  const int BH = p->B * p->H;
  const int nblk = ceil_div(p->N, kTile);
  if (head_sel && (n_sel < 1 || n_sel > BH)) return ROTATTN_ERR_INVALID_ARG;
  if (debug && (bh < 0 || bh >= BH || q_tile < 0 || q_tile >= nblk || !S_dump || !P_dump)) return ROTATTN_ERR_INVALID_ARG;
  constexpr int kSmoothBits = ROTATTN_WS_HAS_QK | ROTATTN_WS_HAS_V | ROTATTN_WS_HAS_STATS;
  if (p->smooth && (ws_state & kSmoothBits) != kSmoothBits) {
    // the smoothing state (means, per-key correction) exists only in the prologue's workspace, and only if smooth_stats ran on it
    set_error_text("rotattn_fwd_int4: smooth = 1 needs ws_state = HAS_QK | HAS_V | HAS_STATS (rotattn_smooth_stats, prepare_qk and "
                   "quant_v must have run on this workspace)");
    return ROTATTN_ERR_INVALID_ARG;
  }
  WsInt4 ws(*p);
  if (ws_bytes < ws.total) return ROTATTN_ERR_WORKSPACE_TOO_SMALL;
  if ((st = check_device_sm100()) != ROTATTN_OK) return st;
  cudaStream_t cs = (cudaStream_t)stream;
  int8_t* q8 = (int8_t*)workspace + ws.q8;
  int8_t* k8 = (int8_t*)workspace + ws.k8;
  int8_t* v8t = (int8_t*)workspace + ws.v8t;
  float* ksp = (float*)((uint8_t*)workspace + ws.ksp);
  if (!(ws_state & ROTATTN_WS_HAS_QK)) {
    if ((st = launch_unpack_qk(*p, Q4, q8, cs)) != ROTATTN_OK) return st;
    if ((st = launch_unpack_qk(*p, K4, k8, cs)) != ROTATTN_OK) return st;
    if (p->qk_group == 1 && (st = launch_pad_ks(*p, Ks, ksp, ws.npad, cs)) != ROTATTN_OK) return st;
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
  a.Qs = Qs; a.Ks = Ks; a.KsP = ksp; a.Vs = Vs; a.O = (__half*)O; a.head_sel = head_sel;
  a.KcP = (const float*)((uint8_t*)workspace + ws.kcp);
  a.means = (const float*)((uint8_t*)workspace + ws.means);
  a.S_dump = S_dump; a.P_dump = P_dump; a.PV_dump = PV_dump;
  a.N = p->N; a.nblk = nblk; a.npad = ws.npad; a.dbg_bh = bh; a.dbg_qtile = q_tile;
  a.scale_log2 = (float)(1.4426950408889634 / std::sqrt((double)p->D) * (double)kAccScale);   // S arrives as acc * 2^-18
  dim3 grid(debug ? 1 : nblk, debug ? 1 : (head_sel ? n_sel : BH));
  if (debug) return launch_fwd_int4_debug(*p, tq, tk, tv, a, grid, cs);
  return p->D == 128 ? launch_fwd_int4_d128(*p, tq, tk, tv, a, grid, cs) : launch_fwd_int4_d64(*p, tq, tk, tv, a, grid, cs);
}

}  // namespace

extern "C" int rotattn_fwd_int4(const rotattn_params* p, const uint8_t* Q4, const float* Qs, const uint8_t* K4,
                                const float* Ks, const uint8_t* V4, const float* Vs, void* O, const int32_t* head_sel,
                                int32_t n_sel, void* workspace, size_t ws_bytes, int32_t ws_state, void* stream) {
  return fwd_int4_common(p, Q4, Qs, K4, Ks, V4, Vs, O, head_sel, n_sel, workspace, ws_bytes, ws_state, stream,
                         false, 0, 0, nullptr, nullptr, nullptr);
}

extern "C" int rotattn_fwd_int4_debug(const rotattn_params* p, const uint8_t* Q4, const float* Qs, const uint8_t* K4,
                                      const float* Ks, const uint8_t* V4, const float* Vs, int32_t bh, int32_t q_tile,
                                      int32_t* S_dump, uint8_t* P_dump, int32_t* PV_dump, void* O_tile, void* workspace,
                                      size_t ws_bytes, int32_t ws_state, void* stream) {
  return fwd_int4_common(p, Q4, Qs, K4, Ks, V4, Vs, O_tile, nullptr, 0, workspace, ws_bytes, ws_state, stream,
                         true, bh, q_tile, S_dump, P_dump, PV_dump);
}
