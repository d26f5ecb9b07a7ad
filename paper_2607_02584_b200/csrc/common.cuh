// Shared host/device declarations of librotattn (not part of the public ABI).
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include <stddef.h>
#include <atomic>
#include "rotattn_debug.h"

namespace rotattn {

constexpr int kTile = 128;        // query tile = KV block = V group (readings 11, 18)
constexpr int kQKRowBytes = 128;  // widened int8 Q/K rows are always 128 B (D=64 rows are zero-padded)

inline __host__ __device__ int ceil_div(int a, int b) { return (a + b - 1) / b; }
inline __host__ __device__ size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Layout of the INT4-path workspace (rotattn_workspace_bytes(p, 0) == (p, 1)): library-private derived copies written by
// prepare_qk / quant_v (or rebuilt from the packed public buffers by the unpack kernels).
struct WsInt4 {
  size_t q8, k8, v8t;     // operand bytes: Q8,K8 [BH,N,128], V8^T [BH,D,npad]
  size_t ksp;             // float [BH,npad]: per-token key scales padded to whole 128-key blocks (bulk-copied next to the K tiles)
  size_t kcp;             // float [BH,npad]: smoothing only, per-key correction mean(Q).K'_j / sqrt(D) * log2e (added to S in fp32)
  size_t sums;            // int64 [BH,3,D]: smoothing only, fixed-point column sums of y_Q, y_K, V
  size_t means;           // float [BH,3,D]: smoothing only, the column means
  size_t total;
  int npad;
  __host__ explicit WsInt4(const rotattn_params& p) {
    size_t bh = (size_t)p.B * p.H;
    npad = ceil_div(p.N, kTile) * kTile;
    size_t qk = align_up(bh * (size_t)p.N * kQKRowBytes, 1024);
    q8 = 0;
    k8 = q8 + qk;
    v8t = k8 + qk;
    ksp = v8t + align_up(bh * (size_t)p.D * npad, 1024);
    kcp = ksp + align_up(bh * (size_t)npad * 4, 1024);
    sums = kcp + align_up(bh * (size_t)npad * 4, 1024);
    means = sums + align_up(bh * 3 * (size_t)p.D * 8, 1024);
    total = means + align_up(bh * 3 * (size_t)p.D * 4, 1024);
  }
};

// error plumbing
void set_cuda_error(cudaError_t e, const char* where);
void set_error_text(const char* text);
int check_device_sm100();   // ROTATTN_OK or ROTATTN_ERR_UNSUPPORTED / ROTATTN_ERR_CUDA

#define ROTATTN_CUDA_TRY(expr)                                   \
  do {                                                           \
    cudaError_t _e = (expr);                                     \
    if (_e != cudaSuccess) {                                     \
      ::rotattn::set_cuda_error(_e, #expr);                      \
      return ROTATTN_ERR_CUDA;                                   \
    }                                                            \
  } while (0)

// "Has the one-time set-up of this kernel run on device d?"  cudaFuncSetAttribute is per device (per context), so a flag
// per process would leave the second GPU of a single-process multi-GPU host without its shared-memory opt-in.  One bit per
// device ordinal; running the set-up twice from two racing host threads is harmless (it is idempotent), ordinals >= 64
// simply repeat it on every launch.
struct PerDeviceOnce {
  std::atomic<uint64_t> bits{0};
  bool done(int dev) const { return dev >= 0 && dev < 64 && ((bits.load(std::memory_order_acquire) >> dev) & 1u); }
  void mark(int dev) { if (dev >= 0 && dev < 64) bits.fetch_or(uint64_t(1) << dev, std::memory_order_release); }
};

// internal launchers (prologue.cu)
int launch_unpack_qk(const rotattn_params& p, const uint8_t* X4, int8_t* X8, cudaStream_t st);
int launch_pad_ks(const rotattn_params& p, const float* Ks, float* KsP, int npad, cudaStream_t st);
int launch_unpack_vt(const rotattn_params& p, const uint8_t* V4, int8_t* V8T, int npad, cudaStream_t st);

}  // namespace rotattn
