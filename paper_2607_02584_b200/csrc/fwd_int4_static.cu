// rotattn_fwd_int4_static: the INT4 attention forward for callers that have no device memory to give and may not ask
// the CUDA runtime for any.
//
// Who that is.  A video-DiT serving process usually hands the whole of HBM to its own arena at start-up (weights plus
// an activation plan worked out once) and forbids cudaMalloc afterwards: an allocation in the middle of a denoising
// step synchronises the whole device and stalls every other stream, and it can simply fail because the arena already
// owns the memory.  The same holds for an operator plugged into somebody else's runtime through a fixed signature
// "inputs in, outputs out": there is no slot for a workspace pointer and no allocator the plug-in is allowed to touch.
// rotattn_fwd_int4 cannot serve those callers, because it needs a workspace (rotattn_workspace_bytes(p, 1)) for the
// one-byte-per-code operand copies that the tensor cores read.
//
// What this file does about it.  The workspace lives in g_static_ws below, a file-scope device array of
// ROTATTN_STATIC_WS_BYTES that is part of the library image: the driver places it on every GPU that loads this module
// and keeps it there until the process exits.  The entry point passes that array to the unchanged rotattn_fwd_int4
// with ws_state = 0, so the operand copies are rebuilt from the caller's packed buffers on every call and the
// attention kernel itself is the one every other test covers.  No cudaMalloc, cudaFree, cudaMallocAsync or library
// routine that allocates is called here or below (tensor maps are encoded on the host stack, kernels are launched,
// function attributes are set - nothing else).
//
// The array's name in HOST code is only a handle of the host-side shadow of the symbol, not a device address: handing
// `g_static_ws` itself to a kernel would make it fault (or, where the GPU can reach host memory, scribble over the
// wrong place).  The device address comes from cudaGetSymbolAddress, asked once per device with that device current;
// see static_ws_address().
#include <mutex>
#include <cstdio>
#include "common.cuh"

namespace {

static __device__ __align__(256) unsigned char g_static_ws[ROTATTN_STATIC_WS_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_addr_mutex;
void* g_addr[kMaxDevices] = {};          // device address of g_static_ws on device i, nullptr = not asked yet

// Device address of the built-in workspace on the CURRENT device.  The first call on a device asks the runtime
// (which also makes it load this module there - the one-time set-up that must not happen under stream capture).
int static_ws_address(void** out) {
  int dev = -1;
  ROTATTN_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) {
    rotattn::set_error_text("rotattn_fwd_int4_static: device ordinal beyond the 64 this table holds");
    return ROTATTN_ERR_UNSUPPORTED;
  }
  std::lock_guard<std::mutex> lock(g_addr_mutex);
  if (!g_addr[dev]) {
    void* ptr = nullptr;
    ROTATTN_CUDA_TRY(cudaGetSymbolAddress(&ptr, g_static_ws));
    if (!ptr) {
      rotattn::set_error_text("rotattn_fwd_int4_static: cudaGetSymbolAddress returned a null address");
      return ROTATTN_ERR_CUDA;
    }
    g_addr[dev] = ptr;
  }
  *out = g_addr[dev];
  return ROTATTN_OK;
}

}  // namespace

extern "C" int rotattn_fwd_int4_static(const rotattn_params* p, const uint8_t* Q4, const float* Qs, const uint8_t* K4,
                                       const float* Ks, const uint8_t* V4, const float* Vs, void* O,
                                       const int32_t* head_sel, int32_t n_sel, void* stream) {
  int st = rotattn_validate(p);
  if (st != ROTATTN_OK) return st;
  if (p->smooth) {      // the smoothing state is written by the prologue into ITS workspace; there is none here
    rotattn::set_error_text("rotattn_fwd_int4_static: smooth = 1 needs the prologue's workspace, use rotattn_fwd_int4");
    return ROTATTN_ERR_UNSUPPORTED;
  }
  const size_t need = rotattn_workspace_bytes(p, 1);
  if (need > (size_t)ROTATTN_STATIC_WS_BYTES) {
    char msg[200];
    snprintf(msg, sizeof(msg), "rotattn_fwd_int4_static: this shape needs %zu bytes of workspace, the built-in one holds %zu",
             need, (size_t)ROTATTN_STATIC_WS_BYTES);
    rotattn::set_error_text(msg);
    return ROTATTN_ERR_WORKSPACE_TOO_SMALL;
  }
  if ((st = rotattn::check_device_sm100()) != ROTATTN_OK) return st;
  void* ws = nullptr;
  if ((st = static_ws_address(&ws)) != ROTATTN_OK) return st;
  // ws_state = 0: the unpack kernels rewrite every byte the attention kernel will read for this shape (operand bytes
  // of all B*H heads, the zero padding of V^T up to a whole key block, the padded key scales), so whatever an earlier
  // call with another shape left in the array is never seen and nothing needs clearing first.
  return rotattn_fwd_int4(p, Q4, Qs, K4, Ks, V4, Vs, O, head_sel, n_sel, ws, (size_t)ROTATTN_STATIC_WS_BYTES, 0, stream);
}
