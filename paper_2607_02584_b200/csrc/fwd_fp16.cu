#include "tc_common.cuh"
using namespace rotattn;
extern "C" int rotattn_fwd_fp16(const rotattn_params* p, const void*, const void*, const void*, void*, const int32_t*, int32_t,
                                void*, size_t, void*) {
  (void)p; return ROTATTN_ERR_UNSUPPORTED;
}
