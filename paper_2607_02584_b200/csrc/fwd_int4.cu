#include "tc_common.cuh"
using namespace rotattn;
extern "C" int rotattn_fwd_int4(const rotattn_params* p, const uint8_t*, const float*, const uint8_t*, const float*,
                                const uint8_t*, const float*, void*, const int32_t*, int32_t, void*, size_t, int32_t, void*) {
  (void)p; return ROTATTN_ERR_UNSUPPORTED;
}
extern "C" int rotattn_fwd_int4_debug(const rotattn_params* p, const uint8_t*, const float*, const uint8_t*, const float*,
                                      const uint8_t*, const float*, int32_t, int32_t, int32_t*, uint8_t*, void*, void*, size_t,
                                      int32_t, void*) {
  (void)p; return ROTATTN_ERR_UNSUPPORTED;
}
