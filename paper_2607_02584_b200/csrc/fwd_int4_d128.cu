// One translation unit per flavour of fwd_int4_kernel (fwd_int4_kernel.cuh) so that the variants compile in parallel.
#include "fwd_int4_kernel.cuh"

namespace rotattn {

int launch_fwd_int4_d128(const rotattn_params& p, const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv,
                         const FwdInt4Args& a, dim3 grid, cudaStream_t cs) {
  return launch_variants<128, false>(p, tq, tk, tv, a, grid, cs);
}

}  // namespace rotattn
