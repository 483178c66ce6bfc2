// pair_kind_angular.cu -- the CUTE_ANGULAR instantiations of the pair kernel (pair_kernel.cuh).
#include "pair_kernel.cuh"

namespace cute {

cudaError_t launch_kind_angular(const PairParams &p, int blocks, size_t smem, cudaStream_t s)
{
    return p.logbins ? launch_t<CUTE_ANGULAR, false, true>(p, blocks, smem, s) : launch_t<CUTE_ANGULAR, false, false>(p, blocks, smem, s);
}

} // namespace cute
