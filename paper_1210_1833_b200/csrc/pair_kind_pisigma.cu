// pair_kind_pisigma.cu -- the CUTE_PISIGMA instantiations of the pair kernel (pair_kernel.cuh).
#include "pair_kernel.cuh"

namespace cute {

cudaError_t launch_kind_pisigma(const PairParams &p, int blocks, size_t smem, cudaStream_t s)
{
    return launch_t<CUTE_PISIGMA, false, false>(p, blocks, smem, s);
}

} // namespace cute
