// pair_kind_radial.cu -- the CUTE_RADIAL instantiations of the pair kernel (pair_kernel.cuh).
#include "pair_kernel.cuh"

namespace cute {

cudaError_t launch_kind_radial(const PairParams &p, int blocks, size_t smem, cudaStream_t s)
{
    return launch_t<CUTE_RADIAL, false, false>(p, blocks, smem, s);
}

} // namespace cute
