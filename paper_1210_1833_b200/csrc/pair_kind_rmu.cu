// pair_kind_rmu.cu -- the CUTE_RMU instantiations of the pair kernel (pair_kernel.cuh).
#include "pair_kernel.cuh"

namespace cute {

cudaError_t launch_kind_rmu(const PairParams &p, int blocks, size_t smem, cudaStream_t s)
{
    return launch_t<CUTE_RMU, false, false>(p, blocks, smem, s);
}

} // namespace cute
