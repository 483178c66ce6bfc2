// pair_kind_monopole.cu -- the CUTE_MONOPOLE instantiations of the pair kernel (pair_kernel.cuh).
#include "pair_kernel.cuh"

namespace cute {

cudaError_t launch_kind_monopole(const PairParams &p, int blocks, size_t smem, cudaStream_t s)
{
    const bool minimg = (p.mode == CUTE_GRID_NONE && p.L > 0.0);
    const bool lg = p.logbins != 0;
    if (minimg) return lg ? launch_t<CUTE_MONOPOLE, true, true>(p, blocks, smem, s) : launch_t<CUTE_MONOPOLE, true, false>(p, blocks, smem, s);
    return lg ? launch_t<CUTE_MONOPOLE, false, true>(p, blocks, smem, s) : launch_t<CUTE_MONOPOLE, false, false>(p, blocks, smem, s);
}

} // namespace cute
