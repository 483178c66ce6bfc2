// pair_count.cu -- host side of the pair kernel (pair_kernel.cuh): shared-memory planning and dispatch to the
// per-kind instantiations (pair_kind_*.cu, compiled in parallel).
#include "cute_internal.h"

namespace cute {

static constexpr int kSmemBudget = 227 * 1024;
constexpr uint32_t kTileBytesHost = kTile * 16;

static inline uint32_t hist_bytes(int nhist_pad, int colshift)
{
    return ((((uint32_t)nhist_pad << colshift) * 4 + 15) & ~15u);
}

static inline uint32_t warp_smem_bytes(bool needlo, int nhist_pad, int colshift, bool shared_hist)
{
    uint32_t b = kStages * kTileBytesHost * (needlo ? 2 : 1) + kSegSlots * 16 + kRefineCap * 16 + kPairCap * 16 + 32;
    if (!shared_hist) b += hist_bytes(nhist_pad, colshift);
    return (b + 127) & ~127u;
}

int plan_pair_kernel(PairParams &p, int want_warps, int want_cols)
{
    // Warps hide the latency of the dependent MUFU/FFMA chains and ncu shows throughput growing with the warp
    // count up to 16.  Default = 8 private histogram columns per warp, as many warps as fit.  A histogram too
    // large for 16 warps with private copies (the 2-D kinds) becomes ONE copy per CTA shared by all its warps.
    const bool needlo = (p.kind == CUTE_RMU || p.kind == CUTE_PISIGMA || (p.weighted && p.kind != CUTE_ANGULAR));
    p.hist_shared = 0;
    const int clist[] = {3, 0, 5};
    for (int ci = 0; ci < 3; ci++) {
        if (want_cols > 0 && (1 << clist[ci]) != want_cols) continue;
        const uint32_t per = warp_smem_bytes(needlo, p.nhist_pad, clist[ci], false);
        int w = (int)((size_t)kSmemBudget / per);
        if (w > kMaxWarps) w = kMaxWarps;
        if (want_warps > 0) { if (want_warps > w) continue; w = want_warps; }
        else if (want_cols <= 0 && w < kMaxWarps && clist[ci] != 5) continue;   // would cost warps: share instead
        else if (want_cols <= 0 && clist[ci] == 5) continue;
        if (w < 1) continue;
        p.colshift = clist[ci]; p.warps = w; p.smem_per_warp = per;
        return (int)(per * (uint32_t)w);
    }
    if (want_cols > 0) return -1;
    {   // shared copy, one column
        const uint32_t per = warp_smem_bytes(needlo, p.nhist_pad, 0, true), hb = hist_bytes(p.nhist_pad, 0);
        if ((size_t)hb + per > (size_t)kSmemBudget) return -1;
        int w = (int)(((size_t)kSmemBudget - hb) / per);
        if (w > kMaxWarps) w = kMaxWarps;
        if (want_warps > 0) { if (want_warps > w) return -1; w = want_warps; }
        p.hist_shared = 1; p.colshift = 0; p.warps = w; p.smem_per_warp = per;
        return (int)(per * (uint32_t)w + hb);
    }
}

cudaError_t launch_pair_kernel(const PairParams &p, int blocks, cudaStream_t s)
{
    const size_t smem = (size_t)p.smem_per_warp * p.warps + (p.hist_shared ? hist_bytes(p.nhist_pad, 0) : 0);
    switch (p.kind) {
    case CUTE_MONOPOLE: return launch_kind_monopole(p, blocks, smem, s);
    case CUTE_ANGULAR: return launch_kind_angular(p, blocks, smem, s);
    case CUTE_RMU: return launch_kind_rmu(p, blocks, smem, s);
    case CUTE_RADIAL: return launch_kind_radial(p, blocks, smem, s);
    case CUTE_PISIGMA: return launch_kind_pisigma(p, blocks, smem, s);
    }
    return cudaErrorInvalidValue;
}

} // namespace cute
