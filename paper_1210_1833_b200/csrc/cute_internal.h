// cute_internal.h -- structures shared by the grid build, the pair kernels and the host API.
// (Internal to the CUDA path; the oracle under oracle/ shares nothing with this.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/cute_b200.h"

namespace cute {

// ---- compile-time shape of the pair kernel -------------------------------------------------
constexpr int kIPerLane = 4;                      // R: i-points held in registers per lane
constexpr int kChunk = 32 * kIPerLane;            // 128 i-points per work item (one warp)
constexpr int kTile = 128;                        // j-points per shared-memory tile (2 KB of float4)
constexpr int kStages = 2;                        // double buffering
constexpr int kSegBatch = 32;                     // neighbour rows expanded per batch (one per lane)
constexpr int kSegSlots = 3 * kSegBatch;          // <= 3 contiguous j-segments per neighbour row
constexpr int kRefineCap = 64;                    // flagged blocks queued per warp for re-examination (pair_kernel.cuh)
#ifndef CUTE_MAX_WARPS
#define CUTE_MAX_WARPS 16                         // warps per CTA = per SM (registers: 65536 / (32 * warps) per thread)
#endif
constexpr int kPairCap = 96;                      // uncertain pairs queued per warp for float64 (settled 32 at a time)
constexpr int kMaxWarps = CUTE_MAX_WARPS;
constexpr float kSentinel = 1.0e18f;              // coordinate of a padding i-point (never in range)
constexpr uint32_t kEpochJ = 1u << 22;            // flush a warp's uint32 histogram after this many j

struct Chunk {            // one work item's i side: <=128 consecutive cell-sorted points of one cell row
    uint32_t i_begin;
    uint32_t i_count;
    uint32_t row;         // cy + ncy * cz  (BOX3D), band (SPHERE), 0 (NONE)
    uint32_t cx01;        // first | last<<16 cell index along x of the chunk's points
};

struct GridView {         // device-side view of one built grid
    const float4 *hi;     // [n] cell-sorted (x,y,z,w)
    const float4 *lo;     // [n] low parts or nullptr
    const double *p64;    // [n_pad][4] float64 canonical coordinates (one 32-byte record per point) or nullptr
    const uint32_t *cell_start; // [ncells+1]
    const Chunk *chunks;
    const int *row_kx;    // SPHERE: per-row half-width in cells along RA (or nullptr)
    const int *row_ylo, *row_yhi; // SPHERE: per-row range of neighbour rows
    uint32_t n, n_pad, nchunks;
    int ncx, ncy, ncz;
};

} // namespace cute

// The opaque handle of the C ABI (host memory only).
struct cute_grid {
    cute::GridView view;
    cute_grid_spec spec;      // resolved spec (explicit origin/size/ncell)
    int coord, dtype;
    int has_lo, has_f64;
    int weighted;             // hi.w holds uint32 weights
    uint32_t wmax;            // largest weight
    double cell[3];
    double maxabs;            // largest |coordinate| (bound used for the float32 error model)
    double bbox[6];           // min xyz, max xyz of the raw coordinates (zeros when not computed)
    int has_bbox;
    int64_t ncells, nrows;
    const uint32_t *d_perm;
    double build_bytes;
};

namespace cute {

// ---- pair-kernel parameters ------------------------------------------------------------------
// float32 bin map of one variable: t = S*g(q) + O in units of bins, where g = sqrt(q) (linear bins) or
// log2(q) (log bins) [angular: of q times a fitted cubic c1..c4].  The pair is binned by the fast path only
// if t is farther than tau from every integer; otherwise it is recomputed in float64.
struct FastAxis {
    float S, O, c1, c2, c3, c4;
    float tau, tau_w;      // tau_eff = tau + tau_w * w   (w: kind-specific, see pair_count.cu)
    int n;
};

struct PairParams {
    GridView g1, g2;
    int kind, is_auto, mode, periodic;
    int logbins;                 // variable 1: 0 linear, 1 log
    int angpoly;                 // ANGULAR linear bins: theta = sqrt(q) * poly(q)
    int always_refine;           // 1: every pair passing the coarse test is recomputed in float64
    int weighted;                // pairs count w_i * w_j (uint32 bit patterns in hi.w, or in lo.x when weight_in_lo)
    int weight_in_lo;            // xyz catalogues: hi.w holds |x|^2, the weight travels in lo.x
    int self_bin;                // weighted auto-correlation: bin of zero separation (or -1)
    uint32_t epoch_j;            // flush a warp's uint32 histogram after this many j-points
    int n1, n2, n2eff, nhist;    // nhist = n1 * n2eff
    int n2p, nhist_pad;          // shared-memory histogram with dump borders: n2p = n2 + 2 (1-D: 1), nhist_pad = (n1 + 2) * n2p
    int simple;                  // linear bins from 0 on every axis (and, r-mu, the |l|^-2 term folded): kernel variant PK_SIMPLE
    int colshift;                // histogram columns per warp copy = 1 << colshift (32, 8 or 1)
    int hist_shared;             // 1: one histogram copy per CTA (large 2-D histograms), flushed with atomicExch
    float q_hi;                  // coarse float32 range test on q (padded)
    float q_small;               // ANGULAR: pairs with q below this are always recomputed in float64 (theta < theta_min)
    float q_mid, tau_mid;        // ANGULAR log bins: a1.tau holds for chord^2 >= q_mid, tau_mid for q_small <= chord^2 < q_mid
    float tau_a, tau_b;          // ... and a pair's own bound is tau_a + tau_b / chord
    float dz_hi;                 // RADIAL: coarse test on |dz|
    FastAxis a1, a2;
    // float64 side (refine path): exact definition
    double lo1, hi1, lo2, hi2, L, aperture;
    const double *edges1, *edges2;   // device copies of cute_bin_edges()
    int closed_top2;
    // geometry
    float Lf;
    int kx, ky, kz;
    float ax, ay, az;            // cell sizes
    float ox, inv_ax;            // BOX3D: origin and 1/cell along x
    float rmax2;                 // row-pruning radius^2 (padded)
    float trim_pad;              // added to the x half-width of a trimmed row: float32 rounding of the trim itself
    int ring;                    // SPHERE: RA axis covers 360 deg (neighbour window wraps)
    // work
    uint32_t *queue;             // [0] next item
    uint32_t *status;            // [0] error word
    unsigned long long *stats;   // [0] evaluated, [1] refined, [2] items, [3] flushes
    unsigned long long *hist;    // [nhist] global result
    uint32_t item_begin, item_end, nsplit, jsplit;
    uint32_t flush_items;
    int warps;                   // warps per CTA
    uint32_t smem_per_warp;      // bytes
};

// number of kernels this library has launched (reported by cute_launch_count)
void note_launches(int n);

// host-side launchers (pair_count.cu / pair_kind_*.cu / grid_build.cu)
cudaError_t launch_pair_kernel(const PairParams &p, int blocks, cudaStream_t s);
cudaError_t launch_kind_monopole(const PairParams &p, int blocks, size_t smem, cudaStream_t s);
cudaError_t launch_kind_angular(const PairParams &p, int blocks, size_t smem, cudaStream_t s);
cudaError_t launch_kind_rmu(const PairParams &p, int blocks, size_t smem, cudaStream_t s);
cudaError_t launch_kind_radial(const PairParams &p, int blocks, size_t smem, cudaStream_t s);
cudaError_t launch_kind_pisigma(const PairParams &p, int blocks, size_t smem, cudaStream_t s);
// fills colshift, warps, smem_per_warp; returns total dynamic shared memory or -1 if it cannot fit
int plan_pair_kernel(PairParams &p, int want_warps, int want_cols);

struct BuildPlan {
    // inputs
    const void *c0, *c1, *c2;
    const uint32_t *weight;       // optional (RADEC only): goes into hi.w as a bit pattern, p64[3] as a double
    int64_t n;
    int coord, dtype, mode, periodic;
    int order_only;    // mode NONE: the cells only ORDER the points (spatially coherent warps); one row, all pairs
    double origin[3], inv_cell[3], size[3];
    int nc[3];
    double thetamax;
    int want_lo, want_f64;
    // workspace
    float4 *hi, *lo;
    double *p64;
    uint32_t n_pad;
    uint32_t *perm, *count, *cell_start, *scan_tmp, *row_nchunks, *row_chunk_start;
    Chunk *chunks;
    int *row_kx, *row_ylo, *row_yhi;
    uint32_t *status;  // [0] err, [1] nchunks, [2] largest weight
    double *bbox;      // [6] min xyz, max xyz
    int64_t ncells, nrows;
    // two-level partition of large catalogues (grid_build.cu): records grouped by bucket, per-(bucket, CTA) counts
    void *part_tmp;
    uint32_t *part_table;
    int part_G, part_B, part_cpb;   // CTAs of the coarse pass, buckets, fine cells per bucket (0: one-pass build)
    int part_shift;                 // log2(part_cpb)
};

// large catalogues are built by a coarse partition into buckets of consecutive cells + one CTA per bucket
constexpr int64_t kPartMinN = 1 << 20;
constexpr int kPartMaxBuckets = 1024, kPartMaxCellsPerBucket = 16384;
inline void part_shape(int64_t ncells, int *B, int *cpb)
{
    int64_t c = 1;   // a power of two: bucket = cell >> log2(cpb)
    while (c * kPartMaxBuckets < ncells && c < kPartMaxCellsPerBucket) c *= 2;
    *cpb = (int)c;
    *B = (int)((ncells + c - 1) / c);
}
cudaError_t run_bbox(const BuildPlan &b, cudaStream_t s);       // leaves 6 order-preserving int64 images in b.bbox
void decode_bbox(const long long raw[6], double out[6]);
cudaError_t run_build(const BuildPlan &b, cudaStream_t s);
cudaError_t run_pixelize(const BuildPlan &b, uint32_t *count, uint32_t *pos, uint32_t *scan_tmp, double *pra, double *pdec,
                         uint32_t *pw, cudaStream_t s);   // b: SPHERE geometry; pos[ncells] = number of non-empty pixels

} // namespace cute
