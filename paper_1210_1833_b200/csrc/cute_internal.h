// cute_internal.h -- structures shared by the grid build, the pair kernels and the host API.
// (Internal to the CUDA path; the oracle under oracle/ shares nothing with this.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/cute_b200.h"

namespace cute {

// ---- compile-time shape of the pair kernel -------------------------------------------------
constexpr int kLanes = 32;
constexpr int kIPerLane = 4;                      // R: i-points held in registers per lane
constexpr int kChunk = kLanes * kIPerLane;        // 128 i-points per work item
constexpr int kConsumerWarps = 8;
constexpr int kConsumerThreads = kConsumerWarps * 32;
constexpr int kThreads = kConsumerThreads + 32;   // + 1 producer warp
constexpr int kTile = 512;                        // j-points per shared-memory tile (8 KB of float4)
constexpr int kStages = 4;
constexpr int kJSplit = 64 * kTile;               // brute force: j-range per work item
constexpr float kSentinel = 1.0e18f;              // coordinate of a padding i-point (never in range)
constexpr unsigned kMagicBits = 0x4B400000u;      // bits of 1.5 * 2^23
#define CUTE_MAGIC_F 12582912.0f

struct Chunk {            // one work item's i side: <=128 consecutive cell-sorted points of one cell row
    uint32_t i_begin;
    uint32_t i_count;
    uint32_t row;         // cy + ncy * cz  (BOX3D), band (SPHERE), 0 (NONE)
    uint32_t cx01;        // first | last<<16 cell index along x of the chunk's points
};

struct GridView {         // device-side view of one built grid
    const float4 *hi;     // [n] cell-sorted (x,y,z,w)
    const float4 *lo;     // [n] low parts or nullptr
    const double *p64;    // SoA [4][n_pad] float64 canonical coordinates or nullptr
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
    double cell[3];
    double maxabs;            // largest |coordinate| (bound used for the float32 error model)
    int64_t ncells, nrows;
    const uint32_t *d_perm;
    double build_bytes;
};

namespace cute {

// ---- pair-kernel parameters ------------------------------------------------------------------
struct FastAxis {      // float32 bin map  t = g*S + O  (in bins), evaluated at t-tau and t+tau
    float S, Oa, Ob;   // Oa = O - tau, Ob = O + tau
    float c1, c2;      // ANGULAR: series correction coefficients (see pair_count.cu)
    int n;
};

struct PairParams {
    GridView g1, g2;
    int kind, is_auto, mode, periodic;
    int binmode;                 // 0: linear lo=0, 1: linear, 2: log
    int always_refine;           // 1: every pair passing the coarse test is recomputed in float64
    int n1, n2, n2eff, nhist;    // nhist = (n1+2)*n2eff (one guard row below and above)
    float q_lo, q_hi;            // coarse float32 range test on q (padded by half a bin)
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
    float rmax2;                 // pruning radius^2 (padded)
    float rmax;
    // work
    uint32_t *queue;             // [0] next item
    uint32_t *status;            // [0] error word
    unsigned long long *stats;   // [0] evaluated, [1] refined, [2] items, [3] flushes
    unsigned long long *partial; // [blocks][nhist]
    uint32_t item_begin, item_end, nsplit;
    uint32_t flush_items;
};

// host-side launchers (pair_count.cu / grid_build.cu)
cudaError_t launch_pair_kernel(const PairParams &p, int blocks, cudaStream_t s);
cudaError_t launch_reduce(const unsigned long long *partial, int blocks, int n1, int n2eff, unsigned long long *hist, cudaStream_t s);
int pair_kernel_smem_bytes(const PairParams &p);
int pair_kernel_max_blocks_per_sm(const PairParams &p);

struct BuildPlan {
    // inputs
    const void *c0, *c1, *c2;
    int64_t n;
    int coord, dtype, mode, periodic;
    double origin[3], inv_cell[3], size[3];
    int nc[3];
    double thetamax;
    int want_lo, want_f64;
    // workspace
    float4 *hi, *lo;
    double *p64;
    uint32_t n_pad;
    uint32_t *perm, *cid_sorted, *cell_id, *rank, *count, *cell_start, *scan_tmp, *row_nchunks, *row_chunk_start;
    Chunk *chunks;
    int *row_kx, *row_ylo, *row_yhi;
    uint32_t *status;  // [0] err, [1] nchunks
    double *bbox;      // [6] min xyz, max xyz, [6] maxabs
    int64_t ncells, nrows;
};
cudaError_t run_bbox(const BuildPlan &b, cudaStream_t s);
cudaError_t run_build(const BuildPlan &b, cudaStream_t s);

} // namespace cute
