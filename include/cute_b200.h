/*
 * cute_b200.h -- C ABI of the B200-native pair-counting hot path of CUTE (arXiv 1210.1833).
 *
 * Problem statement (sec. III.A): "DD, DR and RR are computed by autocorrelating
 * or crosscorrelating each pair of catalogs ... calculating the distance between each pair of
 * objects, determining the bin corresponding to that distance and increasing the histogram count
 * on that bin", i.e. Eq. 11; with neighbour searching by cubical cells or pixels
 * (sec. III.C) and the estimators of Eqs. 13-15 on the host.
 *
 * Conventions (readings of the paper are listed in DESIGN.md):
 *  - Every function returns an int status: 0 = CUTE_OK, < 0 error, > 0 warning.  No exceptions,
 *    no abort, no stdout.  cute_strerror() gives a static string.
 *  - "device" pointers are CUDA device pointers owned by the caller (PyTorch tensors in this
 *    repository); the library never allocates or frees device memory.  "host" pointers are plain
 *    host memory.  Streams are passed as void* (a cudaStream_t; NULL = legacy default stream).
 *  - Auto-correlation (second grid NULL or equal to the first) counts UNORDERED pairs i<j;
 *    cross-correlation counts all N1*N2 pairs (forced by Eq. 15).
 *  - Bin k holds pairs with e_k <= v < e_{k+1}; out-of-range pairs are dropped.  2-D histograms
 *    are stored first-variable-major: index = k1 * n2 + k2.
 *  - Histograms are uint64 ("long integers").
 *  - The GPU histogram equals the float64 definition exactly except for pairs whose binned variable
 *    lies at float64-rounding distance of a bin edge.
 */
#ifndef CUTE_B200_H
#define CUTE_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CUTE_ABI_VERSION 1

/* status codes */
#define CUTE_OK 0
#define CUTE_ERR_INVALID_ARG (-1)
#define CUTE_ERR_UNSUPPORTED (-2)
#define CUTE_ERR_WORKSPACE_TOO_SMALL (-3)
#define CUTE_ERR_CUDA (-4)
#define CUTE_ERR_OVERFLOW (-5)
#define CUTE_ERR_POINT_OUT_OF_BOX (-6)
#define CUTE_ERR_GRID_MISMATCH (-7)
#define CUTE_ERR_STATIC_SCRATCH_LIMIT (-8) /* cute_count_pairs_static: the binning needs more than CUTE_STATIC_SCRATCH_BYTES */
#define CUTE_WARN_EMPTY_BIN 1

/* kinds of correlation function ("CUTE calculates 4 different correlation functions (3-D,
 * monopole, angular and radial)") */
#define CUTE_ANGULAR 0  /* w(theta): v = theta [rad]                     */
#define CUTE_MONOPOLE 1 /* xi_0(r): v = r; periodic box: PAPER.md:245-249       */
#define CUTE_RMU 2      /* xi(r,mu): v = (r, mu), mid-point line of sight */
#define CUTE_RADIAL 3   /* xi_r(zbar,dz): pairs with theta < aperture, v = (zbar, dz) */
#define CUTE_PISIGMA 4  /* xi(pi,sigma): v = (pi, sigma), pi = r mu, sigma = sqrt(r^2 - pi^2), Eq. 2 */

/* catalogue coordinates */
#define CUTE_COORD_XYZ 0     /* c0,c1,c2 = x,y,z (Mpc/h)              -> MONOPOLE, RMU, PISIGMA */
#define CUTE_COORD_RADEC 1   /* c0,c1 = RA,Dec in degrees; c2 ignored -> ANGULAR       */
#define CUTE_COORD_RADECZ 2  /* c0,c1 = RA,Dec in degrees; c2 = z     -> RADIAL (and ANGULAR) */
#define CUTE_F32 0
#define CUTE_F64 1

/* neighbour-search modes */
#define CUTE_GRID_NONE 0   /* no cells: brute force, every pair is evaluated       */
#define CUTE_GRID_BOX3D 1  /* cubical cells                                        */
#define CUTE_GRID_SPHERE 2 /* pixels with constant limits in (sin dec, RA)     */

/* A catalogue in structure-of-arrays form (as in the paper's listing).
 * Pointers are DEVICE pointers for cute_make_grid and HOST pointers for cute_count_pairs_host.
 * z -> comoving distance is the caller's job (float64 on the host). */
typedef struct cute_catalog {
    size_t struct_size; /* = sizeof(cute_catalog) */
    int64_t n;          /* number of objects, >= 0 */
    int coord;          /* CUTE_COORD_*            */
    int dtype;          /* CUTE_F32 | CUTE_F64     */
    const void *c0, *c1, *c2;
    const uint32_t *weight; /* optional integer weights, 1 <= w <= 65535 (objects per pixel of a pixel map,        */
                            /* PAPER.md:233; or any integer weight per object); NULL = unweighted.  RA/Dec and xyz */
                            /* catalogues (ANGULAR, MONOPOLE, RMU, PISIGMA; not RADIAL).  A pair counts w_i w_j;   */
                            /* in an auto-correlation the w_i objects of one point count as w_i (w_i - 1)/2 pairs  */
                            /* at zero separation (exactly as w_i repeated objects would).                         */
} cute_catalog;

/* How to build the cell list.
 *  BOX3D : origin[3], size[3] in Mpc/h (size[d] <= 0: bounding box of the catalogue, computed on the
 *          device; for a cross-correlation pass the same explicit box to both grids), ncell[3]
 *          (ncell[d] <= 0: chosen by the library from rmax), periodic != 0 => origin must be 0 and
 *          size[0]=size[1]=size[2]=L.
 *  SPHERE: axis 0 = RA: origin[0] = RA0 [deg], size[0] = span [deg] (< 360: RA is taken modulo 360
 *          relative to RA0, so a footprint straddling RA=0 is fine); axis 1 = sin(Dec): origin[1],
 *          size[1] (dimensionless, within [-1,1]); ncell[0], ncell[1]; axis 2 unused.
 *  rmax  : largest separation that will be asked for with this grid: r [Mpc/h] for BOX3D,
 *          theta [rad] for SPHERE (the radial aperture or the last theta edge).
 *  Two grids used together in a cross-correlation must carry identical specs. */
typedef struct cute_grid_spec {
    size_t struct_size;
    int mode;      /* CUTE_GRID_* */
    int periodic;  /* BOX3D only  */
    double origin[3];
    double size[3];
    int ncell[3];
    double rmax;
    int kind_mask; /* bit k set: the grid will be used for kind k (CUTE_ANGULAR=0 ...); 0 = any kind the   */
                   /* coordinates allow.  Lets the build skip arrays a kind does not read (the low parts). */
    int no_perm;   /* != 0: do not write the sorted-slot -> input-index permutation (cute_grid_info.d_perm = NULL); */
                   /* pair counting never reads it, and it is a random 4-byte store per object                     */
    int build_path; /* 0: chosen by size (catalogues of >= 2^20 objects are built by a two-level partition: coarse   */
                   /* buckets of consecutive cells, then one CTA per bucket in shared memory); 1: one-pass counting */
                   /* sort; 2: partition.  Same result up to the (arbitrary) order inside a cell.                  */
} cute_grid_spec;

/* Binning.  Variable 1: theta [rad] (ANGULAR), r (MONOPOLE, RMU), zbar (RADIAL), pi (PISIGMA); linear or, if
 * log1 != 0, logarithmic: e_k = lo1 (hi1/lo1)^(k/n1) ("logarithmic binning").
 * Variable 2 (n2 = 0 for 1-D kinds): mu in [lo2,hi2] (RMU; mu = 1 belongs to the last bin when
 * hi2 >= 1), dz (RADIAL), sigma (PISIGMA; a grid must then have rmax >= sqrt(hi1^2 + hi2^2)); always linear.  aperture_rad: RADIAL only, strict theta < aperture.
 * box_L > 0: periodic box of side L, minimum-image separations (MONOPOLE only; needs hi1 <= L/2).  Brute force
 * (grid mode NONE) then needs the catalogues to span at most L per axis (coordinates wrapped into one box side;
 * else CUTE_ERR_POINT_OUT_OF_BOX); a periodic BOX3D grid needs them inside [0, L). */
typedef struct cute_bin_spec {
    size_t struct_size;
    int n1; double lo1, hi1; int log1;
    int n2; double lo2, hi2;
    double aperture_rad;
    double box_L;
} cute_bin_spec;

/* Optional launch controls (NULL = defaults).  All fields 0 = default. */
typedef struct cute_count_opts {
    size_t struct_size;
    int blocks;            /* persistent CTAs to launch (default: one per SM)                        */
    int64_t item_begin;    /* shard of the work-item list [item_begin, item_end) handled by this call */
    int64_t item_end;      /* (0,0 with shard == 0 = all). Items partition the pairs, so shards add up exactly */
    double tau_scale;      /* multiplies the refine half-width (>1 refines more pairs; results must   */
                           /* not change).  0 = 1.0                                                   */
    int force_refine;      /* != 0: every in-range pair is recomputed in float64                      */
    int flush_items;       /* flush the shared-memory histogram every this many work items (testing   */
                           /* the uint32 epoch logic); 0 = only when the epoch bound requires it      */
    int warps;             /* warps per CTA (1,2,4,6,8,12,16); 0 = chosen by the library              */
    int hist_cols;         /* private histogram columns per warp: 32 (one per lane), 8 or 1; 0 = auto */
    int shard;             /* != 0: [item_begin, item_end) is honoured even when it is empty (a rank whose   */
                           /* share of the items is [0,0) counts nothing instead of everything)               */
} cute_count_opts;

/* Facts about a built grid (for tests and reports). */
typedef struct cute_grid_info {
    size_t struct_size;
    int64_t n;
    int mode, periodic, kind_coord, dtype, has_lo, has_f64;
    int ncell[3];
    double origin[3], cell[3];
    double size[3];           /* resolved box: pass origin, size, ncell to the second grid of a cross-correlation */
    int64_t ncells, nrows, nchunks;
    const void *d_hi;         /* float4[n]   cell-sorted (x,y,z,w)                */
    const void *d_lo;         /* float4[n]   low parts (or NULL)                  */
    const void *d_perm;       /* uint32[n]   sorted slot -> original index        */
    const void *d_cell_start; /* uint32[ncells+1]                                 */
    double build_bytes;       /* algorithmic HBM bytes of the build   */
} cute_grid_info;

typedef struct cute_grid cute_grid; /* opaque host handle; holds pointers INTO the caller's workspace */

int cute_version(void);
const char *cute_strerror(int status);
/* Number of CUDA kernels this library has launched in this process so far (for reports). */
uint64_t cute_launch_count(void);

/* Bounding box of the raw coordinates ("a box encompassing the whole catalog is first
 * determined"): bounds[0..2] = minima of c0,c1,c2, bounds[3..5] = maxima (HOST, out).  cat pointers are
 * DEVICE pointers; d_tmp is a DEVICE buffer of >= 64 bytes.  Synchronises the stream.  Used to give the
 * two grids of a cross-correlation one common explicit box. */
int cute_catalog_bounds(const cute_catalog *cat, void *d_tmp, void *stream, double bounds[6]);

/* Pixel map of an angular catalogue ("create a pixel map from the catalog and then correlate the
 * pixels (weighting each of them by the number of objects that fall inside it)"): n_ra x n_u pixels with constant
 * limits in RA [ra0, ra0 + dra) (degrees, modulo 360 relative to ra0) and sin(Dec) [u0, u0 + du).
 * cat: DEVICE, CUTE_COORD_RADEC(Z), unweighted.  Outputs (DEVICE, room for min(n, n_ra*n_u) entries each): centre RA
 * and Dec [deg, float64] and object count of every NON-EMPTY pixel, in pixel order (sin(Dec)-major); *npix (HOST) =
 * their number.  The result is a weighted CUTE_COORD_RADEC catalogue for cute_make_grid.  d_workspace: DEVICE,
 * cute_pixelize_workspace_bytes(n_ra, n_u).  Synchronises the stream. */
int cute_pixelize_workspace_bytes(int n_ra, int n_u, size_t *bytes);
int cute_pixelize(const cute_catalog *cat, double ra0, double dra, double u0, double du, int n_ra, int n_u,
                  double *d_pix_ra, double *d_pix_dec, uint32_t *d_pix_weight, int64_t *npix,
                  void *d_workspace, size_t bytes, void *stream);

/* Size of the device workspace cute_make_grid needs for this catalogue and spec (256-byte granular). */
int cute_grid_workspace_bytes(const cute_catalog *cat, const cute_grid_spec *spec, size_t *bytes);

/* Cell-list build ("To each cell we associate the positions of all the objects that
 * fall inside it"): canonicalise (unit vectors, hi/lo split), cell index + cell histogram, exclusive
 * scan, scatter into cell-sorted float4 arrays, chunk table.  Runs on `stream`; synchronises the
 * stream once to read back the error word and the chunk count.  cat pointers are DEVICE pointers and
 * are not referenced after the call returns.  *out must be released with cute_free_grid, which
 * never frees device memory.  mode NONE gives a single-cell grid (brute force). */
int cute_make_grid(const cute_catalog *cat, const cute_grid_spec *spec, void *d_workspace, size_t bytes,
                   void *stream, cute_grid **out);
void cute_free_grid(cute_grid *g);
int cute_grid_get_info(const cute_grid *g, cute_grid_info *info);

/* Scratch the pair counter needs (work-queue counter, status word, statistics, bin edges). */
int cute_count_scratch_bytes(const cute_bin_spec *bins, const cute_count_opts *opts, size_t *bytes);

/* The pair count (CUDA prior art PAPER.md:159-192).  d_hist: DEVICE uint64[n1*max(n2,1)],
 * overwritten.  g2 == NULL or g2 == g1: auto-correlation.  Enqueued on `stream`; returns after
 * enqueue.  Deferred device errors are read with cute_count_status. */
int cute_count_pairs(int kind, const cute_grid *g1, const cute_grid *g2, const cute_bin_spec *bins,
                     uint64_t *d_hist, void *d_scratch, size_t scratch_bytes,
                     const cute_count_opts *opts, void *stream);

/* Number of work items cute_count_pairs enumerates for these arguments (they partition the pairs: shards
 * [item_begin, item_end) given through cute_count_opts add up exactly to the full histogram). */
int cute_count_items(int kind, const cute_grid *g1, const cute_grid *g2, const cute_bin_spec *bins,
                     const cute_count_opts *opts, int64_t *nitems);

/* Sharding of a pair count over `world` ranks: [*begin, *end) of the nitems work items that rank
 * `rank` handles (pass them as cute_count_opts.item_begin / item_end with shard = 1).  Items are chunk-major (item =
 * chunk * nsplit + split, nchunks from cute_grid_info).  Cross-correlations and cell-list counts have ~uniform work per
 * item; a brute-force AUTO-correlation (auto_brute != 0) is a triangle -- chunk c meets only j > i -- so its cuts are
 * placed at equal areas, 1 - (1 - x)^2.  The shards partition [0, nitems): integer partial histograms add up exactly --
 * PROVIDED every shard is counted on the SAME built grid or a byte copy of its workspace.  The order of the points inside
 * a cell is decided by atomic cursors and differs from one cute_make_grid call to the next, so item k of two separate
 * builds of one catalogue does not hold the same 128 points: ranks that each built their own grid must first overwrite
 * their workspace with one rank's (a broadcast; layout and host handle are identical, they do not depend on that order). */
int cute_shard_items(int64_t nitems, int64_t nchunks, int rank, int world, int auto_brute, int64_t *begin, int64_t *end);

/* Grid sizing from the data ("a box encompassing the whole catalog is first determined", PAPER.md:208-215
 * for pixels): fills *spec for `kind` with mode BOX3D or SPHERE so that ONE spec serves all the ncat catalogues (DEVICE
 * pointers) of a correlation function -- their common bounding box, padded; BOX3D: box_L > 0 gives the periodic box
 * [0,L)^3, ncell is left to cute_make_grid unless given; SPHERE: pixels of side pix_frac * rmax [rad] with constant
 * limits in RA and sin(Dec), the full ring when the footprint is wider than 180 degrees in RA (or straddles RA = 0).
 * rmax: largest separation (r, or theta in rad).  d_tmp: DEVICE >= 64 bytes.  Synchronises the stream. */
int cute_auto_grid_spec(int kind, int mode, const cute_catalog *const *cats, int ncat, double rmax, double box_L,
                        double pix_frac, const int ncell[3], int no_perm, void *d_tmp, void *stream, cute_grid_spec *spec);

/* Synchronises `stream` and returns the deferred status of the last cute_count_pairs that used
 * d_scratch.  stats (host, may be NULL): [0] separations evaluated, [1] pairs recomputed in float64,
 * [2] work items, [3] shared-memory histogram flushes. */
int cute_count_status(void *d_scratch, void *stream, uint64_t stats[4]);

/* The pair count for callers that cannot allocate device memory -- cute_count_pairs without the d_scratch argument.
 *
 * cute_count_pairs leaves every allocation to its caller, down to the small scratch block (work counter, status word,
 * statistics, bin edges) of cute_count_scratch_bytes.  Not every caller can come up with one: an analysis hook that
 * runs inside a simulation whose memory manager claimed the whole device at start-up and passes it only the particle
 * data and a histogram to fill, a plug-in held to a host application's fixed memory budget, a thread for which
 * cudaMalloc is off limits because it would stall the device under a time-critical loop or because another thread of
 * the process is recording a stream at that moment.  For them the scratch is a fixed array of
 * CUTE_STATIC_SCRATCH_BYTES inside the library image: each GPU that loads the library gives up that much memory until
 * the process ends, and this function, like the rest of the library, calls neither cudaMalloc nor cudaFree nor any
 * routine that allocates device memory.
 *
 * Arguments and result are those of cute_count_pairs (the caller still owns the grids and d_hist, DEVICE
 * uint64[n1*max(n2,1)], overwritten), with these differences:
 *  - Limit: the bin edges must fit the array: 8 * (n1 + n2 + 2) + 64 bytes, rounded up to 256, may not exceed
 *    CUTE_STATIC_SCRATCH_BYTES (n1 + n2 <= 8182 bins).  Finer binning is refused with
 *    CUTE_ERR_STATIC_SCRATCH_LIMIT before anything is enqueued; use cute_count_pairs with your own scratch instead.
 *  - It finishes the job: after enqueuing on `stream` it waits for the stream and returns the final status, deferred
 *    device errors included (what cute_count_status would report); stats (HOST, may be NULL) as in cute_count_status.
 *  - First call on a device: looks up the array's device address (no allocation; the current device must be the one
 *    the grids live on).  Make that first call outside any stream capture.
 *  - Sharing: all calls on one device use the same array, which still holds the previous call's contents; the words
 *    that must start at zero are cleared on `stream` at the start of every call.  Counts that overlapped on the GPU
 *    would corrupt each other (one work counter, one set of edges), so calls from several host threads of one process
 *    are made to take turns per device (a lock held until the call's work is done).  Up to 64 devices. */
#define CUTE_STATIC_SCRATCH_BYTES 65536
int cute_count_pairs_static(int kind, const cute_grid *g1, const cute_grid *g2, const cute_bin_spec *bins,
                            uint64_t *d_hist, const cute_count_opts *opts, void *stream, uint64_t stats[4]);

/* End-to-end entry point with HOST buffers: copies the catalogue(s) to the device, builds the
 * grid(s), counts, copies the histogram back.  cat2 == NULL: auto.  d_workspace: DEVICE, at least
 * cute_host_workspace_bytes().  opts may be NULL.  Synchronous. */
int cute_host_workspace_bytes(const cute_catalog *cat1, const cute_catalog *cat2, const cute_grid_spec *spec,
                              const cute_bin_spec *bins, size_t *bytes);
int cute_count_pairs_host(int kind, const cute_catalog *cat1, const cute_catalog *cat2, const cute_grid_spec *spec,
                          const cute_bin_spec *bins, const cute_count_opts *opts, uint64_t *h_hist, void *d_workspace,
                          size_t bytes, void *stream);

/* Density-grid monopole of a periodic box (the second algorithm of CUTE_box): "the particle content of
 * the catalog is first interpolated to a grid and the overdensity field delta is estimated at every grid point using a TSC
 * algorithm.  Then pairs of grid points are correlated, and a weight delta_i delta_j is given to each pair", xi(r) =
 * <delta(x) delta(x + r)> (Eq. 17); the relative offsets and their bins are found once.  Readings (N4): grid
 * points = centres (g + 1/2) L/ng of the ng^3 cells; TSC = second-order B-spline per axis; delta = rho ng^3 / N - 1; every
 * ordered pair of distinct grid points with the minimum image, r = (L/ng) |v|, half-open bins (variable 1 of `bins`,
 * linear or log, hi1 <= L/2; the other fields are ignored).  cat: DEVICE, CUTE_COORD_XYZ in [0, L) (taken modulo L),
 * float32 or float64, unweighted.  Outputs (HOST, n1 entries; h_sum_dd and h_npairs may be NULL): xi, the sums of
 * delta delta and the numbers of grid-point pairs per bin; d_delta (DEVICE, ng^3 doubles, index (gz ng + gy) ng + gx, may
 * be NULL) receives the overdensity field.  Float64 throughout: equal to a serial float64 evaluation up to the order of
 * the additions.  A bin no offset falls in gets xi = 0 and CUTE_WARN_EMPTY_BIN.  Synchronises the stream. */
int cute_density_grid_workspace_bytes(int ng, const cute_bin_spec *bins, double L, size_t *bytes);
int cute_density_grid_xi(const cute_catalog *cat, double L, int ng, const cute_bin_spec *bins, double *h_xi, double *h_sum_dd,
                         uint64_t *h_npairs, double *d_delta, void *d_workspace, size_t bytes, void *stream);

/* Microbenchmarks of the units the pair kernel's roofline is made of (FP32 / packed FP32x2 /
 * integer issue rates, MUFU, shared-memory atomics versus same-address multiplicity, broadcast LDS, and mixes that
 * show which instructions share an issue port).  One persistent 512-thread CTA per SM, timed with clock64() inside the
 * kernels.  Outputs (HOST, n >= cute_peak_count() entries each): lane-operations per clock per SM (a packed f32x2
 * instruction counts 2 per lane) and warp-instructions per clock per SM (may be NULL); cute_peak_name(k) names entry k.
 * d_tmp: DEVICE scratch, 256-byte aligned, >= 1 MiB.  Synchronises the stream. */
int cute_peak_count(void);
const char *cute_peak_name(int idx);
int cute_measure_peaks(double *lane_ops_per_clk_sm, double *instr_per_clk_sm, int n, void *d_tmp, size_t bytes, void *stream);

/* ---- host-side helpers (all pointers HOST) ---- */
/* Bin edges, the single definition: n+1 doubles for axis 0 or 1. */
int cute_bin_edges(const cute_bin_spec *bins, int axis, double *edges_out);
/* Landy-Szalay estimator, Eq. 15. Bins with RR = 0 get xi = 0 and CUTE_WARN_EMPTY_BIN. */
int cute_landy_szalay(const uint64_t *dd, const uint64_t *dr, const uint64_t *rr, uint64_t nd, uint64_t nr,
                      int nbins, double *xi);
/* Natural estimator, Eq. 14. */
int cute_natural_estimator(const uint64_t *dd, const uint64_t *rr, uint64_t nd, uint64_t nr, int nbins, double *xi);
/* Multipoles of xi(r,mu), Eqs. 3-4: xi_l(r) = (2l+1) int_0^1 xi(r,mu) P_l(mu) dmu for l = 0, 2, 4
 * (mid-point rule over the mu bins, which must span [0,1]).  xi: HOST [n_r][n_mu]; out: HOST [3][n_r]. */
int cute_multipoles(const double *xi, int n_r, int n_mu, double *out);
/* Expected unordered pairs of a uniform periodic box, N(N-1)/2 * (4pi/3)(e_{k+1}^3-e_k^3)/L^3
 * (Eqs. 12-13, exact shell volume), and xi = DD/RR - 1. */
int cute_periodic_rr(uint64_t n, double L, const cute_bin_spec *bins, double *rr);
int cute_periodic_xi(const uint64_t *dd, uint64_t n, double L, const cute_bin_spec *bins, double *xi);

#ifdef __cplusplus
}
#endif
#endif /* CUTE_B200_H */
