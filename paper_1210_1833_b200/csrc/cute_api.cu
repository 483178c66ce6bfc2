// cute_api.cu -- the C ABI of include/cute_b200.h: validation, workspace layout, launch planning,
// the float32 error model that decides which pairs are recomputed in float64, and the host-side
// estimators (Eqs. 13-15).
#include "cute_internal.h"
#include <math.h>
#include <new>
#include <stdlib.h>
#include <string.h>
#include <vector>

using namespace cute;

#include <atomic>
static std::atomic<unsigned long long> g_launches{0};
namespace cute { void note_launches(int n) { g_launches += (unsigned long long)n; } }

namespace {

constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr double kU = 1.0 / 16777216.0;   // 2^-24: float32 unit round-off

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

inline int sm_count()
{
    static int n = 0;
    if (!n) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    }
    return n;
}

// ---- workspace layout of one grid -------------------------------------------------------------
struct Layout {
    size_t hi, lo, p64, perm, count, cell_start, scan_tmp, row_nchunks, row_chunk_start, chunks,
        row_kx, row_ylo, row_yhi, status, bbox, part_tmp, part_table, total;
    int part_G, part_Bmax;   // CTAs of the coarse pass; largest bucket count the partition table has room for
    uint32_t n_pad;
    int64_t max_cells, max_rows, max_chunks;
};

constexpr int64_t kOrderCellsMax = 65536;   // mode NONE: cells that only order the points (32^3 or 256^2)

inline int64_t cell_cap(int64_t n) { return n * 2 > 4096 ? n * 2 : 4096; }

inline int part_ctas() { return 2 * sm_count(); }

// rec_bytes: bytes of one raw record of the partition path (16: float32 xyz, 32: otherwise); used when n >= kPartMinN
// Which build a catalogue takes (measured on B200, profiles/r02_build_c5.md, r02_build_c4.md and DESIGN.md 5.1):
//  * float64 / RA-Dec catalogues of >= 2^20 objects: the two-level partition (32-byte records that carry their cell, so
//    sin() and the FP64 cell arithmetic run twice instead of four times: C4 0.42 -> 0.34 ms);
//  * float32 xyz: the partition only when there are many cells (C5, 125 000 cells: 0.89 ms against 1.09 ms one-pass; with
//    64 000 cells the one-pass sort wins, 0.70 against 0.86 ms -- its scattered stores thrash less).
// The workspace is sized for either (the cell count is not known before the box is); build_path = 1 / 2 force one.
// may_partition: can ANY cell count up to max_cells take the partition path?  (Decides whether the workspace reserves the
// partition's record buffer, 16-32 bytes per point: a float32 xyz catalogue whose cells cannot exceed 90 000 -- brute
// force with its <= 32^3 ordering cells, or an explicit small ncell -- never does, and does not pay for it.)
inline bool use_partition(int64_t n, const cute_catalog *c, const cute_grid_spec *s, int64_t ncells)
{
    if (!(n > 0 && (s->build_path == 2 || (s->build_path == 0 && n >= kPartMinN)))) return false;
    const bool f32xyz = c->dtype == CUTE_F32 && c->coord == CUTE_COORD_XYZ;
    return s->build_path == 2 || !f32xyz || ncells > 90000;
}
inline bool may_partition(int64_t n, const cute_catalog *c, const cute_grid_spec *s, int64_t max_cells)
{
    return use_partition(n, c, s, max_cells);   // use_partition is monotone in the cell count
}

Layout make_layout(int64_t n, int want_lo, int want_f64, int64_t max_cells, int64_t max_rows, int rec_bytes)
{
    Layout L;
    memset(&L, 0, sizeof(L));
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
    L.n_pad = (uint32_t)align_up((size_t)(n > 0 ? n : 1), 32);
    L.max_cells = max_cells; L.max_rows = max_rows;
    L.max_chunks = n / kChunk + max_rows + 1;
    L.status = take(16);
    L.bbox = take(8 * 8);
    L.hi = take((size_t)L.n_pad * 16);
    L.lo = want_lo ? take((size_t)L.n_pad * 16) : 0;
    L.p64 = want_f64 ? take((size_t)L.n_pad * 32) : 0;
    L.perm = take((size_t)L.n_pad * 4);
    L.count = take((size_t)(max_cells + 2) * 4);
    L.cell_start = take((size_t)(max_cells + 2) * 4);
    int64_t m = max_cells > max_rows ? max_cells : max_rows;
    L.part_G = part_ctas();
    if (rec_bytes > 0) {
        // The build calls part_shape with the ACTUAL cell count, known only once the box is, and the bucket count is not
        // monotone in the cell count (it lands anywhere in (512, 1024] below the cells-per-bucket cap): size the table
        // for the largest count any ncells <= max_cells can give, max(B(max_cells), kPartMaxBuckets).
        int B, cpb;
        part_shape(max_cells, &B, &cpb);
        if (B < kPartMaxBuckets) B = kPartMaxBuckets;
        L.part_Bmax = B;
        const int64_t tab = (int64_t)B * L.part_G;
        L.part_tmp = take((size_t)L.n_pad * (size_t)rec_bytes);
        L.part_table = take((size_t)(2 * tab + 128) * 4);
        if (tab > m) m = tab;
    }
    L.scan_tmp = take((size_t)(m / 4096 + 2) * 4);
    L.row_nchunks = take((size_t)(max_rows + 2) * 4);
    L.row_chunk_start = take((size_t)(max_rows + 2) * 4);
    L.chunks = take((size_t)L.max_chunks * sizeof(Chunk));
    L.row_kx = take((size_t)(max_rows + 1) * 4);
    L.row_ylo = take((size_t)(max_rows + 1) * 4);
    L.row_yhi = take((size_t)(max_rows + 1) * 4);
    L.total = off;
    return L;
}

int check_catalog(const cute_catalog *c)
{
    if (!c || c->struct_size != sizeof(cute_catalog)) return CUTE_ERR_INVALID_ARG;
    if (c->n < 0 || c->n > 0x7fffffff) return CUTE_ERR_INVALID_ARG;
    if (c->coord < CUTE_COORD_XYZ || c->coord > CUTE_COORD_RADECZ) return CUTE_ERR_INVALID_ARG;
    if (c->dtype != CUTE_F32 && c->dtype != CUTE_F64) return CUTE_ERR_INVALID_ARG;
    if (c->n > 0) {
        if (!c->c0 || !c->c1) return CUTE_ERR_INVALID_ARG;
        if (c->coord != CUTE_COORD_RADEC && !c->c2) return CUTE_ERR_INVALID_ARG;
    }
    if (c->weight && c->coord == CUTE_COORD_RADECZ) return CUTE_ERR_UNSUPPORTED;  // (the radial kind is unweighted)
    return CUTE_OK;
}

int check_grid_spec(const cute_catalog *c, const cute_grid_spec *s)
{
    if (!s || s->struct_size != sizeof(cute_grid_spec)) return CUTE_ERR_INVALID_ARG;
    if (s->mode < CUTE_GRID_NONE || s->mode > CUTE_GRID_SPHERE) return CUTE_ERR_INVALID_ARG;
    if (s->mode == CUTE_GRID_BOX3D && c->coord != CUTE_COORD_XYZ) return CUTE_ERR_INVALID_ARG;
    if (s->mode == CUTE_GRID_SPHERE && c->coord == CUTE_COORD_XYZ) return CUTE_ERR_INVALID_ARG;
    if (s->mode != CUTE_GRID_NONE && !(s->rmax > 0.0)) return CUTE_ERR_INVALID_ARG;
    if (s->mode == CUTE_GRID_BOX3D && s->periodic) {
        if (!(s->size[0] > 0.0) || s->size[1] != s->size[0] || s->size[2] != s->size[0]) return CUTE_ERR_INVALID_ARG;
        if (s->origin[0] != 0.0 || s->origin[1] != 0.0 || s->origin[2] != 0.0) return CUTE_ERR_INVALID_ARG;
    }
    if (s->mode == CUTE_GRID_SPHERE) {
        if (!(s->size[0] > 0.0) || s->size[0] > 360.0 || !(s->size[1] > 0.0)) return CUTE_ERR_INVALID_ARG;
        if (s->origin[1] < -1.0 - 1e-12 || s->origin[1] + s->size[1] > 1.0 + 1e-12) return CUTE_ERR_INVALID_ARG;
        if (s->ncell[0] <= 0 || s->ncell[1] <= 0) return CUTE_ERR_INVALID_ARG;
        if (s->ncell[0] > 65535) return CUTE_ERR_INVALID_ARG;
        if (s->size[0] < 360.0) {
            // an RA span short of the full ring has no wrap-around neighbours: refuse spans so wide that two
            // points could be within rmax of each other THROUGH the gap (the caller must use size[0] = 360)
            const double umax = fmax(fabs(s->origin[1]), fabs(s->origin[1] + s->size[1]));
            const double cosd = sqrt(fmax(0.0, 1.0 - umax * umax));
            if (!(sin(fmin(s->rmax, 0.5 * kPi)) < cosd)) return CUTE_ERR_INVALID_ARG;   // cap reaches a pole
            const double win = asin(sin(s->rmax) / cosd) * (180.0 / kPi);
            if (360.0 - s->size[0] < win) return CUTE_ERR_INVALID_ARG;
        }
    }
    return CUTE_OK;
}

void wants(const cute_catalog *c, const cute_grid_spec *s, int *want_lo, int *want_f64)
{
    int mask = s->kind_mask;
    if (c->coord == CUTE_COORD_XYZ) {
        *want_lo = (mask == 0) || (mask & ((1 << CUTE_RMU) | (1 << CUTE_PISIGMA))) || c->weight != nullptr;   // weights travel in lo.x
        *want_f64 = c->dtype == CUTE_F64;
    } else {
        *want_lo = 0;    // the angular fast path reads the float32 unit vectors only; tiny angles go to float64
        *want_f64 = 1;   // unit vectors are computed in float64 whatever the input type
    }
}

void cell_bounds(const cute_catalog *c, const cute_grid_spec *s, int64_t *max_cells, int64_t *max_rows)
{
    if (s->mode == CUTE_GRID_NONE) { *max_cells = kOrderCellsMax; *max_rows = 1; return; }   // ordering cells
    if (s->mode == CUTE_GRID_SPHERE) { *max_cells = (int64_t)s->ncell[0] * s->ncell[1]; *max_rows = s->ncell[1]; return; }
    if (s->ncell[0] > 0 && s->ncell[1] > 0 && s->ncell[2] > 0) {
        *max_cells = (int64_t)s->ncell[0] * s->ncell[1] * s->ncell[2];
        *max_rows = (int64_t)s->ncell[1] * s->ncell[2];
    } else {
        *max_cells = cell_cap(c->n);
        *max_rows = cell_cap(c->n);
    }
}

} // namespace

extern "C" {

int cute_version(void) { return CUTE_ABI_VERSION; }

uint64_t cute_launch_count(void) { return g_launches.load(); }

const char *cute_strerror(int status)
{
    switch (status) {
    case CUTE_OK: return "ok";
    case CUTE_ERR_INVALID_ARG: return "invalid argument";
    case CUTE_ERR_UNSUPPORTED: return "unsupported combination of kind, grid and binning";
    case CUTE_ERR_WORKSPACE_TOO_SMALL: return "device workspace too small";
    case CUTE_ERR_CUDA: return "CUDA error";
    case CUTE_ERR_OVERFLOW: return "counter overflow";
    case CUTE_ERR_POINT_OUT_OF_BOX: return "a point lies outside the grid box (or is not finite)";
    case CUTE_ERR_GRID_MISMATCH: return "the two grids of a cross-correlation carry different specs";
    case CUTE_ERR_STATIC_SCRATCH_LIMIT: return "too many bins for the built-in scratch of cute_count_pairs_static (CUTE_STATIC_SCRATCH_BYTES): use cute_count_pairs with caller-provided scratch";
    case CUTE_WARN_EMPTY_BIN: return "warning: a bin with RR = 0 got xi = 0";
    }
    return "unknown status";
}

int cute_catalog_bounds(const cute_catalog *cat, void *d_tmp, void *stream, double bounds[6])
{
    int rc = check_catalog(cat);
    if (rc) return rc;
    if (!d_tmp || !bounds || ((uintptr_t)d_tmp & 7)) return CUTE_ERR_INVALID_ARG;
    for (int d = 0; d < 6; d++) bounds[d] = 0.0;
    if (cat->n == 0) return CUTE_OK;
    BuildPlan b;
    memset(&b, 0, sizeof(b));
    b.c0 = cat->c0; b.c1 = cat->c1; b.c2 = cat->coord == CUTE_COORD_RADEC ? cat->c0 : cat->c2;
    b.n = cat->n; b.dtype = cat->dtype; b.bbox = (double *)d_tmp;
    cudaStream_t s = (cudaStream_t)stream;
    if (run_bbox(b, s) != cudaSuccess) return CUTE_ERR_CUDA;
    long long raw[6];
    if (cudaMemcpyAsync(raw, d_tmp, 48, cudaMemcpyDeviceToHost, s) != cudaSuccess || cudaStreamSynchronize(s) != cudaSuccess)
        return CUTE_ERR_CUDA;
    decode_bbox(raw, bounds);
    for (int d = 0; d < 6; d++) if (!isfinite(bounds[d])) return CUTE_ERR_POINT_OUT_OF_BOX;
    return CUTE_OK;
}

int cute_pixelize_workspace_bytes(int n_ra, int n_u, size_t *bytes)
{
    if (!bytes || n_ra < 1 || n_u < 1 || (int64_t)n_ra * n_u > (1ll << 28)) return CUTE_ERR_INVALID_ARG;
    const size_t np = (size_t)n_ra * n_u;
    *bytes = 256 + 2 * align_up((np + 2) * 4, 256) + align_up((np / 4096 + 2) * 4, 256);
    return CUTE_OK;
}

int cute_pixelize(const cute_catalog *cat, double ra0, double dra, double u0, double du, int n_ra, int n_u,
                  double *d_pix_ra, double *d_pix_dec, uint32_t *d_pix_weight, int64_t *npix,
                  void *d_workspace, size_t bytes, void *stream)
{
    int rc = check_catalog(cat);
    if (rc) return rc;
    size_t need = 0;
    if ((rc = cute_pixelize_workspace_bytes(n_ra, n_u, &need))) return rc;
    if (cat->coord == CUTE_COORD_XYZ || cat->weight) return CUTE_ERR_INVALID_ARG;
    if (!(dra > 0.0) || dra > 360.0 || !(du > 0.0) || u0 < -1.0 - 1e-12 || u0 + du > 1.0 + 1e-12) return CUTE_ERR_INVALID_ARG;
    if (!d_pix_ra || !d_pix_dec || !d_pix_weight || !npix || !d_workspace || ((uintptr_t)d_workspace & 255)) return CUTE_ERR_INVALID_ARG;
    if (bytes < need) return CUTE_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t np = (size_t)n_ra * n_u;
    unsigned char *w = (unsigned char *)d_workspace;
    BuildPlan b;
    memset(&b, 0, sizeof(b));
    b.c0 = cat->c0; b.c1 = cat->c1; b.c2 = cat->c0;
    b.n = cat->n; b.coord = CUTE_COORD_RADEC; b.dtype = cat->dtype; b.mode = CUTE_GRID_SPHERE;
    b.origin[0] = ra0; b.size[0] = dra; b.origin[1] = u0; b.size[1] = du;
    b.nc[0] = n_ra; b.nc[1] = n_u; b.nc[2] = 1;
    b.inv_cell[0] = n_ra / dra; b.inv_cell[1] = n_u / du;
    b.ncells = (int64_t)np; b.nrows = n_u;
    b.status = (uint32_t *)w;
    uint32_t *count = (uint32_t *)(w + 256);
    uint32_t *pos = (uint32_t *)(w + 256 + align_up((np + 2) * 4, 256));
    uint32_t *tmp = (uint32_t *)(w + 256 + 2 * align_up((np + 2) * 4, 256));
    if (run_pixelize(b, count, pos, tmp, d_pix_ra, d_pix_dec, d_pix_weight, s) != cudaSuccess) return CUTE_ERR_CUDA;
    uint32_t st = 0, m = 0;
    if (cudaMemcpyAsync(&st, b.status, 4, cudaMemcpyDeviceToHost, s) != cudaSuccess ||
        cudaMemcpyAsync(&m, pos + np, 4, cudaMemcpyDeviceToHost, s) != cudaSuccess || cudaStreamSynchronize(s) != cudaSuccess)
        return CUTE_ERR_CUDA;
    if (st) return CUTE_ERR_POINT_OUT_OF_BOX;
    *npix = (int64_t)m;
    return CUTE_OK;
}

int cute_grid_workspace_bytes(const cute_catalog *cat, const cute_grid_spec *spec, size_t *bytes)
{
    int rc = check_catalog(cat);
    if (rc) return rc;
    if ((rc = check_grid_spec(cat, spec))) return rc;
    if (!bytes) return CUTE_ERR_INVALID_ARG;
    int want_lo, want_f64;
    int64_t mc, mr;
    wants(cat, spec, &want_lo, &want_f64);
    cell_bounds(cat, spec, &mc, &mr);
    if (mc > 0x7ffffff0ll) return CUTE_ERR_INVALID_ARG;
    *bytes = make_layout(cat->n, want_lo, want_f64, mc, mr, !may_partition(cat->n, cat, spec, mc) ? 0 : (cat->dtype == CUTE_F32 && cat->coord == CUTE_COORD_XYZ) ? 16 : 32).total;
    return CUTE_OK;
}

int cute_make_grid(const cute_catalog *cat, const cute_grid_spec *spec, void *d_workspace, size_t bytes, void *stream,
                   cute_grid **out)
{
    int rc = check_catalog(cat);
    if (rc) return rc;
    if ((rc = check_grid_spec(cat, spec))) return rc;
    if (!out || !d_workspace || ((uintptr_t)d_workspace & 255)) return CUTE_ERR_INVALID_ARG;
    *out = nullptr;
    cudaStream_t s = (cudaStream_t)stream;
    int want_lo, want_f64;
    int64_t mc, mr;
    wants(cat, spec, &want_lo, &want_f64);
    cell_bounds(cat, spec, &mc, &mr);
    const Layout L = make_layout(cat->n, want_lo, want_f64, mc, mr, !may_partition(cat->n, cat, spec, mc) ? 0 : (cat->dtype == CUTE_F32 && cat->coord == CUTE_COORD_XYZ) ? 16 : 32);
    if (bytes < L.total) return CUTE_ERR_WORKSPACE_TOO_SMALL;
    unsigned char *w = (unsigned char *)d_workspace;

    BuildPlan b;
    memset(&b, 0, sizeof(b));
    b.c0 = cat->c0; b.c1 = cat->c1; b.c2 = cat->coord == CUTE_COORD_RADEC ? cat->c0 : cat->c2;
    b.weight = cat->weight;
    b.n = cat->n; b.coord = cat->coord; b.dtype = cat->dtype; b.mode = spec->mode; b.periodic = spec->periodic;
    b.want_lo = want_lo; b.want_f64 = want_f64; b.n_pad = L.n_pad;
    b.hi = (float4 *)(w + L.hi); b.lo = want_lo ? (float4 *)(w + L.lo) : nullptr;
    b.p64 = want_f64 ? (double *)(w + L.p64) : nullptr;
    b.perm = spec->no_perm ? nullptr : (uint32_t *)(w + L.perm);
    b.count = (uint32_t *)(w + L.count); b.cell_start = (uint32_t *)(w + L.cell_start);
    b.scan_tmp = (uint32_t *)(w + L.scan_tmp); b.row_nchunks = (uint32_t *)(w + L.row_nchunks);
    b.row_chunk_start = (uint32_t *)(w + L.row_chunk_start); b.chunks = (Chunk *)(w + L.chunks);
    b.row_kx = (int *)(w + L.row_kx); b.row_ylo = (int *)(w + L.row_ylo); b.row_yhi = (int *)(w + L.row_yhi);
    b.status = (uint32_t *)(w + L.status); b.bbox = (double *)(w + L.bbox);
    b.thetamax = spec->rmax;

    // bounding box of the raw coordinates ("a box encompassing the whole catalog is
    // first determined"); also gives the magnitude bound of the float32 error model
    // It is skipped when the caller gave the box (BOX3D with explicit sizes) or nothing needs it (RA/Dec pixels).
    double bbox[6] = {0, 0, 0, 0, 0, 0};
    const bool box_given = spec->mode == CUTE_GRID_BOX3D && spec->size[0] > 0.0 && spec->size[1] > 0.0 && spec->size[2] > 0.0;
    const bool need_bbox = cat->n > 0 && !box_given && !(spec->mode == CUTE_GRID_SPHERE && cat->coord == CUTE_COORD_RADEC);
    if (need_bbox) {
        long long raw[6];
        if (run_bbox(b, s) != cudaSuccess) return CUTE_ERR_CUDA;
        if (cudaMemcpyAsync(raw, b.bbox, sizeof(raw), cudaMemcpyDeviceToHost, s) != cudaSuccess) return CUTE_ERR_CUDA;
        if (cudaStreamSynchronize(s) != cudaSuccess) return CUTE_ERR_CUDA;
        decode_bbox(raw, bbox);
        for (int d = 0; d < 6; d++) if (!isfinite(bbox[d])) return CUTE_ERR_POINT_OUT_OF_BOX;
    } else if (box_given) {
        for (int d = 0; d < 3; d++) { bbox[d] = spec->origin[d]; bbox[3 + d] = spec->origin[d] + spec->size[d]; }
    }

    cute_grid *g = new (std::nothrow) cute_grid;
    if (!g) return CUTE_ERR_INVALID_ARG;
    memset(g, 0, sizeof(*g));
    g->spec = *spec;
    g->coord = cat->coord; g->dtype = cat->dtype; g->has_lo = want_lo; g->has_f64 = want_f64;
    int nc[3] = {1, 1, 1};
    if (spec->mode == CUTE_GRID_BOX3D) {
        for (int d = 0; d < 3; d++) {
            if (!(spec->size[d] > 0.0)) {   // bounding box, widened a little so that the maximum falls inside
                double ext = bbox[3 + d] - bbox[d];
                double pad = 1e-6 * (ext > 0 ? ext : 1.0) + 1e-9 * fmax(fabs(bbox[d]), fabs(bbox[3 + d]));
                g->spec.origin[d] = bbox[d] - pad;
                g->spec.size[d] = ext + 2 * pad;
            }
        }
        int64_t cap = mc;
        for (int d = 0; d < 3; d++) {
            if (spec->ncell[d] > 0) nc[d] = spec->ncell[d];
            else {   // Cell side along y and z: a = rmax / k with an INTEGER k (k cells reach exactly rmax: a side just
                     // below rmax / k costs a whole extra layer of rows), k such that a 128-point work item is about as long
                     // along x as a row is wide (128 = 1.7 n a^3): longer items are sticks that almost every j-point is
                     // partly in range of, shorter ones waste the trimming.  Along x, the contiguous axis, the cells only
                     // set the granularity of the trimmed j-ranges: a / 4.  Measured (cell sweeps): C5
                     // (40, 40, 40) 618 ms -> (10, 40, 40) 562 ms; C3 (50, 50, 50) 49.6 ms -> (17, 67, 67) 44.6 ms; round 1's
                     // rmax/2 and rmax/4 cubes: 58 and 649 ms.  A non-periodic catalogue rarely fills its bounding box
                     // (a survey footprint fills about a third of it): its density is taken three times the box average.
                const double vol = g->spec.size[0] * g->spec.size[1] * g->spec.size[2];
                const double dens = (cat->n > 0 && vol > 0.0 ? (double)cat->n / vol : 0.0) * (spec->periodic ? 1.0 : 3.0);
                int kk = dens > 0.0 ? (int)lround(spec->rmax / cbrt(75.0 / dens)) : 2;
                kk = kk < 2 ? 2 : (kk > 5 ? 5 : kk);
                const double a_want = spec->rmax / kk * (d == 0 ? 0.25 : 1.0);
                double t = floor(g->spec.size[d] / a_want * (1.0 + 1e-12));
                nc[d] = t < 1 ? 1 : (t > 1024 ? 1024 : (int)t);
                if (spec->periodic) {   // nearest cell count with nc >= 2 ceil(rmax/a) + 1
                    auto ok = [&](int n) { return n >= 1 && n >= 2 * (int)ceil(spec->rmax * n / g->spec.size[d] * (1.0 - 1e-12)) + 1; };
                    int best = 0;
                    for (int n = nc[d]; n >= 3 && !best; n--) if (ok(n)) best = n;
                    for (int n = nc[d] + 1; n <= nc[d] + 64 && !best; n++) if (ok(n)) best = n;
                    if (!best) { delete g; return CUTE_ERR_UNSUPPORTED; }
                    nc[d] = best;
                }
            }
        }
        if (!(spec->ncell[0] > 0 && spec->ncell[1] > 0 && spec->ncell[2] > 0))
            while ((int64_t)nc[0] * nc[1] * nc[2] > cap || (int64_t)nc[1] * nc[2] > mr) {
                int dmax = nc[0] >= nc[1] && nc[0] >= nc[2] ? 0 : (nc[1] >= nc[2] ? 1 : 2);
                nc[dmax] = (nc[dmax] * 3 + 3) / 4;
            }
        if (nc[0] > 65535) { delete g; return CUTE_ERR_INVALID_ARG; }
        for (int d = 0; d < 3; d++) {
            g->cell[d] = g->spec.size[d] / nc[d];
            b.origin[d] = g->spec.origin[d]; b.size[d] = g->spec.size[d]; b.inv_cell[d] = nc[d] / g->spec.size[d];
        }
        if (spec->periodic)
            for (int d = 0; d < 3; d++) {
                int k = (int)ceil(spec->rmax / g->cell[d] * (1.0 - 1e-12));
                if (nc[d] < 2 * k + 1) { delete g; return CUTE_ERR_UNSUPPORTED; }   // a cell would be met through two images
            }
    } else if (spec->mode == CUTE_GRID_SPHERE) {
        nc[0] = spec->ncell[0]; nc[1] = spec->ncell[1];
        for (int d = 0; d < 2; d++) {
            g->cell[d] = spec->size[d] / nc[d];
            b.origin[d] = spec->origin[d]; b.size[d] = spec->size[d]; b.inv_cell[d] = nc[d] / spec->size[d];
        }
    }
    for (int d = 0; d < 3; d++) { b.nc[d] = nc[d]; g->spec.ncell[d] = nc[d]; }
    b.ncells = (int64_t)nc[0] * nc[1] * nc[2];
    b.nrows = (int64_t)nc[1] * nc[2];
    g->ncells = b.ncells; g->nrows = b.nrows;
    if (spec->mode == CUTE_GRID_NONE && cat->n > 0) {
        // Brute force evaluates every pair, in any order: sort the points by the cells of a coarse box (or
        // pixel map) over the bounding box, ~48 points per cell, so that the 128 i-points of a warp and the
        // j-points of a tile are neighbours in space and the in-range test is (nearly) uniform over the warp.
        b.order_only = 1;
        b.periodic = 0;
        int m;
        if (cat->coord == CUTE_COORD_XYZ) {
            b.mode = CUTE_GRID_BOX3D;
            m = (int)lround(cbrt((double)cat->n / 48.0));
            m = m < 1 ? 1 : (m > 32 ? 32 : m);
            for (int d = 0; d < 3; d++) {
                const double ext = bbox[3 + d] - bbox[d];
                const double pad = 1e-6 * (ext > 0 ? ext : 1.0) + 1e-9 * fmax(fabs(bbox[d]), fabs(bbox[3 + d]));
                b.origin[d] = bbox[d] - pad; b.size[d] = ext + 2 * pad; b.nc[d] = m; b.inv_cell[d] = m / b.size[d];
            }
        } else {
            b.mode = CUTE_GRID_SPHERE;
            m = (int)lround(sqrt((double)cat->n / 48.0));
            m = m < 1 ? 1 : (m > 256 ? 256 : m);
            const double ext = fmin(360.0, (bbox[3] - bbox[0]) * (1.0 + 1e-9) + 1e-9);
            b.origin[0] = ext < 360.0 ? bbox[0] - 0.5 * (ext - (bbox[3] - bbox[0])) : 0.0;
            b.size[0] = ext;
            const double u0 = fmax(-1.0, sin(fmax(-90.0, bbox[1]) * (kPi / 180.0)) - 1e-9);
            const double u1 = fmin(1.0, sin(fmin(90.0, bbox[4]) * (kPi / 180.0)) + 1e-9);
            b.origin[1] = u0; b.size[1] = fmax(u1 - u0, 1e-9);
            b.nc[0] = m; b.nc[1] = m; b.nc[2] = 1;
            b.inv_cell[0] = m / b.size[0]; b.inv_cell[1] = m / b.size[1];
        }
        b.ncells = (int64_t)b.nc[0] * b.nc[1] * b.nc[2];
        b.nrows = 1;
    }
    // magnitude bound
    double m = 0.0;
    if (cat->coord == CUTE_COORD_XYZ) for (int d = 0; d < 6; d++) m = fmax(m, fabs(bbox[d]));
    else m = fmax(fabs(bbox[2]), fabs(bbox[5]));   // RADECZ: |z| (unit vectors are <= 1)
    g->maxabs = m;
    for (int d = 0; d < 6; d++) g->bbox[d] = bbox[d];
    g->has_bbox = (need_bbox || box_given) ? 1 : 0;

    if (use_partition(cat->n, cat, spec, b.ncells) && b.mode != CUTE_GRID_NONE) {   // large catalogue: two-level partition (grid_build.cu)
        b.part_tmp = w + L.part_tmp; b.part_table = (uint32_t *)(w + L.part_table); b.part_G = L.part_G;
        part_shape(b.ncells, &b.part_B, &b.part_cpb);
        if (b.part_B > L.part_Bmax) { delete g; return CUTE_ERR_WORKSPACE_TOO_SMALL; }   // (cannot happen: make_layout)
        b.part_shift = 0;
        while ((1 << b.part_shift) < b.part_cpb) b.part_shift++;
    }
    if (run_build(b, s) != cudaSuccess) { delete g; return CUTE_ERR_CUDA; }
    uint32_t st[3] = {0, 0, 0};
    if (cudaMemcpyAsync(st, b.status, 12, cudaMemcpyDeviceToHost, s) != cudaSuccess || cudaStreamSynchronize(s) != cudaSuccess) {
        delete g;
        return CUTE_ERR_CUDA;
    }
    if (st[0]) { delete g; return CUTE_ERR_POINT_OUT_OF_BOX; }
    if ((int64_t)st[1] > L.max_chunks) { delete g; return CUTE_ERR_WORKSPACE_TOO_SMALL; }

    GridView &v = g->view;
    v.hi = b.hi; v.lo = b.lo; v.p64 = b.p64; v.cell_start = b.cell_start; v.chunks = b.chunks;
    v.row_kx = b.row_kx; v.row_ylo = b.row_ylo; v.row_yhi = b.row_yhi;
    v.n = (uint32_t)cat->n; v.n_pad = L.n_pad; v.nchunks = st[1];
    v.ncx = nc[0]; v.ncy = nc[1]; v.ncz = nc[2];
    g->d_perm = b.perm;
    g->weighted = cat->weight != nullptr; g->wmax = st[2] > 0 ? st[2] : 1u;
    // algorithmic HBM bytes of the build: read the coordinates twice (cell id,
    // scatter), write hi (+lo, +p64) and perm; counts, scan and cursors per cell
    const double in_b = (cat->dtype == CUTE_F64 ? 8.0 : 4.0) * (cat->coord == CUTE_COORD_RADEC ? 2 : 3);
    g->build_bytes = (double)cat->n * (2 * in_b + 16 + (want_lo ? 16 : 0) + (want_f64 ? 32 : 0) + (spec->no_perm ? 0 : 4)) + (double)b.ncells * 20;
    *out = g;
    return CUTE_OK;
}

void cute_free_grid(cute_grid *g) { delete g; }

int cute_grid_get_info(const cute_grid *g, cute_grid_info *info)
{
    if (!g || !info || info->struct_size != sizeof(cute_grid_info)) return CUTE_ERR_INVALID_ARG;
    info->n = g->view.n; info->mode = g->spec.mode; info->periodic = g->spec.periodic;
    info->kind_coord = g->coord; info->dtype = g->dtype; info->has_lo = g->has_lo; info->has_f64 = g->has_f64;
    for (int d = 0; d < 3; d++) { info->ncell[d] = g->spec.ncell[d]; info->origin[d] = g->spec.origin[d]; info->cell[d] = g->cell[d]; info->size[d] = g->spec.size[d]; }
    info->ncells = g->ncells; info->nrows = g->nrows; info->nchunks = g->view.nchunks;
    info->d_hi = g->view.hi; info->d_lo = g->view.lo; info->d_perm = g->d_perm; info->d_cell_start = g->view.cell_start;
    info->build_bytes = g->build_bytes;
    return CUTE_OK;
}

} // extern "C"

// =============================================================================== pair counting
namespace {

int check_bins(int kind, const cute_bin_spec *b)
{
    if (!b || b->struct_size != sizeof(cute_bin_spec)) return CUTE_ERR_INVALID_ARG;
    if (kind < CUTE_ANGULAR || kind > CUTE_PISIGMA) return CUTE_ERR_INVALID_ARG;
    if (b->n1 < 1 || b->n1 > 65536 || !(b->lo1 < b->hi1) || !(b->lo1 >= 0.0)) return CUTE_ERR_INVALID_ARG;
    if (b->log1 && !(b->lo1 > 0.0)) return CUTE_ERR_INVALID_ARG;
    const bool two = (kind == CUTE_RMU || kind == CUTE_RADIAL || kind == CUTE_PISIGMA);
    if (two && (b->n2 < 1 || b->n2 > 65536 || !(b->lo2 < b->hi2) || !(b->lo2 >= 0.0))) return CUTE_ERR_INVALID_ARG;
    if (!two && b->n2 != 0) return CUTE_ERR_INVALID_ARG;
    if ((int64_t)b->n1 * (b->n2 > 0 ? b->n2 : 1) > (1 << 20)) return CUTE_ERR_INVALID_ARG;
    if (kind == CUTE_RADIAL && !(b->aperture_rad > 0.0 && b->aperture_rad < kPi)) return CUTE_ERR_INVALID_ARG;
    if (kind == CUTE_ANGULAR && b->hi1 > kPi) return CUTE_ERR_INVALID_ARG;
    if (b->box_L != 0.0) {
        if (kind != CUTE_MONOPOLE || !(b->box_L > 0.0)) return CUTE_ERR_UNSUPPORTED;
        if (b->hi1 > 0.5 * b->box_L) return CUTE_ERR_INVALID_ARG;   // uniqueness of the minimum image (reading S13)
    }
    if ((kind == CUTE_RMU || kind == CUTE_PISIGMA) && b->log1) return CUTE_ERR_UNSUPPORTED;
    return CUTE_OK;
}

void fill_edges(const cute_bin_spec *b, int axis, double *e)
{
    const int n = axis == 0 ? b->n1 : b->n2;
    const double lo = axis == 0 ? b->lo1 : b->lo2, hi = axis == 0 ? b->hi1 : b->hi2;
    const int lg = axis == 0 ? b->log1 : 0;
    for (int k = 0; k <= n; k++)
        e[k] = lg ? exp(log(lo) + (double)k * (log(hi) - log(lo)) / (double)n) : lo + (hi - lo) * (double)k / (double)n;
    e[0] = lo; e[n] = hi;
}

struct ScratchLayout { size_t queue, status, stats, edges1, edges2, total; };
ScratchLayout scratch_layout(const cute_bin_spec *b)
{
    ScratchLayout S;
    S.queue = 0; S.status = 16; S.stats = 32; S.edges1 = 64;
    S.edges2 = S.edges1 + 8 * (size_t)(b->n1 + 1);
    S.total = align_up(S.edges2 + 8 * (size_t)(b->n2 + 1), 256);
    return S;
}

inline double chord_of(double theta) { return 2.0 * sin(0.5 * theta); }

// theta/chord as a function of q = chord^2: theta = 2 asin(c/2)
inline double theta_over_chord(double q)
{
    if (q < 1e-8) return 1.0 + q / 24.0 + q * q * (3.0 / 640.0);
    const double c = sqrt(q);
    return 2.0 * asin(fmin(1.0, 0.5 * c)) / c;
}

// c0 + c1 q + c2 q^2 + c3 q^3 through F at the four Chebyshev nodes of [0, qmax]: a near-minimax cubic, orders of
// magnitude closer than the Taylor coefficients at the far end of the range (theta up to tens of degrees)
template <class Fn>
void fit_cubic(Fn F, double qmax, double c[4])
{
    double x[4], d[4];
    for (int k = 0; k < 4; k++) { x[k] = 0.5 * qmax * (1.0 + cos((2 * k + 1) * kPi / 8.0)); d[k] = F(x[k]); }
    for (int j = 1; j < 4; j++)                       // Newton divided differences, in place
        for (int k = 3; k >= j; k--) d[k] = (d[k] - d[k - 1]) / (x[k] - x[k - j]);
    // expand d0 + d1 (q-x0) + d2 (q-x0)(q-x1) + d3 (q-x0)(q-x1)(q-x2) into monomials (Horner from the top)
    double p[4] = {d[3], 0.0, 0.0, 0.0};
    for (int j = 2; j >= 0; j--) {
        for (int k = 3; k > 0; k--) p[k] = p[k - 1] - x[j] * p[k];   // multiply by (q - x_j)
        p[0] = -x[j] * p[0] + d[j];
    }
    c[0] = p[0]; c[1] = p[1]; c[2] = p[2]; c[3] = p[3];
}

// The float32 error model.  Fills a1, a2, q_hi, dz_hi.  `tau` bounds |t_float32 - t_exact| in bins;
// derivation in DESIGN.md "Precision".
int plan_fast_path(PairParams &p, int kind, const cute_grid *g1, const cute_grid *g2, const cute_bin_spec *b, double tau_scale)
{
    const double M = fmax(g1->maxabs, g2->maxabs);
    const bool f64in = (g1->dtype == CUTE_F64) || (g2->dtype == CUTE_F64);
    const bool minimg = (kind == CUTE_MONOPOLE && p.mode == CUTE_GRID_NONE && b->box_L > 0.0);
    const double n1 = b->n1;
    FastAxis &A = p.a1, &B = p.a2;
    memset(&A, 0, sizeof(A));
    memset(&B, 0, sizeof(B));
    A.n = b->n1; B.n = b->n2;
    double tau1 = 0.0, rpad = 0.0;
    if (kind == CUTE_PISIGMA) {
        // pi = |s.l| / |l| with s.l = |x_i|^2 - |x_j|^2 from the hi/lo squares (no cancellation) and
        // |l|^2 = 2|x_i|^2 + 2|x_j|^2 - q;  sigma = sqrt(q - pi^2).  Errors: q carries the float32 input rounding
        // (e_r on r), pi only relative rounding, sigma inherits both divided by sigma: tau_2 = a + b / sigma.
        const double e_d = (f64in ? 2.0 * kU * M : 0.0) + kU * (sqrt(b->hi1 * b->hi1 + b->hi2 * b->hi2) * 1.01);
        const double e_r = sqrt(3.0) * e_d;
        const double rmaxp = sqrt(b->hi1 * b->hi1 + b->hi2 * b->hi2);
        const double inv1 = n1 / (b->hi1 - b->lo1), inv2 = (double)b->n2 / (b->hi2 - b->lo2);
        A.S = (float)inv1; A.O = (float)(-b->lo1 * inv1);
        B.S = (float)inv2; B.O = (float)(-b->lo2 * inv2);
        // e_pi, the absolute error of pi, depends on the pair: |l|^2 = 2(|x_i|^2 + |x_j|^2) - q cancels when |l| << |x|
        // (error 8u M^2 on |l|^2, i.e. pi * 4u M^2 / |l|^2 on pi), and s.l carries 2^-40 M^2 absolute (generous):
        //   e_pi = Ep0 + Kp w1^2,  w1 = 1/|l|   (kernel: A.c2 + A.c1 w1^2, scaled by 1.25 tau_scale here)
        const double sc = 1.25 * tau_scale;
        const double Ep0 = sc * (16.0 * kU * rmaxp + ldexp(1.0, -40) * (M * M + 1.0));
        const double Kp = sc * (4.0 * kU * (3.0 * M * M + 1.0) * rmaxp + ldexp(1.0, -40) * (M * M + 1.0));
        A.c1 = (float)Kp; A.c2 = (float)Ep0;
        tau1 = 4.0 * kU * (inv1 * b->hi1 + fabs((double)A.O) + n1 + 1.0);          // constant part; + S1 e_pi in the kernel
        // d(sigma) = (r e_r + pi e_pi) / sigma:  tau_2 = B.tau + w2 (B.tau_w + A.c3 e_pi),  w2 = 1/sigma
        B.tau = (float)(sc * (inv2 * 16.0 * kU * rmaxp + 4.0 * kU * (inv2 * b->hi2 + fabs((double)B.O) + b->n2 + 1.0)));
        B.tau_w = (float)(sc * inv2 * rmaxp * e_r * 1.01);
        A.c3 = (float)(inv2 * rmaxp * 1.01);
        const double rpad = (rmaxp * (1.0 + 1e-4) + e_r) * (1.0 + 16.0 * kU);
        p.q_hi = (float)(rpad * rpad * (1.0 + 8.0 * kU));
        if (b->lo1 == 0.0 && b->lo2 == 0.0) p.simple = 1;
    } else if (kind == CUTE_MONOPOLE || kind == CUTE_RMU) {
        // error of one separation component: input rounding, subtraction rounding, periodic image
        // (brute-force minimum image |d'| = min(|d|, L - |d|): the roundings of d and of L - |d| are <= uL each; 3uL is kept)
        double e_d = (f64in ? 2.0 * kU * M : 0.0) + kU * (minimg ? 3.0 * b->box_L : b->hi1 * 1.01);
        if (p.periodic && !minimg) {
            // the periodic image is taken by subtracting L from the larger coordinate: exact (Sterbenz) when the wrapped
            // cells lie in the upper half of the box, i.e. nc >= 2k + 2 on every axis; else one rounding at ulp(2L)
            bool exact = true;
            for (int d = 0; d < 3; d++) {
                const int k = (int)ceil(g1->spec.rmax / g1->cell[d] * (1.0 - 1e-12));
                if (g1->spec.ncell[d] < 2 * k + 2) exact = false;
            }
            if (!exact) e_d += 2.0 * kU * 2.0 * b->box_L;
        }
        const double e_r = sqrt(3.0) * e_d;                    // | |d+e| - |d| | <= |e|
        const double rel = 8.0 * kU;                           // q accumulation + MUFU sqrt/lg2
        if (b->log1) {
            const double sc = n1 / log(b->hi1 / b->lo1);       // dt = sc * dr/r
            A.S = (float)(0.5 * sc * log(2.0));                // t = sc*ln(r/lo) = (sc ln2 / 2) * log2(q) - sc ln(lo)
            A.O = (float)(-sc * log(b->lo1));
            if (kind == CUTE_MONOPOLE) {
                // pair-dependent: tau = tau1 + tau_w / r (kernel), tau_w = sc e_r
                tau1 = sc * rel + 0.5 * sc * log(2.0) * (1.0 / 2097152.0) +
                       4.0 * kU * (fabs((double)A.S) * 260.0 + fabs((double)A.O) + n1 + 1.0);
                A.tau_w = (float)(1.25 * tau_scale * sc * e_r);
                rpad = b->hi1 * (1.0 + 2.0 * (tau1 + sc * e_r / b->hi1) / sc);
            } else {
                tau1 = sc * (e_r / b->lo1 + rel) + 0.5 * sc * log(2.0) * (1.0 / 2097152.0) +
                       4.0 * kU * (fabs((double)A.S) * 260.0 + fabs((double)A.O) + n1 + 1.0);
                rpad = b->hi1 * (1.0 + 2.0 * tau1 / sc);
            }
        } else {
            const double inv = n1 / (b->hi1 - b->lo1);
            A.S = (float)inv;
            A.O = (float)(-b->lo1 * inv);
            tau1 = inv * (e_r + rel * b->hi1) + 4.0 * kU * (inv * b->hi1 + fabs((double)A.O) + n1 + 1.0);
            rpad = b->hi1 + 2.0 * tau1 / inv;
        }
        tau1 *= 1.25 * tau_scale;
        rpad = (rpad + e_r) * (1.0 + 16.0 * kU);
        p.q_hi = (float)(rpad * rpad * (1.0 + 8.0 * kU));
        if (kind == CUTE_RMU) {
            const double inv2 = (double)b->n2 / (b->hi2 - b->lo2);
            B.S = (float)inv2;
            B.O = (float)(-b->lo2 * inv2);
            // dmu <= mu * (sqrt3 e_d / r) + 16u ;  1/r = w * |l| <= w * 2 sqrt3 M
            B.tau = (float)(1.25 * tau_scale * (inv2 * 16.0 * kU + 4.0 * kU * (inv2 + fabs((double)B.O) + b->n2 + 1.0)));
            B.tau_w = (float)(1.25 * tau_scale * inv2 * e_r * 2.0 * sqrt(3.0) * M);
            // |l|^2 = 2(|x_i|^2 + |x_j|^2) - q cancels when |l| << |x| (a catalogue around the origin): its
            // error 8u 3M^2 enters mu as mu * 4u 3M^2 / |l|^2, and 1/|l|^2 = w^2 q in the kernel
            A.c1 = (float)(1.25 * tau_scale * inv2 * 4.0 * kU * (3.0 * M * M + 1.0));
            // A catalogue far from the origin (every survey footprint): |l| = |2 x_i + (x_j - x_i)| >= 2 dmin - r, so the
            // |l|^-2 term is bounded by a constant and folded into tau; with bins from 0 this is the PK_SIMPLE variant
            auto dmin = [](const cute_grid *g) {
                double d2 = 0.0;
                for (int d = 0; d < 3; d++) {
                    const double lo = g->bbox[d], hi = g->bbox[3 + d];
                    const double a = lo > 0.0 ? lo : (hi < 0.0 ? -hi : 0.0);
                    d2 += a * a;
                }
                return g->has_bbox ? sqrt(d2) : 0.0;
            };
            const double lmin = 2.0 * fmax(dmin(g1), dmin(g2)) * (1.0 - 1e-6) - sqrt((double)p.q_hi) * 1.001;
            if (lmin > 0.0 && b->lo1 == 0.0 && b->lo2 == 0.0) {
                B.tau = (float)((double)B.tau + (double)A.c1 / (lmin * lmin) * 1.001);
                p.simple = 1;
            }
        } else if (b->lo1 == 0.0 && !b->log1) p.simple = 1;
    } else {
        // unit vectors.  ANGULAR: float32 components (each within u of the float64 one), so the chord carries an
        // ABSOLUTE error sqrt3 * 2u ~ 2e-7; RADIAL: coarse test only.
        const double th_hi = kind == CUTE_ANGULAR ? b->hi1 : b->aperture_rad;
        const double c_hi = chord_of(th_hi), q_hi = c_hi * c_hi;
        if (kind == CUTE_RADIAL) {
            const double c = c_hi * (1.0 + 1e-6) + 8.0 * kU;
            p.q_hi = (float)(c * c * (1.0 + 8.0 * kU));
            p.dz_hi = (float)(b->hi2 * (1.0 + 1e-6) + 4.0 * kU * M + 1e-30);
            p.always_refine = 1;
            return CUTE_OK;
        }
        const double c_lo = chord_of(b->lo1 > 0.0 ? b->lo1 : 0.0);
        const double e_abs = sqrt(3.0) * 2.0 * kU * 1.001;
        const double stretch = 1.0 / sqrt(fmax(1e-6, 1.0 - 0.25 * q_hi));     // d theta / d chord
        const double rel = 12.0 * kU;
        const int NS = 4096;
        double series_err = 0.0;
        if (b->log1) {
            // t = sc * ln(theta/lo) = (sc ln2/2) log2(theta^2) - sc ln(lo)
            const double sc = n1 / log(b->hi1 / b->lo1);
            A.S = (float)(0.5 * sc * log(2.0));
            A.O = (float)(-sc * log(b->lo1));
            // theta^2 = 4 asin^2(c/2) = q (1 + q/12 + q^2/90 + q^3/560 + ...): the kernel takes log2 of q*poly(q)
            // (Taylor: 1, 1/12, 1/90; fitted over the range actually binned instead)
            double cf[4];
            fit_cubic([](double q) { const double t = theta_over_chord(q); return t * t; }, fmin(4.0, q_hi * 1.02), cf);
            A.c1 = (float)cf[0]; A.c2 = (float)cf[1]; A.c3 = (float)cf[2]; A.c4 = (float)cf[3];
            for (int i = 1; i <= NS; i++) {
                const double q = fmin(4.0, q_hi * 1.02) * (double)i / NS;
                const double toc = theta_over_chord(q);
                const double se = (double)A.c1 + q * ((double)A.c2 + q * ((double)A.c3 + q * (double)A.c4));
                series_err = fmax(series_err, 0.5 * sc * fabs(log(toc * toc / se)));
            }
            // The absolute chord error is a RELATIVE error e_abs / c of theta, so tau = tau_a + tau_b / c depends on the pair.
            // The kernel's one threshold (a1.tau) is sized for chords >= c_mid, which is nearly every pair (the number of
            // pairs grows as theta^2); a block holding a closer pair is tested with tau_mid (sized for the closest chord
            // that is still decided in float32, c_min) and its pairs are then decided one by one with their own tau.
            // Pairs closer than c_min always go to float64; c_min is where tau reaches 0.1 bin (or lo, if that is larger).
            // Below lo nothing can be mis-binned INTO range as long as lo >> e_abs.
            if (c_lo < 16.0 * e_abs) p.always_refine = 1;          // (bins finer than the float32 unit vectors resolve)
            const double lgmax = fabs(log2(fmax(c_lo * c_lo * 0.25, 1e-37))) + 2.0;
            const double ks = 1.25 * tau_scale;
            const double tau_a = ks * (sc * stretch * rel + (double)A.S * (1.0 / 2097152.0 + 2.0 * kU * lgmax) +
                                       4.0 * kU * ((double)A.S * lgmax + fabs((double)A.O) + n1 + 1.0) + 1.5 * series_err);
            const double tau_b = ks * sc * stretch * e_abs;
            double c_min = fmax(c_lo, tau_b / 0.1);
            c_min = fmin(c_min, 0.5 * c_hi);
            double c_mid = fmax(c_min, fmin(0.1 * c_hi, 64.0 * cbrt(sc * stretch * e_abs * c_hi * c_hi)));
            c_mid = fmin(c_mid, 0.5 * c_hi);
            if (c_min <= c_lo) p.q_small = 0.f;
            else { const double cs = c_min * 1.001 + 2.0 * e_abs; p.q_small = (float)(cs * cs * (1.0 + 16.0 * kU)); }
            { const double cs = c_mid * 1.001 + 2.0 * e_abs; p.q_mid = (float)(cs * cs * (1.0 + 16.0 * kU)); }
            // (the float32 chord is within e_abs of the true one: 1 / c_true <= (1 + 2 e_abs / c) / c_float32, c >= c_lo)
            p.tau_a = (float)(tau_a * 1.0001);
            p.tau_b = (float)(tau_b * (1.0 + 2.0 * e_abs / fmax(c_min, 1e-18)) * 1.001);
            p.tau_mid = (float)(tau_a + tau_b / fmax(c_min, 1e-18));
            tau1 = tau_a + tau_b / c_mid;
            const double cp = chord_of(fmin(kPi, b->hi1 * (1.0 + 2.0 * tau1 / sc))) * (1.0 + 32.0 * kU) + e_abs;
            p.q_hi = (float)(fmin(4.0, cp * cp) * (1.0 + 8.0 * kU));
        } else {
            // t = (theta - lo)/D,  theta = c (1 + q/24 + 3 q^2/640 + ...)
            const double inv = n1 / (b->hi1 - b->lo1);
            A.S = (float)inv;
            A.O = (float)(-b->lo1 * inv);
            // (Taylor: 1, 1/24, 3/640; fitted over the range actually binned instead)
            double cf[4];
            fit_cubic([](double q) { return theta_over_chord(q); }, fmin(4.0, q_hi * 1.02), cf);
            A.c1 = (float)cf[0]; A.c2 = (float)cf[1]; A.c3 = (float)cf[2]; A.c4 = (float)cf[3];
            for (int i = 0; i <= NS; i++) {
                const double q = fmin(4.0, q_hi * 1.02) * (double)i / NS;
                const double c = sqrt(q);
                const double ex = c * theta_over_chord(q);
                const double se = c * ((double)A.c1 + q * ((double)A.c2 + q * ((double)A.c3 + q * (double)A.c4)));
                series_err = fmax(series_err, fabs(ex - se));
            }
            tau1 = inv * (stretch * (e_abs + rel * c_hi) + 1.5 * series_err) + 4.0 * kU * (inv * th_hi + fabs((double)A.O) + n1 + 1.0);
            tau1 *= 1.25 * tau_scale;
            const double cp = chord_of(fmin(kPi, b->hi1 + 2.0 * tau1 / inv)) * (1.0 + 32.0 * kU) + e_abs;
            p.q_hi = (float)(fmin(4.0, cp * cp) * (1.0 + 8.0 * kU));
            p.angpoly = 1;
        }
        if (p.q_hi >= 4.0f) p.q_hi = 5.0f;   // whole sphere in range
        if (tau1 > 0.2) p.always_refine = 1;  // bins too fine for float32 unit vectors: everything in float64
    }
    A.tau = (float)tau1;
    return CUTE_OK;
}

bool same_spec(const cute_grid *a, const cute_grid *b)
{
    if (a->spec.mode != b->spec.mode || a->spec.periodic != b->spec.periodic || a->coord != b->coord) {
        // coordinates may differ only between RADEC and RADECZ
        if (a->spec.mode != b->spec.mode || a->spec.periodic != b->spec.periodic) return false;
        if (a->coord == CUTE_COORD_XYZ || b->coord == CUTE_COORD_XYZ) return false;
    }
    if (a->spec.mode == CUTE_GRID_NONE) return true;
    for (int d = 0; d < 3; d++) {
        if (a->spec.ncell[d] != b->spec.ncell[d]) return false;
        if (a->spec.mode == CUTE_GRID_SPHERE && d == 2) continue;
        if (a->spec.origin[d] != b->spec.origin[d] || a->spec.size[d] != b->spec.size[d]) return false;
    }
    return a->spec.rmax == b->spec.rmax;
}

} // namespace

extern "C" {

int cute_bin_edges(const cute_bin_spec *bins, int axis, double *edges_out)
{
    if (!bins || bins->struct_size != sizeof(cute_bin_spec) || !edges_out || axis < 0 || axis > 1) return CUTE_ERR_INVALID_ARG;
    const int n = axis == 0 ? bins->n1 : bins->n2;
    const double lo = axis == 0 ? bins->lo1 : bins->lo2, hi = axis == 0 ? bins->hi1 : bins->hi2;
    if (n < 1 || !(lo < hi) || (axis == 0 && bins->log1 && !(lo > 0.0))) return CUTE_ERR_INVALID_ARG;
    fill_edges(bins, axis, edges_out);
    return CUTE_OK;
}

int cute_count_scratch_bytes(const cute_bin_spec *bins, const cute_count_opts *opts, size_t *bytes)
{
    (void)opts;
    if (!bins || bins->struct_size != sizeof(cute_bin_spec) || !bytes || bins->n1 < 1 || bins->n2 < 0) return CUTE_ERR_INVALID_ARG;
    *bytes = scratch_layout(bins).total;
    return CUTE_OK;
}

// plans (and, unless nitems_out is given, enqueues) one pair count
static int count_impl(int kind, const cute_grid *g1, const cute_grid *g2, const cute_bin_spec *bins, uint64_t *d_hist,
                      void *d_scratch, size_t scratch_bytes, const cute_count_opts *opts, void *stream, int64_t *nitems_out)
{
    const bool dry = nitems_out != nullptr;
    int rc = check_bins(kind, bins);
    if (rc) return rc;
    if (!g1) return CUTE_ERR_INVALID_ARG;
    if (!dry && (!d_hist || !d_scratch || ((uintptr_t)d_scratch & 15))) return CUTE_ERR_INVALID_ARG;
    if (opts && opts->struct_size != sizeof(cute_count_opts)) return CUTE_ERR_INVALID_ARG;
    const bool is_auto = (g2 == nullptr || g2 == g1);
    if (is_auto) g2 = g1;
    if (!is_auto && !same_spec(g1, g2)) return CUTE_ERR_GRID_MISMATCH;
    const ScratchLayout SL = scratch_layout(bins);
    if (!dry && scratch_bytes < SL.total) return CUTE_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t s = (cudaStream_t)stream;
    const int mode = g1->spec.mode;
    // kind / coordinates / grid compatibility
    const bool xyz = g1->coord == CUTE_COORD_XYZ;
    if ((kind == CUTE_MONOPOLE || kind == CUTE_RMU || kind == CUTE_PISIGMA) != xyz) return CUTE_ERR_INVALID_ARG;
    if (kind == CUTE_RADIAL && (g1->coord != CUTE_COORD_RADECZ || g2->coord != CUTE_COORD_RADECZ)) return CUTE_ERR_INVALID_ARG;
    if ((kind == CUTE_RMU || kind == CUTE_PISIGMA) && (!g1->has_lo || !g2->has_lo)) return CUTE_ERR_INVALID_ARG;
    if ((kind == CUTE_RMU || kind == CUTE_PISIGMA) && mode == CUTE_GRID_BOX3D && g1->spec.periodic) return CUTE_ERR_UNSUPPORTED;
    const double vmax = kind == CUTE_RADIAL ? bins->aperture_rad
                                           : (kind == CUTE_PISIGMA ? sqrt(bins->hi1 * bins->hi1 + bins->hi2 * bins->hi2) : bins->hi1);
    if (mode != CUTE_GRID_NONE && vmax > g1->spec.rmax * (1.0 + 1e-12)) return CUTE_ERR_INVALID_ARG;
    if (mode == CUTE_GRID_BOX3D && g1->spec.periodic) {
        if (kind != CUTE_MONOPOLE || bins->box_L != g1->spec.size[0]) return CUTE_ERR_INVALID_ARG;
    } else if (mode == CUTE_GRID_BOX3D && bins->box_L > 0.0) return CUTE_ERR_INVALID_ARG;

    if (mode == CUTE_GRID_NONE && bins->box_L > 0.0 && g1->view.n > 0 && g2->view.n > 0) {
        // the float32 fast path takes the minimum image as min(|d|, L - |d|), which needs |d| <= L: refuse
        // catalogues that span more than one box side (unwrapped coordinates) instead of binning them wrongly
        for (int d = 0; d < 3; d++) {
            const double lo = fmin(g1->bbox[d], g2->bbox[d]), hi = fmax(g1->bbox[3 + d], g2->bbox[3 + d]);
            if (!g1->has_bbox || !g2->has_bbox || !(hi - lo <= bins->box_L)) return CUTE_ERR_POINT_OUT_OF_BOX;
        }
    }
    if (g1->weighted != g2->weighted) return CUTE_ERR_INVALID_ARG;
    if (g1->weighted && kind == CUTE_RADIAL) return CUTE_ERR_UNSUPPORTED;
    if (g1->weighted && xyz && (!g1->has_lo || !g2->has_lo)) return CUTE_ERR_INVALID_ARG;
    PairParams p;
    memset(&p, 0, sizeof(p));
    p.g1 = g1->view; p.g2 = g2->view;
    p.weighted = g1->weighted;
    p.weight_in_lo = (g1->weighted && xyz) ? 1 : 0;
    // the w objects of one weighted point are w (w - 1) / 2 pairs at zero separation: cell (0 [, 0]) when the bins start at 0
    p.self_bin = (p.weighted && is_auto && bins->lo1 == 0.0 && !bins->log1 && (bins->n2 == 0 || bins->lo2 == 0.0)) ? 0 : -1;
    p.epoch_j = kEpochJ;
    if (p.weighted) {
        // a uint32 counter receives at most 128 increments of w1max*w2max per j-point; the epoch is checked once
        // per tile, so one tile of slack is kept (epoch 0 = flush after every tile)
        const uint64_t per_j = 128ull * g1->wmax * g2->wmax;
        const uint64_t e = 0xffffffffull / per_j;
        if (e < (uint64_t)kTile) return CUTE_ERR_OVERFLOW;            // w1max * w2max > 2^18
        p.epoch_j = (uint32_t)(e - kTile < kEpochJ ? e - kTile : kEpochJ);
    }
    p.kind = kind; p.is_auto = is_auto; p.mode = mode;
    p.periodic = (mode == CUTE_GRID_BOX3D && g1->spec.periodic) ? 1 : 0;
    p.logbins = bins->log1 ? 1 : 0;
    p.n1 = bins->n1; p.n2 = bins->n2; p.n2eff = bins->n2 > 0 ? bins->n2 : 1; p.nhist = p.n1 * p.n2eff;
    p.n2p = bins->n2 > 0 ? bins->n2 + 2 : 1; p.nhist_pad = (p.n1 + 2) * p.n2p;   // dump borders (pair_kernel.cuh)
    p.lo1 = bins->lo1; p.hi1 = bins->hi1; p.lo2 = bins->lo2; p.hi2 = bins->hi2;
    p.L = kind == CUTE_MONOPOLE ? bins->box_L : 0.0; p.aperture = bins->aperture_rad;
    p.Lf = (float)p.L;
    p.closed_top2 = (kind == CUTE_RMU && bins->hi2 >= 1.0);
    const double tau_scale = (opts && opts->tau_scale > 0.0) ? opts->tau_scale : 1.0;
    if ((rc = plan_fast_path(p, kind, g1, g2, bins, tau_scale))) return rc;
    if (opts && opts->force_refine) p.always_refine = 1;
    if (mode == CUTE_GRID_BOX3D) {
        const double rr = g1->spec.rmax;
        p.kx = (int)ceil(rr / g1->cell[0] * (1.0 - 1e-12));    // k = ceil(Rmax/a), reading G3; a pair this rounding could miss has r within 1e-12 of Rmax
        p.ky = (int)ceil(rr / g1->cell[1] * (1.0 - 1e-12));
        p.kz = (int)ceil(rr / g1->cell[2] * (1.0 - 1e-12));
        if (!p.periodic) { p.kx = p.kx < p.g2.ncx ? p.kx : p.g2.ncx; p.ky = p.ky < p.g2.ncy ? p.ky : p.g2.ncy; p.kz = p.kz < p.g2.ncz ? p.kz : p.g2.ncz; }
        p.ax = (float)g1->cell[0]; p.ay = (float)g1->cell[1]; p.az = (float)g1->cell[2];
        p.rmax2 = (float)(rr * rr * 1.001);
        p.ox = (float)g1->spec.origin[0]; p.inv_ax = (float)(1.0 / g1->cell[0]);
        // the trim is float32 arithmetic on float32 coordinates: cover its rounding (a few ulp of the largest |x|)
        p.trim_pad = (float)(16.0 * kU * (fmax(g1->maxabs, g2->maxabs) + fabs(g1->spec.origin[0]) + rr));
    }
    if (mode == CUTE_GRID_SPHERE) p.ring = g1->spec.size[0] >= 360.0 ? 1 : 0;

    unsigned char *sc = (unsigned char *)d_scratch;
    p.queue = (uint32_t *)(sc + SL.queue); p.status = (uint32_t *)(sc + SL.status);
    p.stats = (unsigned long long *)(sc + SL.stats);
    p.edges1 = (const double *)(sc + SL.edges1); p.edges2 = (const double *)(sc + SL.edges2);
    p.hist = (unsigned long long *)d_hist;
    std::vector<double> e((size_t)bins->n1 + 1 + (size_t)bins->n2 + 1);
    fill_edges(bins, 0, e.data());
    if (bins->n2 > 0) fill_edges(bins, 1, e.data() + bins->n1 + 1);
    if (!dry) {
        if (cudaMemsetAsync(sc, 0, 64, s) != cudaSuccess) return CUTE_ERR_CUDA;
        if (cudaMemcpyAsync(sc + SL.edges1, e.data(), e.size() * 8, cudaMemcpyHostToDevice, s) != cudaSuccess) return CUTE_ERR_CUDA;
        if (cudaMemsetAsync(d_hist, 0, (size_t)p.nhist * 8, s) != cudaSuccess) return CUTE_ERR_CUDA;
    }
    if (p.g1.n == 0 || p.g2.n == 0 || (is_auto && p.g1.n < 2)) { if (dry) *nitems_out = 0; return CUTE_OK; }   // N in {0,1}: zeros

    if (plan_pair_kernel(p, opts ? opts->warps : 0, opts ? opts->hist_cols : 0) < 0) return CUTE_ERR_UNSUPPORTED;
    if (p.hist_shared) {
        // all warps feed one counter, and each of them may overshoot its share by one tile before it checks
        if (p.weighted) {
            const uint64_t per_j = 128ull * g1->wmax * g2->wmax;
            const uint64_t e = 0x7fffffffull / per_j;   // (the shared copy is read as a signed 32-bit number: moved counts)
            if (e < (uint64_t)kTile * (uint64_t)p.warps + (uint64_t)p.warps) return CUTE_ERR_OVERFLOW;
            const uint64_t share = (e - (uint64_t)kTile * (uint64_t)p.warps) / (uint64_t)p.warps;
            p.epoch_j = (uint32_t)(share < (uint64_t)p.epoch_j ? share : (uint64_t)p.epoch_j);
        } else p.epoch_j = p.epoch_j / (uint32_t)p.warps > 0 ? p.epoch_j / (uint32_t)p.warps : 1u;
    }
    const int blocks = (opts && opts->blocks > 0) ? opts->blocks : sm_count();
    // work items: grid mode = chunks; brute force = chunks x j-splits, enough for ~16 items per warp
    uint64_t nitems = p.g1.nchunks;
    p.nsplit = 1; p.jsplit = p.g2.n;
    if (mode == CUTE_GRID_NONE) {
        const uint64_t target = 16ull * (uint64_t)blocks * p.warps;
        uint64_t ns = (target + nitems - 1) / nitems;
        const uint64_t max_ns = ((uint64_t)p.g2.n + kTile - 1) / kTile;
        ns = ns < 1 ? 1 : (ns > max_ns ? max_ns : ns);
        uint64_t js = ((uint64_t)p.g2.n + ns - 1) / ns;
        js = (js + kTile - 1) / kTile * kTile;
        if (js > (1u << 21)) js = 1u << 21;
        p.jsplit = (uint32_t)js;
        p.nsplit = (uint32_t)(((uint64_t)p.g2.n + js - 1) / js);
        nitems *= p.nsplit;
    }
    else {
        // cell lists: a chunk's neighbour rows are dealt to nsplit items (row nb goes to item nb % nsplit) when the
        // chunks alone would leave fewer than ~8 items per warp (sparse catalogues: C3 has 4088 chunks for 2368 warps)
        const uint64_t target = 8ull * (uint64_t)blocks * p.warps;
        int rows_nb = mode == CUTE_GRID_BOX3D ? (2 * p.ky + 1) * (2 * p.kz + 1) : 3;
        if (p.is_auto) rows_nb = (rows_nb + 1) / 2;
        uint64_t ns = nitems > 0 ? (target + nitems - 1) / nitems : 1;
        ns = ns < 1 ? 1 : (ns > (uint64_t)rows_nb ? (uint64_t)rows_nb : ns);
        p.nsplit = (uint32_t)ns;
        nitems *= p.nsplit;
    }
    if (nitems > 0xfffffff0ull) return CUTE_ERR_OVERFLOW;
    if (dry) { *nitems_out = (int64_t)nitems; return CUTE_OK; }
    p.item_begin = 0; p.item_end = (uint32_t)nitems;
    if (opts && (opts->shard || opts->item_begin || opts->item_end)) {
        if (opts->item_begin < 0 || opts->item_end < opts->item_begin) return CUTE_ERR_INVALID_ARG;
        p.item_begin = (uint32_t)(opts->item_begin < (int64_t)nitems ? opts->item_begin : (int64_t)nitems);
        p.item_end = (uint32_t)(opts->item_end < (int64_t)nitems ? opts->item_end : (int64_t)nitems);
    }
    p.flush_items = opts ? (uint32_t)opts->flush_items : 0u;
    if (launch_pair_kernel(p, blocks, s) != cudaSuccess) return CUTE_ERR_CUDA;
    return CUTE_OK;
}

int cute_count_pairs(int kind, const cute_grid *g1, const cute_grid *g2, const cute_bin_spec *bins, uint64_t *d_hist,
                     void *d_scratch, size_t scratch_bytes, const cute_count_opts *opts, void *stream)
{
    return count_impl(kind, g1, g2, bins, d_hist, d_scratch, scratch_bytes, opts, stream, nullptr);
}

int cute_count_items(int kind, const cute_grid *g1, const cute_grid *g2, const cute_bin_spec *bins, const cute_count_opts *opts,
                     int64_t *nitems)
{
    // number of work items cute_count_pairs enumerates for these arguments (for sharding with item_begin/item_end)
    if (!nitems) return CUTE_ERR_INVALID_ARG;
    return count_impl(kind, g1, g2, bins, nullptr, nullptr, 0, opts, nullptr, nitems);
}

int cute_shard_items(int64_t nitems, int64_t nchunks, int rank, int world, int auto_brute, int64_t *begin, int64_t *end)
{
    if (!begin || !end || nitems < 0 || nchunks < 0 || world < 1 || rank < 0 || rank >= world) return CUTE_ERR_INVALID_ARG;
    if (world == 1) { *begin = 0; *end = nitems; return CUTE_OK; }
    const int64_t nsplit = nchunks > 0 && nitems / nchunks > 0 ? nitems / nchunks : 1;
    auto cut = [&](int r) -> int64_t {
        if (r <= 0) return 0;
        if (r >= world) return nitems;
        const double f = (double)r / (double)world;
        const double x = auto_brute ? 1.0 - sqrt(fmax(0.0, 1.0 - f)) : f;
        int64_t c = (int64_t)llround(x * (double)nchunks) * nsplit;
        return c < 0 ? 0 : (c > nitems ? nitems : c);
    };
    *begin = cut(rank); *end = cut(rank + 1);
    if (*end < *begin) *end = *begin;
    return CUTE_OK;
}

int cute_auto_grid_spec(int kind, int mode, const cute_catalog *const *cats, int ncat, double rmax, double box_L,
                        double pix_frac, const int ncell[3], int no_perm, void *d_tmp, void *stream, cute_grid_spec *spec)
{
    if (!spec || !cats || ncat < 1 || ncat > 8 || kind < CUTE_ANGULAR || kind > CUTE_PISIGMA) return CUTE_ERR_INVALID_ARG;
    if (mode < CUTE_GRID_NONE || mode > CUTE_GRID_SPHERE) return CUTE_ERR_INVALID_ARG;
    memset(spec, 0, sizeof(*spec));
    spec->struct_size = sizeof(*spec);
    spec->mode = mode; spec->kind_mask = 1 << kind; spec->no_perm = no_perm;
    if (mode == CUTE_GRID_NONE) return CUTE_OK;
    if (!(rmax > 0.0)) return CUTE_ERR_INVALID_ARG;
    spec->rmax = rmax;
    if (ncell) for (int d = 0; d < 3; d++) spec->ncell[d] = ncell[d];
    if (mode == CUTE_GRID_BOX3D && box_L > 0.0) {
        spec->periodic = 1;
        for (int d = 0; d < 3; d++) spec->size[d] = box_L;
        return CUTE_OK;
    }
    // common bounding box of the raw coordinates
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    bool any = false;
    for (int k = 0; k < ncat; k++) {
        if (!cats[k]) return CUTE_ERR_INVALID_ARG;
        if (cats[k]->n == 0) continue;
        double b[6];
        int rc = cute_catalog_bounds(cats[k], d_tmp, stream, b);
        if (rc) return rc;
        for (int d = 0; d < 3; d++) { lo[d] = fmin(lo[d], b[d]); hi[d] = fmax(hi[d], b[3 + d]); }
        any = true;
    }
    if (!any) for (int d = 0; d < 3; d++) { lo[d] = 0.0; hi[d] = 1.0; }
    if (mode == CUTE_GRID_BOX3D) {
        for (int d = 0; d < 3; d++) {
            const double ext = hi[d] - lo[d];
            const double pad = 1e-6 * (ext > 1.0 ? ext : 1.0) + 1e-9 * fmax(fabs(lo[d]), fabs(hi[d]));
            spec->origin[d] = lo[d] - pad;
            spec->size[d] = ext + 2.0 * pad;
        }
        return CUTE_OK;
    }
    // SPHERE: pixels with constant limits in (RA, sin Dec); RA must not wrap inside the footprint
    if (!(pix_frac > 0.0)) pix_frac = 2.0;
    const double pix = pix_frac * rmax;                       // pixel side [rad]
    double dra = fmin(360.0, (hi[0] - lo[0]) * (1.0 + 1e-9) + 1e-9);
    if (dra > 180.0) dra = 360.0;                             // wide or seam-straddling footprint: pixels over the full ring
    const double ra0 = dra < 360.0 ? lo[0] - 0.5 * (dra - (hi[0] - lo[0])) : 0.0;
    const double u_lo = fmax(-1.0, sin(fmax(-90.0, lo[1]) * (kPi / 180.0)) - 1e-12);
    const double u_hi = fmin(1.0, sin(fmin(90.0, hi[1]) * (kPi / 180.0)) + 1e-12);
    const double du = fmax(u_hi - u_lo, 1e-12);
    const double dmin = (lo[1] * hi[1] > 0.0) ? fmin(fabs(lo[1]), fabs(hi[1])) : 0.0;   // the widest parallel of the footprint
    const double cmax = cos(dmin * (kPi / 180.0));
    double nra = floor(dra * (kPi / 180.0) * cmax / pix), nu = floor(du / pix);
    nra = nra < 1.0 ? 1.0 : (nra > 65535.0 ? 65535.0 : nra);
    nu = nu < 1.0 ? 1.0 : (nu > 1048576.0 ? 1048576.0 : nu);
    spec->origin[0] = ra0; spec->origin[1] = u_lo;
    spec->size[0] = dra; spec->size[1] = du;
    if (!(ncell && ncell[0] > 0 && ncell[1] > 0)) { spec->ncell[0] = (int)nra; spec->ncell[1] = (int)nu; }
    spec->ncell[2] = 1;
    return CUTE_OK;
}

int cute_count_status(void *d_scratch, void *stream, uint64_t stats[4])
{
    if (!d_scratch) return CUTE_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    unsigned char h[64];
    if (cudaMemcpyAsync(h, d_scratch, 64, cudaMemcpyDeviceToHost, s) != cudaSuccess) return CUTE_ERR_CUDA;
    if (cudaStreamSynchronize(s) != cudaSuccess) return CUTE_ERR_CUDA;
    if (stats) memcpy(stats, h + 32, 32);
    uint32_t st;
    memcpy(&st, h + 16, 4);
    if (st & 2u) return CUTE_ERR_OVERFLOW;
    if (st) return CUTE_ERR_CUDA;
    return CUTE_OK;
}

} // extern "C"

// =============================================================================== end-to-end with host buffers
namespace {

size_t cat_bytes(const cute_catalog *c)
{
    const size_t col = align_up((size_t)(c->n > 0 ? c->n : 1) * (c->dtype == CUTE_F64 ? 8 : 4), 256);
    return col * 3 + (c->weight ? align_up((size_t)(c->n > 0 ? c->n : 1) * 4, 256) : 0);
}

} // namespace

extern "C" {

int cute_host_workspace_bytes(const cute_catalog *cat1, const cute_catalog *cat2, const cute_grid_spec *spec,
                              const cute_bin_spec *bins, size_t *bytes)
{
    if (!bytes || !bins || bins->struct_size != sizeof(cute_bin_spec)) return CUTE_ERR_INVALID_ARG;
    size_t total = 0, w = 0;
    int rc = cute_grid_workspace_bytes(cat1, spec, &w);
    if (rc) return rc;
    total += align_up(w, 256) + cat_bytes(cat1);
    if (cat2) {
        if ((rc = cute_grid_workspace_bytes(cat2, spec, &w))) return rc;
        total += align_up(w, 256) + cat_bytes(cat2);
    }
    total += align_up((size_t)bins->n1 * (bins->n2 > 0 ? bins->n2 : 1) * 8, 256);
    total += scratch_layout(bins).total;
    *bytes = total;
    return CUTE_OK;
}

int cute_count_pairs_host(int kind, const cute_catalog *cat1, const cute_catalog *cat2, const cute_grid_spec *spec,
                          const cute_bin_spec *bins, const cute_count_opts *opts, uint64_t *h_hist, void *d_workspace,
                          size_t bytes, void *stream)
{
    size_t need = 0;
    int rc = cute_host_workspace_bytes(cat1, cat2, spec, bins, &need);
    if (rc) return rc;
    if (!h_hist || !d_workspace || ((uintptr_t)d_workspace & 255)) return CUTE_ERR_INVALID_ARG;
    if (bytes < need) return CUTE_ERR_WORKSPACE_TOO_SMALL;
    if ((rc = check_bins(kind, bins))) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    unsigned char *w = (unsigned char *)d_workspace;
    const cute_catalog *cats[2] = {cat1, cat2};
    cute_grid *grids[2] = {nullptr, nullptr};
    for (int k = 0; k < 2 && rc == CUTE_OK; k++) {
        const cute_catalog *c = cats[k];
        if (!c) break;
        cute_catalog dc = *c;
        const size_t esz = c->dtype == CUTE_F64 ? 8 : 4;
        const size_t col = align_up((size_t)(c->n > 0 ? c->n : 1) * esz, 256);
        const void *src[3] = {c->c0, c->c1, c->c2};
        const void **dst[3] = {&dc.c0, &dc.c1, &dc.c2};
        for (int d = 0; d < 3; d++) {
            *dst[d] = w + col * d;
            if (src[d] && c->n > 0 && cudaMemcpyAsync(w + col * d, src[d], (size_t)c->n * esz, cudaMemcpyHostToDevice, s) != cudaSuccess)
                rc = CUTE_ERR_CUDA;
            if (!src[d]) *dst[d] = nullptr;
        }
        w += col * 3;
        if (c->weight) {
            dc.weight = (const uint32_t *)w;
            if (c->n > 0 && cudaMemcpyAsync(w, c->weight, (size_t)c->n * 4, cudaMemcpyHostToDevice, s) != cudaSuccess) rc = CUTE_ERR_CUDA;
            w += align_up((size_t)(c->n > 0 ? c->n : 1) * 4, 256);
        }
        size_t gw = 0;
        if (rc == CUTE_OK) rc = cute_grid_workspace_bytes(c, spec, &gw);
        if (rc == CUTE_OK) rc = cute_make_grid(&dc, spec, w, gw, stream, &grids[k]);
        w += align_up(gw, 256);
    }
    if (rc == CUTE_OK) {
        const size_t nh = (size_t)bins->n1 * (bins->n2 > 0 ? bins->n2 : 1);
        uint64_t *d_hist = (uint64_t *)w;
        w += align_up(nh * 8, 256);
        const size_t sb = scratch_layout(bins).total;
        rc = cute_count_pairs(kind, grids[0], grids[1], bins, d_hist, w, sb, opts, stream);
        if (rc == CUTE_OK && cudaMemcpyAsync(h_hist, d_hist, nh * 8, cudaMemcpyDeviceToHost, s) != cudaSuccess) rc = CUTE_ERR_CUDA;
        if (rc == CUTE_OK) rc = cute_count_status(w, stream, nullptr);
    }
    cute_free_grid(grids[0]);
    cute_free_grid(grids[1]);
    return rc;
}

// =============================================================================== host-side estimators
/* Landy-Szalay, Eq. 15: xi = [Nr(Nr-1)/(Nd(Nd-1)) DD - (Nr-1)/Nd DR + RR] / RR with DD and RR
 * unordered pair counts and DR all Nd*Nr pairs. */
int cute_landy_szalay(const uint64_t *dd, const uint64_t *dr, const uint64_t *rr, uint64_t nd, uint64_t nr, int nbins, double *xi)
{
    if (!dd || !dr || !rr || !xi || nbins < 1 || nd < 2 || nr < 2) return CUTE_ERR_INVALID_ARG;
    const double Nd = (double)nd, Nr = (double)nr;
    const double wdd = Nr * (Nr - 1.0) / (Nd * (Nd - 1.0)), wdr = (Nr - 1.0) / Nd;
    int warn = CUTE_OK;
    for (int k = 0; k < nbins; k++) {
        if (rr[k] == 0) { xi[k] = 0.0; warn = CUTE_WARN_EMPTY_BIN; continue; }
        xi[k] = (wdd * (double)dd[k] - wdr * (double)dr[k] + (double)rr[k]) / (double)rr[k];
    }
    return warn;
}

/* natural estimator, Eq. 14: xi = Nr(Nr-1)/(Nd(Nd-1)) DD/RR - 1 */
int cute_natural_estimator(const uint64_t *dd, const uint64_t *rr, uint64_t nd, uint64_t nr, int nbins, double *xi)
{
    if (!dd || !rr || !xi || nbins < 1 || nd < 2 || nr < 2) return CUTE_ERR_INVALID_ARG;
    const double Nd = (double)nd, Nr = (double)nr;
    const double wdd = Nr * (Nr - 1.0) / (Nd * (Nd - 1.0));
    int warn = CUTE_OK;
    for (int k = 0; k < nbins; k++) {
        if (rr[k] == 0) { xi[k] = 0.0; warn = CUTE_WARN_EMPTY_BIN; continue; }
        xi[k] = wdd * (double)dd[k] / (double)rr[k] - 1.0;
    }
    return warn;
}

/* Multipoles, Eqs. 3-4; mid-point rule over the mu bins (reading M1) */
int cute_multipoles(const double *xi, int n_r, int n_mu, double *out)
{
    if (!xi || !out || n_r < 1 || n_mu < 1) return CUTE_ERR_INVALID_ARG;
    const double dmu = 1.0 / (double)n_mu;
    for (int k = 0; k < n_r; k++) {
        double s0 = 0.0, s2 = 0.0, s4 = 0.0;
        for (int m = 0; m < n_mu; m++) {
            const double mu = ((double)m + 0.5) * dmu, m2 = mu * mu, x = xi[(size_t)k * n_mu + m];
            s0 += x;
            s2 += x * (1.5 * m2 - 0.5);
            s4 += x * (4.375 * m2 * m2 - 3.75 * m2 + 0.375);
        }
        out[k] = s0 * dmu; out[n_r + k] = 5.0 * s2 * dmu; out[2 * n_r + k] = 9.0 * s4 * dmu;
    }
    return CUTE_OK;
}

/* Periodic box (Eqs. 12-13, with the exact shell volume and N(N-1)/2 unordered pairs) */
int cute_periodic_rr(uint64_t n, double L, const cute_bin_spec *bins, double *rr)
{
    if (!bins || bins->struct_size != sizeof(cute_bin_spec) || !rr || !(L > 0.0) || bins->n1 < 1 || !(bins->lo1 < bins->hi1)) return CUTE_ERR_INVALID_ARG;
    if (bins->log1 && !(bins->lo1 > 0.0)) return CUTE_ERR_INVALID_ARG;
    std::vector<double> e((size_t)bins->n1 + 1);
    fill_edges(bins, 0, e.data());
    const double np = 0.5 * (double)n * ((double)n - 1.0), v = L * L * L;
    for (int k = 0; k < bins->n1; k++) {
        const double a = e[k], b = e[k + 1];
        rr[k] = np * (4.0 * kPi / 3.0) * (b * b * b - a * a * a) / v;
    }
    return CUTE_OK;
}

int cute_periodic_xi(const uint64_t *dd, uint64_t n, double L, const cute_bin_spec *bins, double *xi)
{
    if (!dd || !xi) return CUTE_ERR_INVALID_ARG;
    int rc = cute_periodic_rr(n, L, bins, xi);
    if (rc) return rc;
    int warn = CUTE_OK;
    for (int k = 0; k < bins->n1; k++) {
        if (!(xi[k] > 0.0)) { xi[k] = 0.0; warn = CUTE_WARN_EMPTY_BIN; continue; }
        xi[k] = (double)dd[k] / xi[k] - 1.0;
    }
    return warn;
}

} // extern "C"
