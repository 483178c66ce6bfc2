// grid_build.cu -- cell-list build on the device ("a box encompassing the whole catalog
// is first determined and divided into cubical cells. To each cell we associate the positions of all
// the objects that fall inside it"; pixels on the sphere PAPER.md:208-215).
// Steps: canonicalise -> cell index + cell histogram -> exclusive scan ->
// scatter into cell-sorted float4 arrays -> chunk table (the work items of the pair kernel).
// HBM-bound, O(N).
#include "cute_internal.h"
#include <math.h>
#include <string.h>

namespace cute {

static constexpr double kPi = 3.14159265358979323846264338327950288;

__device__ __forceinline__ double load_coord(const void *p, int dtype, int64_t i)
{
    return dtype == CUTE_F64 ? reinterpret_cast<const double *>(p)[i] : (double)reinterpret_cast<const float *>(p)[i];
}

// ---- bounding box (only when the caller gives no box) ---------------------------------------
__global__ void k_bbox(BuildPlan b)
{
    __shared__ double smin[3][32], smax[3][32];
    double mn[3] = {1e300, 1e300, 1e300}, mx[3] = {-1e300, -1e300, -1e300};
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < b.n; i += (int64_t)gridDim.x * blockDim.x) {
        double v[3] = {load_coord(b.c0, b.dtype, i), load_coord(b.c1, b.dtype, i), load_coord(b.c2, b.dtype, i)};
        for (int d = 0; d < 3; d++) { mn[d] = fmin(mn[d], v[d]); mx[d] = fmax(mx[d], v[d]); }
    }
    for (int d = 0; d < 3; d++)
        for (int o = 16; o; o >>= 1) {
            mn[d] = fmin(mn[d], __shfl_xor_sync(0xffffffffu, mn[d], o));
            mx[d] = fmax(mx[d], __shfl_xor_sync(0xffffffffu, mx[d], o));
        }
    int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) for (int d = 0; d < 3; d++) { smin[d][w] = mn[d]; smax[d][w] = mx[d]; }
    __syncthreads();
    if (w == 0) {
        int nw = blockDim.x >> 5;
        for (int d = 0; d < 3; d++) {
            double a = l < nw ? smin[d][l] : 1e300, c = l < nw ? smax[d][l] : -1e300;
            for (int o = 16; o; o >>= 1) {
                a = fmin(a, __shfl_xor_sync(0xffffffffu, a, o));
                c = fmax(c, __shfl_xor_sync(0xffffffffu, c, o));
            }
            if (l == 0) {
                // ordered-integer atomics on the bit patterns (monotone map double -> int64)
                long long ia = __double_as_longlong(a), ic = __double_as_longlong(c);
                ia = ia < 0 ? (long long)(0x8000000000000000ull) - ia : ia;
                ic = ic < 0 ? (long long)(0x8000000000000000ull) - ic : ic;
                atomicMin(reinterpret_cast<long long *>(b.bbox) + d, ia);
                atomicMax(reinterpret_cast<long long *>(b.bbox) + 3 + d, ic);
            }
        }
    }
}

// The device holds the box as order-preserving int64 images of the doubles; decode on the host.
void decode_bbox(const long long raw[6], double out[6])
{
    for (int d = 0; d < 6; d++) {
        long long v = raw[d];
        v = v < 0 ? (long long)(0x8000000000000000ull) - v : v;
        memcpy(&out[d], &v, 8);
    }
}

cudaError_t run_bbox(const BuildPlan &b, cudaStream_t s)
{
    // minima start at 0x7f7f... (a huge positive image), maxima at 0x8080... (a huge negative one)
    cudaError_t e;
    if ((e = cudaMemsetAsync(b.bbox, 0x7f, 24, s)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(reinterpret_cast<char *>(b.bbox) + 24, 0x80, 24, s)) != cudaSuccess) return e;
    if (b.n > 0) {
        int blocks = (int)((b.n + 255) / 256);
        if (blocks > 148 * 8) blocks = 148 * 8;
        k_bbox<<<blocks, 256, 0, s>>>(b);
        note_launches(1);
    }
    return cudaGetLastError();
}

// ---- G1: cell index + cell histogram ---------------------------------------------------------
// BOX3D: c = floor((x - x0)/a) per axis, id = (cz*ncy + cy)*ncx + cx (x fastest, so a row of
// neighbours along x is one contiguous range of the sorted array).  SPHERE: pixels with constant
// limits in (sin dec, RA) -- the paper's "spherical cubes".
__device__ __forceinline__ bool cell_of(const BuildPlan &b, double a, double c1, double c2, uint32_t &id)
{
    bool ok = true;
    int k[3] = {0, 0, 0};
    if (b.mode == CUTE_GRID_BOX3D) {
        double v[3] = {a, c1, c2};
        for (int d = 0; d < 3; d++) {
            double t = floor((v[d] - b.origin[d]) * b.inv_cell[d]);
            if (!(t >= 0.0) || !(v[d] - b.origin[d] <= b.size[d]) || (b.periodic && !(v[d] < b.origin[d] + b.size[d]))) ok = false;
            int kk = (t >= 0.0) ? (t < (double)b.nc[d] ? (int)t : b.nc[d] - 1) : 0;
            k[d] = kk;
        }
    } else if (b.mode == CUTE_GRID_SPHERE) {
        double al = fmod(a - b.origin[0], 360.0);
        if (al < 0.0) al += 360.0;
        if (!(al >= 0.0) || !(al <= b.size[0])) ok = false;
        double t = floor(al * b.inv_cell[0]);
        k[0] = (t >= 0.0) ? (t < (double)b.nc[0] ? (int)t : b.nc[0] - 1) : 0;
        double u = sin(c1 * (kPi / 180.0)) - b.origin[1];
        if (!(u >= -1e-15) || !(u <= b.size[1] + 1e-15)) ok = false;
        t = floor(u * b.inv_cell[1]);
        k[1] = (t >= 0.0) ? (t < (double)b.nc[1] ? (int)t : b.nc[1] - 1) : 0;
    }
    id = (uint32_t)((k[2] * b.nc[1] + k[1]) * b.nc[0] + k[0]);
    return ok;
}

// kPts points per thread, loads issued before their uses: these kernels are bound by the latency of dependent
// scattered accesses (ncu: long_scoreboard), so memory-level parallelism per thread is what buys bandwidth.
constexpr int kPts = 4;

__global__ void __launch_bounds__(256) k_cellid(BuildPlan b)
{
    const int64_t base = (int64_t)blockIdx.x * (blockDim.x * kPts) + threadIdx.x;
    double a[kPts], c1[kPts], c2[kPts];
#pragma unroll
    for (int k = 0; k < kPts; k++) {
        const int64_t i = base + (int64_t)k * blockDim.x;
        a[k] = c1[k] = c2[k] = 0.0;
        if (i < b.n) {
            a[k] = load_coord(b.c0, b.dtype, i); c1[k] = load_coord(b.c1, b.dtype, i);
            if (b.coord != CUTE_COORD_RADEC) c2[k] = load_coord(b.c2, b.dtype, i);
        }
    }
    uint32_t id[kPts];
    bool bad = false;
#pragma unroll
    for (int k = 0; k < kPts; k++) {
        const bool ok = cell_of(b, a[k], c1[k], c2[k], id[k]);
        bad = bad || ((base + (int64_t)k * blockDim.x < b.n) && (!ok || !isfinite(a[k]) || !isfinite(c1[k]) || !isfinite(c2[k])));
    }
#pragma unroll
    for (int k = 0; k < kPts; k++)
        if (base + (int64_t)k * blockDim.x < b.n) atomicAdd(&b.count[id[k]], 1u);   // cell histogram (no return value: RED)
    if (bad) atomicExch(&b.status[0], 1u);
}

// ---- G2: exclusive scan (three launches; n <= 2^27 elements) ---------------------------------
constexpr int kScanBlock = 1024, kScanPer = 4, kScanChunk = kScanBlock * kScanPer;

__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t *total, uint32_t *sh)
{
    int l = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t x = v;
    for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (l >= o) x += y; }
    if (l == 31) sh[w] = x;
    __syncthreads();
    if (w == 0) {
        uint32_t s = sh[l];
        for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, s, o); if (l >= o) s += y; }
        sh[l] = s;
    }
    __syncthreads();
    uint32_t base = w ? sh[w - 1] : 0u;
    *total = sh[31];
    return base + x - v;
}

__global__ void __launch_bounds__(kScanBlock) k_scan_sums(const uint32_t *in, int64_t n, uint32_t *sums)
{
    __shared__ uint32_t sh[32];
    int64_t base = (int64_t)blockIdx.x * kScanChunk + threadIdx.x * kScanPer;
    uint32_t s = 0;
    for (int k = 0; k < kScanPer; k++) if (base + k < n) s += in[base + k];
    uint32_t tot;
    block_excl_scan(s, &tot, sh);
    if (threadIdx.x == 0) sums[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(kScanBlock) k_scan_top(uint32_t *sums, int nb)
{
    __shared__ uint32_t sh[32];
    __shared__ uint32_t carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int b0 = 0; b0 < nb; b0 += kScanBlock) {
        int i = b0 + threadIdx.x;
        uint32_t v = i < nb ? sums[i] : 0u, tot;
        uint32_t e = block_excl_scan(v, &tot, sh);
        if (i < nb) sums[i] = e + carry;
        __syncthreads();
        if (threadIdx.x == 0) carry += tot;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(kScanBlock) k_scan_final(const uint32_t *in, int64_t n, const uint32_t *sums, uint32_t *out)
{
    __shared__ uint32_t sh[32];
    int64_t base = (int64_t)blockIdx.x * kScanChunk + threadIdx.x * kScanPer;
    uint32_t v[kScanPer], s = 0;
    for (int k = 0; k < kScanPer; k++) { v[k] = (base + k < n) ? in[base + k] : 0u; s += v[k]; }
    uint32_t tot;
    uint32_t e = block_excl_scan(s, &tot, sh) + sums[blockIdx.x];
    for (int k = 0; k < kScanPer; k++) { if (base + k < n) out[base + k] = e; e += v[k]; }
    // out[n] = grand total: after the loop e holds it in the thread that owns element n-1
    if (base <= n - 1 && n - 1 < base + kScanPer) out[n] = e;
}

static cudaError_t exclusive_scan(const uint32_t *in, int64_t n, uint32_t *out, uint32_t *tmp, cudaStream_t s)
{
    // out has n+1 entries; tmp has ceil(n/kScanChunk) entries
    if (n <= 0) return cudaMemsetAsync(out, 0, 4, s);
    int nb = (int)((n + kScanChunk - 1) / kScanChunk);
    k_scan_sums<<<nb, kScanBlock, 0, s>>>(in, n, tmp);
    k_scan_top<<<1, kScanBlock, 0, s>>>(tmp, nb);
    k_scan_final<<<nb, kScanBlock, 0, s>>>(in, n, tmp, out);
    note_launches(3);
    return cudaGetLastError();
}

// ---- G0 + G3: canonicalise and scatter into cell-sorted arrays --------------------------------
// XYZ: hi = float32(x), lo = float32(x - hi).  RA/Dec: unit vector n = (cos d cos a, cos d sin a,
// sin d) in float64 ("projects all objects in the catalog into the unit sphere"),
// then the same hi/lo split; w carries float32(z) for RADECZ.  p64 keeps the float64 values for
// the refine path.
__global__ void __launch_bounds__(256) k_scatter(BuildPlan b)
{
    const int64_t base = (int64_t)blockIdx.x * (blockDim.x * kPts) + threadIdx.x;
    double a[kPts], c1[kPts], c2[kPts];
    uint32_t slot[kPts];
#pragma unroll
    for (int k = 0; k < kPts; k++) {
        const int64_t i = base + (int64_t)k * blockDim.x;
        a[k] = c1[k] = c2[k] = 0.0;
        slot[k] = 0;
        if (i < b.n) {
            a[k] = load_coord(b.c0, b.dtype, i); c1[k] = load_coord(b.c1, b.dtype, i);
            if (b.coord != CUTE_COORD_RADEC) c2[k] = load_coord(b.c2, b.dtype, i);
            slot[k] = (uint32_t)i;
        }
    }
    if (b.mode != CUTE_GRID_NONE) {
        // slot = the cell's cursor (a copy of cell_start kept in `count`), advanced atomically: the order inside a
        // cell is arbitrary and the histogram must not depend on it (pin V4).  The cell id is recomputed from the
        // coordinates already in registers instead of being cached in HBM.
#pragma unroll
        for (int k = 0; k < kPts; k++) {
            const int64_t i = base + (int64_t)k * blockDim.x;
            uint32_t id;
            cell_of(b, a[k], c1[k], c2[k], id);
            if (i < b.n) slot[k] = atomicAdd(&b.count[id], 1u);
        }
    }
#pragma unroll
    for (int k = 0; k < kPts; k++) {
        const int64_t i = base + (int64_t)k * blockDim.x;
        if (i >= b.n) continue;
        // XYZ: w carries |x|^2 split hi/lo, so that the (r,mu) kernel gets s.l = |x_i|^2 - |x_j|^2 without
        // cancellation (l = x_i + x_j is the mid-point line of sight)
        double v[4] = {a[k], c1[k], c2[k], a[k] * a[k] + c1[k] * c1[k] + c2[k] * c2[k]};
        if (b.coord != CUTE_COORD_XYZ) {
            double al = a[k] * (kPi / 180.0), de = c1[k] * (kPi / 180.0), sa, ca, sd, cd;
            sincos(al, &sa, &ca);
            sincos(de, &sd, &cd);
            v[0] = cd * ca; v[1] = cd * sa; v[2] = sd; v[3] = c2[k];
        }
        float h[4], l[4];
        for (int d = 0; d < 4; d++) { h[d] = (float)v[d]; l[d] = (float)(v[d] - (double)h[d]); }
        if (b.weight) {   // integer weight: bit pattern in hi.w (the pair kernel multiplies integers), exact double in p64
            const uint32_t w = b.weight[i];
            h[3] = __uint_as_float(w); l[3] = 0.f; v[3] = (double)w;
            if (w == 0u || w > 65535u) atomicExch(&b.status[0], 1u);
            atomicMax(&b.status[2], w);
        }
        b.hi[slot[k]] = make_float4(h[0], h[1], h[2], h[3]);
        if (b.want_lo) b.lo[slot[k]] = make_float4(l[0], l[1], l[2], l[3]);
        if (b.want_f64) for (int d = 0; d < 4; d++) b.p64[(size_t)d * b.n_pad + slot[k]] = v[d];
        if (b.perm) b.perm[slot[k]] = (uint32_t)i;
    }
}

// ---- G4: chunk table ---------------------------------------------------------------------------
__global__ void k_row_counts(BuildPlan b)
{
    int64_t r = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (r >= b.nrows) return;
    uint32_t n = (b.mode == CUTE_GRID_NONE || b.order_only) ? (uint32_t)b.n
                                              : b.cell_start[(r + 1) * b.nc[0]] - b.cell_start[r * b.nc[0]];
    b.row_nchunks[r] = (n + kChunk - 1) / kChunk;
}

__global__ void k_chunks(BuildPlan b, uint32_t max_chunks)
{
    uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t total = b.row_chunk_start[b.nrows];
    if (c == 0) b.status[1] = total;
    if (c >= total || c >= max_chunks) return;
    // binary search: last row with row_chunk_start[row] <= c
    int64_t lo = 0, hi = b.nrows - 1;
    while (lo < hi) { int64_t m = (lo + hi + 1) >> 1; if (b.row_chunk_start[m] <= c) lo = m; else hi = m - 1; }
    uint32_t row = (uint32_t)lo, k = c - b.row_chunk_start[row];
    const bool one_row = (b.mode == CUTE_GRID_NONE || b.order_only);
    uint32_t r0 = one_row ? 0u : b.cell_start[(int64_t)row * b.nc[0]];
    uint32_t r1 = one_row ? (uint32_t)b.n : b.cell_start[((int64_t)row + 1) * b.nc[0]];
    Chunk ch;
    ch.i_begin = r0 + k * kChunk;
    ch.i_count = min((uint32_t)kChunk, r1 - ch.i_begin);
    ch.row = row;
    uint32_t cx0 = 0, cx1 = 0;
    if (!one_row) {
        // cell (along x) of a sorted index = last cell of the row whose start is <= the index
        const uint32_t *cs = b.cell_start + (int64_t)row * b.nc[0];
        auto cell_of_index = [&](uint32_t idx) {
            uint32_t lo = 0, hi = (uint32_t)b.nc[0] - 1;
            while (lo < hi) { uint32_t m = (lo + hi + 1) >> 1; if (cs[m] <= idx) lo = m; else hi = m - 1; }
            return lo;
        };
        cx0 = cell_of_index(ch.i_begin);
        cx1 = cell_of_index(ch.i_begin + ch.i_count - 1);
    }
    ch.cx01 = cx0 | (cx1 << 16);
    b.chunks[c] = ch;
}

// SPHERE: per-row search windows from the repaired Eq. 16 (reading G2):
// a cap of radius tmax about a point of declination d spans |d RA| <= asin(sin tmax / cos d) and
// declinations [d - tmax, d + tmax]; for a pixel row take the worst case over the row.
__global__ void k_sphere_rows(BuildPlan b)
{
    int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= b.nc[1]) return;
    double du = b.size[1] / b.nc[1];
    double u0 = fmin(1.0, fmax(-1.0, b.origin[1] + r * du)), u1 = fmin(1.0, fmax(-1.0, b.origin[1] + (r + 1) * du));
    double d0 = asin(u0), d1 = asin(u1), tm = b.thetamax * (1.0 + 1e-9) + 1e-15;
    double dworst = fmax(fabs(d0), fabs(d1));
    int kx;
    if (dworst + tm >= 0.5 * kPi * (1.0 - 1e-9)) kx = b.nc[0];
    else {
        double w = asin(fmin(1.0, sin(tm) / cos(dworst))) * (180.0 / kPi);   // degrees of RA
        double k = ceil(w * b.inv_cell[0] * (1.0 + 1e-9)) + 1.0;
        kx = k < (double)b.nc[0] ? (int)k : b.nc[0];
    }
    b.row_kx[r] = kx;
    double ulo = sin(fmax(-0.5 * kPi, d0 - tm)), uhi = sin(fmin(0.5 * kPi, d1 + tm));
    int ylo = (int)floor((ulo - b.origin[1]) * b.inv_cell[1]) - 1, yhi = (int)floor((uhi - b.origin[1]) * b.inv_cell[1]) + 1;
    b.row_ylo[r] = max(0, min(ylo, r));
    b.row_yhi[r] = min(b.nc[1] - 1, max(yhi, r));
}

cudaError_t run_build(const BuildPlan &b, cudaStream_t s)
{
    cudaError_t e;
    const int T = 256;
    const int pblocks = (int)((b.n + (int64_t)T * kPts - 1) / ((int64_t)T * kPts));
    if ((e = cudaMemsetAsync(b.status, 0, 12, s)) != cudaSuccess) return e;
    if (b.mode != CUTE_GRID_NONE) {
        if ((e = cudaMemsetAsync(b.count, 0, (size_t)(b.ncells + 1) * 4, s)) != cudaSuccess) return e;
        if (b.n > 0) { k_cellid<<<pblocks, T, 0, s>>>(b); note_launches(1); }
        if ((e = exclusive_scan(b.count, b.ncells, b.cell_start, b.scan_tmp, s)) != cudaSuccess) return e;
        // the counters become the per-cell write cursors of the scatter
        if ((e = cudaMemcpyAsync(b.count, b.cell_start, (size_t)b.ncells * 4, cudaMemcpyDeviceToDevice, s)) != cudaSuccess) return e;
    }
    if (b.n > 0) { k_scatter<<<pblocks, T, 0, s>>>(b); note_launches(1); }
    k_row_counts<<<(int)((b.nrows + T - 1) / T), T, 0, s>>>(b);
    if ((e = exclusive_scan(b.row_nchunks, b.nrows, b.row_chunk_start, b.scan_tmp, s)) != cudaSuccess) return e;
    uint32_t max_chunks = (uint32_t)(b.n / kChunk + b.nrows + 1);
    k_chunks<<<(max_chunks + T - 1) / T, T, 0, s>>>(b, max_chunks);
    if (b.mode == CUTE_GRID_SPHERE && !b.order_only) { k_sphere_rows<<<(b.nc[1] + T - 1) / T, T, 0, s>>>(b); note_launches(1); }
    note_launches(2);   // k_row_counts, k_chunks
    return cudaGetLastError();
}

// ---- pixel map: count per pixel, compact the non-empty pixels, emit their centres ----------
__global__ void k_pix_count(BuildPlan b, uint32_t *count)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= b.n) return;
    double a = load_coord(b.c0, b.dtype, i), c1 = load_coord(b.c1, b.dtype, i);
    uint32_t id;
    bool ok = cell_of(b, a, c1, 0.0, id);
    if (!ok || !isfinite(a) || !isfinite(c1)) { atomicExch(&b.status[0], 1u); return; }
    atomicAdd(&count[id], 1u);
}

__global__ void k_pix_flag(const uint32_t *count, int64_t n, uint32_t *flag)
{
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p < n) flag[p] = count[p] ? 1u : 0u;
}

__global__ void k_pix_emit(BuildPlan b, const uint32_t *count, const uint32_t *pos, double *pra, double *pdec, uint32_t *pw)
{
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= b.ncells || !count[p]) return;
    const int kx = (int)(p % b.nc[0]), ky = (int)(p / b.nc[0]);
    // a pixel is represented by its centre in (RA, sin Dec)  (reading P1)
    const double r = b.origin[0] + ((double)kx + 0.5) * (b.size[0] / (double)b.nc[0]);
    double u = b.origin[1] + ((double)ky + 0.5) * (b.size[1] / (double)b.nc[1]);
    u = fmin(1.0, fmax(-1.0, u));
    const uint32_t m = pos[p];
    pra[m] = fmod(r, 360.0);
    pdec[m] = asin(u) * (180.0 / kPi);
    pw[m] = count[p];
}

cudaError_t run_pixelize(const BuildPlan &b, uint32_t *count, uint32_t *pos, uint32_t *scan_tmp, double *pra, double *pdec,
                         uint32_t *pw, cudaStream_t s)
{
    cudaError_t e;
    const int T = 256;
    if ((e = cudaMemsetAsync(b.status, 0, 12, s)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(count, 0, (size_t)b.ncells * 4, s)) != cudaSuccess) return e;
    if (b.n > 0) { k_pix_count<<<(int)((b.n + T - 1) / T), T, 0, s>>>(b, count); note_launches(1); }
    const int pb = (int)((b.ncells + T - 1) / T);
    k_pix_flag<<<pb, T, 0, s>>>(count, b.ncells, pos);
    // in-place exclusive scan of the flags: pos[p] = output slot, pos[ncells] = number of non-empty pixels
    if ((e = exclusive_scan(pos, b.ncells, pos, scan_tmp, s)) != cudaSuccess) return e;
    k_pix_emit<<<pb, T, 0, s>>>(b, count, pos, pra, pdec, pw);
    note_launches(2);
    return cudaGetLastError();
}

} // namespace cute
