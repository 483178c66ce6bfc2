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
// floor of a double in [-2^31, 2^31) without a conversion instruction: a round-down add of 2^52 + 2^51 leaves it in the
// low word (the float64 conversion / rounding instructions run at a fraction of the FP64 add rate)
__device__ __forceinline__ int floor_magic(double t) { return __double2loint(__dadd_rd(t, 6755399441055744.0)); }

// rare: a point on or outside a face of the box (or not finite): clamp its cell, say whether it is legal.
// Returns the cell id in the low word and "legal" in bit 32 (everything by value: nothing goes through local memory).
__device__ __noinline__ unsigned long long cell_fix_box(const BuildPlan &b, double a, double c1, double c2)
{
    const double v[3] = {a, c1, c2};
    int k[3];
    bool ok = true;
#pragma unroll
    for (int d = 0; d < 3; d++) {
        const double t = (v[d] - b.origin[d]) * b.inv_cell[d];
        int kk = floor_magic(t);
        // NaN / inf / far-away coordinates fail the magnitude test (their floor_magic is meaningless);
        // a point exactly on the upper face of a non-periodic box joins the last cell; so does a point of a periodic
        // box that lies below the upper face (in [0, L)) but whose product with 1/cell rounds up to nc
        const bool in = fabs(t) < 2147483648.0 && kk >= 0;
        if (!in || kk >= b.nc[d]) {
            const double off = v[d] - b.origin[d];
            if (!in || !(b.periodic ? off < b.size[d] : off <= b.size[d])) ok = false;
            kk = in ? b.nc[d] - 1 : 0;
        }
        k[d] = kk;
    }
    const uint32_t id = (uint32_t)((k[2] * b.nc[1] + k[1]) * b.nc[0] + k[0]);
    return (unsigned long long)id | (ok ? 1ull << 32 : 0ull);
}

template <int MODE>
__device__ __forceinline__ bool cell_of_t(const BuildPlan &b, double a, double c1, double c2, uint32_t &id)
{
    bool ok = true;
    int k[3] = {0, 0, 0};
    if (MODE == CUTE_GRID_BOX3D) {
        const double t0 = (a - b.origin[0]) * b.inv_cell[0], t1 = (c1 - b.origin[1]) * b.inv_cell[1], t2 = (c2 - b.origin[2]) * b.inv_cell[2];
        k[0] = floor_magic(t0); k[1] = floor_magic(t1); k[2] = floor_magic(t2);
        const bool fine = fabs(t0) < 2147483648.0 && fabs(t1) < 2147483648.0 && fabs(t2) < 2147483648.0 &&
                          (uint32_t)k[0] < (uint32_t)b.nc[0] && (uint32_t)k[1] < (uint32_t)b.nc[1] && (uint32_t)k[2] < (uint32_t)b.nc[2];
        if (!fine) {
            const unsigned long long r = cell_fix_box(b, a, c1, c2);
            id = (uint32_t)r;
            return (r >> 32) != 0;
        }
    } else if (MODE == CUTE_GRID_SPHERE) {
        double al = a - b.origin[0];
        al -= 360.0 * (double)floor_magic(al * (1.0 / 360.0));          // RA modulo 360 relative to RA0
        if (al < 0.0) al += 360.0;
        if (al >= 360.0) al -= 360.0;
        if (!(al >= 0.0) || !(al <= b.size[0]) || !(fabs(a) < 1.0e9) || !isfinite(c1) || !isfinite(c2)) ok = false;
        double t = al * b.inv_cell[0];
        k[0] = (t >= 0.0) ? (t < (double)b.nc[0] ? floor_magic(t) : b.nc[0] - 1) : 0;
        double u = sin(c1 * (kPi / 180.0)) - b.origin[1];
        if (!(u >= -1e-15) || !(u <= b.size[1] + 1e-15)) ok = false;
        t = u * b.inv_cell[1];
        k[1] = (t >= 0.0) ? (t < (double)b.nc[1] ? floor_magic(t) : b.nc[1] - 1) : 0;
    }
    id = (uint32_t)((k[2] * b.nc[1] + k[1]) * b.nc[0] + k[0]);
    return ok;
}

__device__ __forceinline__ bool cell_of(const BuildPlan &b, double a, double c1, double c2, uint32_t &id)
{
    if (b.mode == CUTE_GRID_BOX3D) return cell_of_t<CUTE_GRID_BOX3D>(b, a, c1, c2, id);
    if (b.mode == CUTE_GRID_SPHERE) return cell_of_t<CUTE_GRID_SPHERE>(b, a, c1, c2, id);
    id = 0;
    return true;
}

template <int DT>
__device__ __forceinline__ double load_coord_t(const void *p, int64_t i)
{
    return DT == CUTE_F64 ? reinterpret_cast<const double *>(p)[i] : (double)reinterpret_cast<const float *>(p)[i];
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
__device__ __forceinline__ void emit_point(const BuildPlan &b, uint32_t slot, double a, double c1, double c2, uint32_t i)
{
    // XYZ: w carries |x|^2 split hi/lo, so that the (r,mu) kernel gets s.l = |x_i|^2 - |x_j|^2 without
    // cancellation (l = x_i + x_j is the mid-point line of sight)
    double v[4] = {a, c1, c2, a * a + c1 * c1 + c2 * c2};
    if (b.coord != CUTE_COORD_XYZ) {
        double al = a * (kPi / 180.0), de = c1 * (kPi / 180.0), sa, ca, sd, cd;
        sincos(al, &sa, &ca);
        sincos(de, &sd, &cd);
        v[0] = cd * ca; v[1] = cd * sa; v[2] = sd; v[3] = c2;
    }
    float h[4], l[4];
    for (int d = 0; d < 4; d++) { h[d] = (float)v[d]; l[d] = (float)(v[d] - (double)h[d]); }
    if (b.weight) {   // integer weight: a bit pattern (the pair kernel multiplies integers) in hi.w, or, for xyz
                      // catalogues whose hi.w is |x|^2, in lo.x; RA/Dec: also as an exact double in p64
        const uint32_t w = b.weight[i];
        if (b.coord == CUTE_COORD_XYZ) l[0] = __uint_as_float(w);
        else { h[3] = __uint_as_float(w); l[3] = 0.f; v[3] = (double)w; }
        if (w == 0u || w > 65535u) atomicExch(&b.status[0], 1u);
        atomicMax(&b.status[2], w);
    }
    b.hi[slot] = make_float4(h[0], h[1], h[2], h[3]);
    if (b.want_lo) b.lo[slot] = make_float4(l[0], l[1], l[2], l[3]);
    if (b.want_f64) {   // one 32-byte record per point (two 16-byte stores into one sector; four separate arrays cost four)
        double2 *q = reinterpret_cast<double2 *>(b.p64) + 2 * (size_t)slot;
        q[0] = make_double2(v[0], v[1]); q[1] = make_double2(v[2], v[3]);
    }
    if (b.perm) b.perm[slot] = i;
}

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
        emit_point(b, slot[k], a[k], c1[k], c2[k], (uint32_t)i);
    }
}


// ---- large catalogues: two-level partition ------------------------------------------------------
// The one-pass build above gives every point a random 16-byte store and a returning L2 atomic; at 10^7
// points in random order that is half-used DRAM sectors and ~2x the algorithmic traffic (round-1 ncu).
// Here instead: (1) a coarse pass groups the raw records into <= 1024 BUCKETS of consecutive cells -- each
// CTA owns a contiguous slice of the input and, per bucket, a private output range found by a scan of the
// per-(bucket, CTA) counts, so its shared-memory cursors hand out consecutive slots and L2 sees every line
// filled before it is evicted; (2) one CTA per bucket counts, scans and scatters its few hundred cells
// entirely in shared memory and writes cell_start itself.  No global atomics, every DRAM sector whole.
struct Rec32 { double a, c1, c2; uint32_t idx, cell; };   // raw record of a float64 / RA-Dec catalogue (+ its cell)

template <int DT>
__device__ __forceinline__ void load_raw(const BuildPlan &b, uint32_t i, double &a, double &c1, double &c2)
{
    a = load_coord_t<DT>(b.c0, i); c1 = load_coord_t<DT>(b.c1, i);
    c2 = b.coord != CUTE_COORD_RADEC ? load_coord_t<DT>(b.c2, i) : 0.0;
}

template <int MODE, int DT>
__global__ void __launch_bounds__(512) k_part_hist(BuildPlan b)
{
    extern __shared__ uint32_t sh[];
    const int B = b.part_B, G = b.part_G, g = blockIdx.x;
    for (int k = threadIdx.x; k < B; k += blockDim.x) sh[k] = 0;
    __syncthreads();
    const uint32_t per = (uint32_t)((b.n + G - 1) / G), i0 = min((uint32_t)b.n, (uint32_t)g * per), i1 = min((uint32_t)b.n, i0 + per);
    const uint32_t T = blockDim.x, shift = (uint32_t)b.part_shift;
    bool bad = false;
    uint32_t base = i0;
    for (; base + T * kPts <= i1; base += T * kPts) {        // full trips: no bounds checks, all loads in flight first
        double a[kPts], c1[kPts], c2[kPts];
#pragma unroll
        for (int k = 0; k < kPts; k++) load_raw<DT>(b, base + threadIdx.x + (uint32_t)k * T, a[k], c1[k], c2[k]);
#pragma unroll
        for (int k = 0; k < kPts; k++) {
            uint32_t id;
            bad = !cell_of_t<MODE>(b, a[k], c1[k], c2[k], id) || bad;   // (not finite => not ok)
            atomicAdd(&sh[id >> shift], 1u);
        }
    }
    for (uint32_t i = base + threadIdx.x; i < i1; i += T) {
        double a, c1, c2;
        load_raw<DT>(b, i, a, c1, c2);
        uint32_t id;
        bad = !cell_of_t<MODE>(b, a, c1, c2, id) || bad;
        atomicAdd(&sh[id >> shift], 1u);
    }
    if (bad) atomicExch(&b.status[0], 1u);
    __syncthreads();
    for (int k = threadIdx.x; k < B; k += blockDim.x) b.part_table[(size_t)k * G + g] = sh[k];
}

template <bool F32REC>
__device__ __forceinline__ void store_rec(const BuildPlan &b, uint32_t slot, double a, double c1, double c2, uint32_t i, uint32_t id)
{
    if (F32REC) reinterpret_cast<float4 *>(b.part_tmp)[slot] = make_float4((float)a, (float)c1, (float)c2, __uint_as_float(i));
    else {
        Rec32 r; r.a = a; r.c1 = c1; r.c2 = c2; r.idx = i; r.cell = id;
        reinterpret_cast<Rec32 *>(b.part_tmp)[slot] = r;
    }
}

template <int MODE, int DT, bool F32REC>
__global__ void __launch_bounds__(512) k_part_scatter(BuildPlan b, const uint32_t *table_start)
{
    extern __shared__ uint32_t sh[];
    const int B = b.part_B, G = b.part_G, g = blockIdx.x;
    for (int k = threadIdx.x; k < B; k += blockDim.x) sh[k] = table_start[(size_t)k * G + g];
    __syncthreads();
    const uint32_t per = (uint32_t)((b.n + G - 1) / G), i0 = min((uint32_t)b.n, (uint32_t)g * per), i1 = min((uint32_t)b.n, i0 + per);
    const uint32_t T = blockDim.x, shift = (uint32_t)b.part_shift;
    uint32_t base = i0;
    for (; base + T * kPts <= i1; base += T * kPts) {
        double a[kPts], c1[kPts], c2[kPts];
#pragma unroll
        for (int k = 0; k < kPts; k++) load_raw<DT>(b, base + threadIdx.x + (uint32_t)k * T, a[k], c1[k], c2[k]);
#pragma unroll
        for (int k = 0; k < kPts; k++) {
            uint32_t id;
            cell_of_t<MODE>(b, a[k], c1[k], c2[k], id);
            store_rec<F32REC>(b, atomicAdd(&sh[id >> shift], 1u), a[k], c1[k], c2[k], base + threadIdx.x + (uint32_t)k * T, id);
        }
    }
    for (uint32_t i = base + threadIdx.x; i < i1; i += T) {
        double a, c1, c2;
        load_raw<DT>(b, i, a, c1, c2);
        uint32_t id;
        cell_of_t<MODE>(b, a, c1, c2, id);
        store_rec<F32REC>(b, atomicAdd(&sh[id >> shift], 1u), a, c1, c2, i, id);
    }
}

// 1-D TMA bulk copy global -> shared with an mbarrier (the bucket's records reach shared memory in one instruction,
// issued by one thread: per-thread loads of ~10 records each would expose their latency one after the other)
__device__ __forceinline__ void fine_stage_bulk(void *dst, const void *src, uint32_t bytes, unsigned long long *bar)
{
    const uint32_t b = (uint32_t)__cvta_generic_to_shared(bar), d = (uint32_t)__cvta_generic_to_shared(dst);
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(b) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(b), "r"(bytes) : "memory");
        const uint32_t piece = 1u << 16;                       // pieces of 64 KB
        for (uint32_t o = 0; o < bytes; o += piece) {
            const uint32_t n = bytes - o < piece ? bytes - o : piece;
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(d + o), "l"(reinterpret_cast<const unsigned char *>(src) + o), "r"(n), "r"(b) : "memory");
        }
    }
    __syncthreads();                                           // the barrier is initialised before anybody polls it
    uint32_t ok;
    do {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\nselp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(ok) : "r"(b) : "memory");
    } while (!ok);
}

template <bool F32REC>
__device__ __forceinline__ void load_rec(const BuildPlan &b, uint32_t s, double &a, double &c1, double &c2, uint32_t &idx, uint32_t &cell)
{
    if (F32REC) {   // float32 xyz: no room for the cell in 16 bytes, recomputed (three FP64 multiply-adds)
        const float4 r = reinterpret_cast<const float4 *>(b.part_tmp)[s];
        a = r.x; c1 = r.y; c2 = r.z; idx = __float_as_uint(r.w);
        cell_of_t<CUTE_GRID_BOX3D>(b, a, c1, c2, cell);
    } else {
        const Rec32 r = reinterpret_cast<const Rec32 *>(b.part_tmp)[s];
        a = r.a; c1 = r.c1; c2 = r.c2; idx = r.idx; cell = r.cell;
    }
}

// One CTA per bucket.  The bucket's records are staged in shared memory (one coalesced read from HBM), its cells
// counted and scanned there, and every record is then emitted to its final slot: scattered 16-byte stores, but inside a
// window of a few hundred KB that L2 holds until its lines are whole.  A bucket too large for shared memory (a very
// clustered catalogue) is swept twice from global memory instead (the second sweep hits L2).
template <bool F32REC>
__global__ void __launch_bounds__(1024) k_part_fine(BuildPlan b, const uint32_t *table_start, uint32_t cap)
{
    extern __shared__ __align__(16) unsigned char fsm[];
    __shared__ uint32_t wsum[32];
    const int bk = blockIdx.x, G = b.part_G, cpb = b.part_cpb;
    uint32_t *cnt = reinterpret_cast<uint32_t *>(fsm);          // [cpb] counts, then starts, then cursors
    unsigned char *stage = fsm + (((size_t)cpb * 4 + 15) & ~(size_t)15);
    const uint32_t bs = table_start[(size_t)bk * G], be = table_start[(size_t)(bk + 1) * G];
    const int64_t c0 = (int64_t)bk * cpb;
    const int nc = (int)min((int64_t)cpb, b.ncells - c0);
    const bool staged = be - bs <= cap;
    const uint32_t T = blockDim.x;
    for (int k = threadIdx.x; k < nc; k += T) cnt[k] = 0;
    __syncthreads();
    if (staged) {
        __shared__ unsigned long long stage_bar;
        if (F32REC) {
            if (be > bs) fine_stage_bulk(stage, reinterpret_cast<const float4 *>(b.part_tmp) + bs, (be - bs) * 16u, &stage_bar);
            const float4 *dst = reinterpret_cast<const float4 *>(stage);
            for (uint32_t s = threadIdx.x; s < be - bs; s += T) {
                const float4 r = dst[s];
                uint32_t id;
                cell_of_t<CUTE_GRID_BOX3D>(b, (double)r.x, (double)r.y, (double)r.z, id);
                atomicAdd(&cnt[id - (uint32_t)c0], 1u);
            }
        } else {
            if (be > bs) fine_stage_bulk(stage, reinterpret_cast<const Rec32 *>(b.part_tmp) + bs, (be - bs) * 32u, &stage_bar);
            const Rec32 *dst = reinterpret_cast<const Rec32 *>(stage);
            for (uint32_t s = threadIdx.x; s < be - bs; s += T) atomicAdd(&cnt[dst[s].cell - (uint32_t)c0], 1u);
        }
    } else {
        for (uint32_t s = bs + threadIdx.x; s < be; s += T) {
            double a, c1, c2; uint32_t idx, id;
            load_rec<F32REC>(b, s, a, c1, c2, idx, id);
            atomicAdd(&cnt[id - (uint32_t)c0], 1u);
        }
    }
    __syncthreads();
    // exclusive scan of cnt[0..nc): each thread owns a run of consecutive cells
    const int per = (nc + (int)T - 1) / (int)T;
    const int k0 = min(nc, (int)threadIdx.x * per), k1 = min(nc, k0 + per);
    uint32_t tsum = 0;
    for (int k = k0; k < k1; k++) tsum += cnt[k];
    uint32_t x = tsum;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) wsum[wid] = x;
    __syncthreads();
    if (wid == 0) {
        uint32_t v = lane < (int)(T >> 5) ? wsum[lane] : 0u;
        for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, v, o); if (lane >= o) v += y; }
        wsum[lane] = v;
    }
    __syncthreads();
    uint32_t run = (wid ? wsum[wid - 1] : 0u) + x - tsum;
    for (int k = k0; k < k1; k++) {
        const uint32_t c = cnt[k];
        cnt[k] = run;                                           // local start = cursor
        b.cell_start[c0 + k] = bs + run;
        run += c;
    }
    if (bk == (int)gridDim.x - 1 && threadIdx.x == 0) b.cell_start[b.ncells] = (uint32_t)b.n;
    __syncthreads();
    if (staged) {
        for (uint32_t s = threadIdx.x; s < be - bs; s += T) {
            double a, c1, c2; uint32_t idx, id;
            if (F32REC) {
                const float4 r = reinterpret_cast<const float4 *>(stage)[s];
                a = r.x; c1 = r.y; c2 = r.z; idx = __float_as_uint(r.w);
                cell_of_t<CUTE_GRID_BOX3D>(b, a, c1, c2, id);
            } else {
                const Rec32 r = reinterpret_cast<const Rec32 *>(stage)[s];
                a = r.a; c1 = r.c1; c2 = r.c2; idx = r.idx; id = r.cell;
            }
            emit_point(b, bs + atomicAdd(&cnt[id - (uint32_t)c0], 1u), a, c1, c2, idx);
        }
    } else {
        for (uint32_t s = bs + threadIdx.x; s < be; s += T) {   // second sweep: the bucket is L2-resident
            double a, c1, c2; uint32_t idx, id;
            load_rec<F32REC>(b, s, a, c1, c2, idx, id);
            emit_point(b, bs + atomicAdd(&cnt[id - (uint32_t)c0], 1u), a, c1, c2, idx);
        }
    }
}

static cudaError_t run_partition_build(const BuildPlan &b, cudaStream_t s)
{
    cudaError_t e;
    const bool f32rec = b.dtype == CUTE_F32 && b.coord == CUTE_COORD_XYZ;
    const size_t sh1 = (size_t)b.part_B * 4;
    uint32_t *table_start = b.part_table + (((size_t)b.part_B * b.part_G + 63) / 64 * 64 + 64);
    const bool box = b.mode == CUTE_GRID_BOX3D, f64 = b.dtype == CUTE_F64;
    if (box && f64) k_part_hist<CUTE_GRID_BOX3D, CUTE_F64><<<b.part_G, 512, sh1, s>>>(b);
    else if (box) k_part_hist<CUTE_GRID_BOX3D, CUTE_F32><<<b.part_G, 512, sh1, s>>>(b);
    else if (f64) k_part_hist<CUTE_GRID_SPHERE, CUTE_F64><<<b.part_G, 512, sh1, s>>>(b);
    else k_part_hist<CUTE_GRID_SPHERE, CUTE_F32><<<b.part_G, 512, sh1, s>>>(b);
    if ((e = exclusive_scan(b.part_table, (int64_t)b.part_B * b.part_G, table_start, b.scan_tmp, s)) != cudaSuccess) return e;
    // fine pass: shared memory = cell counters + staging for a bucket 1.5x the mean size (at least 64 KB, at most 200 KB)
    const size_t cnt_b = ((size_t)b.part_cpb * 4 + 15) & ~(size_t)15, rec_b = f32rec ? 16 : 32;
    size_t want = (size_t)(1.5 * (double)b.n / (double)b.part_B) * rec_b + 4096;
    want = want < 64 * 1024 ? 64 * 1024 : want;
    size_t sh2 = cnt_b + want;
    if (sh2 > 200 * 1024) sh2 = 200 * 1024;
    const uint32_t cap = sh2 > cnt_b ? (uint32_t)((sh2 - cnt_b) / rec_b) : 0u;
    if (f32rec) {
        if ((e = cudaFuncSetAttribute(k_part_fine<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh2)) != cudaSuccess) return e;
        k_part_scatter<CUTE_GRID_BOX3D, CUTE_F32, true><<<b.part_G, 512, sh1, s>>>(b, table_start);
        k_part_fine<true><<<b.part_B, 1024, sh2, s>>>(b, table_start, cap);
    } else {
        if ((e = cudaFuncSetAttribute(k_part_fine<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh2)) != cudaSuccess) return e;
        if (box && f64) k_part_scatter<CUTE_GRID_BOX3D, CUTE_F64, false><<<b.part_G, 512, sh1, s>>>(b, table_start);
        else if (box) k_part_scatter<CUTE_GRID_BOX3D, CUTE_F32, false><<<b.part_G, 512, sh1, s>>>(b, table_start);
        else if (f64) k_part_scatter<CUTE_GRID_SPHERE, CUTE_F64, false><<<b.part_G, 512, sh1, s>>>(b, table_start);
        else k_part_scatter<CUTE_GRID_SPHERE, CUTE_F32, false><<<b.part_G, 512, sh1, s>>>(b, table_start);
        k_part_fine<false><<<b.part_B, 1024, sh2, s>>>(b, table_start, cap);
    }
    note_launches(3);
    return cudaGetLastError();
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

// rows <= 4096 * 1024 / ... : the common case (C5: 1600 rows, C4: ~3700) in ONE block instead of four launches
__global__ void __launch_bounds__(1024) k_row_scan_small(BuildPlan b)
{
    __shared__ uint32_t sh[32];
    __shared__ uint32_t carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const bool one_row = (b.mode == CUTE_GRID_NONE || b.order_only);
    for (int64_t r0 = 0; r0 < b.nrows; r0 += blockDim.x) {
        const int64_t r = r0 + threadIdx.x;
        uint32_t v = 0;
        if (r < b.nrows) {
            const uint32_t n = one_row ? (uint32_t)b.n : b.cell_start[(r + 1) * b.nc[0]] - b.cell_start[r * b.nc[0]];
            v = (n + kChunk - 1) / kChunk;
        }
        uint32_t tot;
        const uint32_t e = block_excl_scan(v, &tot, sh);
        if (r < b.nrows) b.row_chunk_start[r] = e + carry;
        __syncthreads();
        if (threadIdx.x == 0) carry += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) b.row_chunk_start[b.nrows] = carry;
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
    if (b.mode != CUTE_GRID_NONE && b.part_cpb > 0 && b.n > 0) {
        if ((e = run_partition_build(b, s)) != cudaSuccess) return e;
    } else if (b.mode != CUTE_GRID_NONE) {
        if ((e = cudaMemsetAsync(b.count, 0, (size_t)(b.ncells + 1) * 4, s)) != cudaSuccess) return e;
        if (b.n > 0) { k_cellid<<<pblocks, T, 0, s>>>(b); note_launches(1); }
        if ((e = exclusive_scan(b.count, b.ncells, b.cell_start, b.scan_tmp, s)) != cudaSuccess) return e;
        // the counters become the per-cell write cursors of the scatter
        if ((e = cudaMemcpyAsync(b.count, b.cell_start, (size_t)b.ncells * 4, cudaMemcpyDeviceToDevice, s)) != cudaSuccess) return e;
    }
    if (b.n > 0 && !(b.mode != CUTE_GRID_NONE && b.part_cpb > 0)) { k_scatter<<<pblocks, T, 0, s>>>(b); note_launches(1); }
    if (b.nrows <= 65536) { k_row_scan_small<<<1, 1024, 0, s>>>(b); note_launches(1); }
    else {
        k_row_counts<<<(int)((b.nrows + T - 1) / T), T, 0, s>>>(b);
        note_launches(1);
        if ((e = exclusive_scan(b.row_nchunks, b.nrows, b.row_chunk_start, b.scan_tmp, s)) != cudaSuccess) return e;
    }
    uint32_t max_chunks = (uint32_t)(b.n / kChunk + b.nrows + 1);
    k_chunks<<<(max_chunks + T - 1) / T, T, 0, s>>>(b, max_chunks);
    if (b.mode == CUTE_GRID_SPHERE && !b.order_only) { k_sphere_rows<<<(b.nc[1] + T - 1) / T, T, 0, s>>>(b); note_launches(1); }
    note_launches(1);   // k_chunks
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
