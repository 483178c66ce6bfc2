// density_grid.cu -- the density-grid monopole of CUTE_box:
// "the particle content of the catalog is first interpolated to a grid and the overdensity field delta is
// estimated at every grid point using a TSC algorithm.  Then pairs of grid points are correlated, and a weight
// delta_i delta_j is given to each pair.  The correlation function is estimated as
//        xi(r) = < delta(x) delta(x + r) >                                                        (Eq. 17)
// ... since the relative distances between neighboring points are the same everywhere, these relative
// distances only have to be calculated once."
// Readings D1-D4: grid points = cell centres (g + 1/2) h; TSC = second-order B-spline per axis;
// delta = rho / (N / ng^3) - 1; every ordered pair (g, g + v), v != 0 with the minimum image, r = h |v|, half-open bins.
// Three kernels: TSC scatter (float64 atomics into the L2-resident grid, three lanes per particle; bound by the L2 atomic units),
// overdensity (elementwise), and the offset-stencil correlation.  The offsets are found and binned ONCE on the host.
// k_grid_corr_rows (offsets of at most 16 cells per axis) treats each (vy, vz) as a 1-D cross-correlation of x-rows for all
// vx at once, register-tiled, rows staged in shared memory by cp.async, half of the offsets swept (xi is even);
// k_grid_corr (anything else) gives every thread one grid point and sweeps the offsets of a bin.
// All arithmetic float64 (the grid fits L2; this path is not the float32 pair kernel), so the result differs from a
// serial float64 loop only by the order of the additions.
#include "cute_internal.h"
#include <math.h>
#include <vector>
#include <algorithm>

namespace cute {

// SMs of the current device (grid sizing only)
static int dg_sm_count()
{
    static int n = 0;
    if (!n) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    }
    return n;
}

__device__ __forceinline__ double tsc_weight(double s)
{
    s = fabs(s);
    if (s <= 0.5) return 0.75 - s * s;
    if (s <= 1.5) return 0.5 * (1.5 - s) * (1.5 - s);
    return 0.0;
}

__device__ __forceinline__ int wrap(int g, int ng)
{
    g %= ng;
    return g < 0 ? g + ng : g;
}

// TSC scatter with THREE lanes per particle, one per x-offset: the three grid points a particle feeds along x are
// adjacent doubles, so a warp instruction carries 10 particles x 3 adjacent addresses = 10-20 sectors to the L2 atomic
// units instead of 32 scattered ones (the scatter is bound by those units, not by HBM; measured on 10^7 particles and a
// 128^3 grid: 1.16 ms with one thread per particle and 27 scattered atomics each, 0.76 ms this way).
__global__ void __launch_bounds__(256) k_tsc3(const void *x, const void *y, const void *z, int dtype, int64_t n, double inv_h, int ng,
                                              double *rho, uint32_t *status)
{
    const int lane = threadIdx.x & 31, pl = lane / 3, xo = lane - 3 * pl;
    const int64_t nwarps = (int64_t)gridDim.x * (blockDim.x >> 5), wg = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    for (int64_t i0 = wg * 10; i0 < n; i0 += nwarps * 10) {
        const int64_t i = i0 + pl;
        if (lane >= 30 || i >= n) continue;
        double p[3];
        if (dtype == CUTE_F64) {
            p[0] = reinterpret_cast<const double *>(x)[i]; p[1] = reinterpret_cast<const double *>(y)[i]; p[2] = reinterpret_cast<const double *>(z)[i];
        } else {
            p[0] = reinterpret_cast<const float *>(x)[i]; p[1] = reinterpret_cast<const float *>(y)[i]; p[2] = reinterpret_cast<const float *>(z)[i];
        }
        int g0[3];
        double w[3][3];
        bool bad = false;
#pragma unroll
        for (int d = 0; d < 3; d++) {
            const double u = p[d] * inv_h;                  // position in units of cells
            if (!(fabs(u) < 1.0e9)) bad = true;
            const double c = floor(u);                      // the particle's own cell
            g0[d] = bad ? 0 : (int)c - 1;
#pragma unroll
            for (int k = 0; k < 3; k++) w[d][k] = tsc_weight(u - (c - 1.0 + (double)k + 0.5));
        }
        if (bad) { atomicExch(status, 1u); continue; }
        const int gx = wrap(g0[0] + xo, ng);
        const double wx = xo == 0 ? w[0][0] : (xo == 1 ? w[0][1] : w[0][2]);
        int gy[3], gz[3];
#pragma unroll
        for (int k = 0; k < 3; k++) { gy[k] = wrap(g0[1] + k, ng); gz[k] = wrap(g0[2] + k, ng); }
#pragma unroll
        for (int a = 0; a < 3; a++)
#pragma unroll
            for (int b = 0; b < 3; b++) atomicAdd(&rho[((size_t)gz[a] * ng + gy[b]) * ng + gx], wx * w[1][b] * w[2][a]);
    }
}

__global__ void k_overdensity(double *rho, int64_t ng3, double inv_mean)
{
    const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (c < ng3) rho[c] = rho[c] * inv_mean - 1.0;
}

// one thread per grid point, offsets sorted by bin: {dx, dy, dz, bin}
constexpr int kCorrThreads = 256;
__global__ void __launch_bounds__(kCorrThreads) k_grid_corr(const double *__restrict__ delta, int ng, const int4 *__restrict__ offs,
                                                            const uint32_t *__restrict__ bin_start, int nbins, double *sum_dd)
{
    __shared__ double red[kCorrThreads / 32];
    const int64_t ng3 = (int64_t)ng * ng * ng;
    const int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const bool live = g < ng3;
    const int gx = live ? (int)(g % ng) : 0, gy = live ? (int)((g / ng) % ng) : 0, gz = live ? (int)(g / ((int64_t)ng * ng)) : 0;
    const double d0 = live ? delta[g] : 0.0;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int k = 0; k < nbins; k++) {
        const uint32_t o0 = bin_start[k], o1 = bin_start[k + 1];
        if (o0 == o1) continue;
        double acc = 0.0;
        for (uint32_t o = o0; o < o1; o++) {
            const int4 v = offs[o];                      // uniform over the block: one broadcast load
            int hx = gx + v.x, hy = gy + v.y, hz = gz + v.z;
            hx += hx < 0 ? ng : (hx >= ng ? -ng : 0);    // |v| < ng / 2: one wrap at most
            hy += hy < 0 ? ng : (hy >= ng ? -ng : 0);
            hz += hz < 0 ? ng : (hz >= ng ? -ng : 0);
            acc = fma(d0, delta[((size_t)hz * ng + hy) * ng + hx], acc);
        }
        for (int s = 16; s; s >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, s);
        if (lane == 0) red[wid] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = 0.0;
            for (int w = 0; w < kCorrThreads / 32; w++) t += red[w];
            atomicAdd(&sum_dd[k], t);
        }
        __syncthreads();
    }
}

// The fast stencil (offsets of at most 16 cells per axis).  xi(v) = <delta(g) delta(g + v)> is even in v, so only the
// half-space vz > 0 | (vz = 0, vy > 0) | (vz = vy = 0, vx > 0) is swept and every sum counts twice.  A CTA owns one
// (vy, vz) and a slab of z; a group of LPR lanes takes one x-row A = delta[gz][gy][.] and the shifted row
// B = delta[gz+vz][gy+vy][.] at a time: B goes to shared memory with a circular halo of M cells, each lane keeps XT = 8
// consecutive points of A in registers, reads its window of 8 + 2M points of B once (LDS.128) and feeds 8 (2M + 1) float64
// multiply-adds into 2M + 1 register accumulators, one per vx -- a 1-D cross-correlation of the two rows for all lags at
// once.  Row pairs reach shared memory by cp.async, three of them in flight per lane group while one is computed.
constexpr int kXT = 8, kStagesDG = 4;
template <int M>
__global__ void __launch_bounds__(256, 1) k_grid_corr_rows(const double *__restrict__ delta, int ng, int m, const int2 *__restrict__ vyz,
                                                           int zsplit, const int *__restrict__ binidx, double *sum_dd, int lpr_log2)
{
    constexpr int W = 2 * M + 1, WIN = kXT + 2 * M;
    extern __shared__ __align__(16) double rows_sm[];
    __shared__ double red[8][W];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int2 v = vyz[blockIdx.x / zsplit];
    const int zs = blockIdx.x % zsplit;
    const int zper = (ng + zsplit - 1) / zsplit, z0 = min(ng, zs * zper), z1 = min(ng, z0 + zper);
    const int r0 = z0 * ng, r1 = z1 * ng;                  // rows (gz * ng + gy) of this slab
    double acc[W];
#pragma unroll
    for (int k = 0; k < W; k++) acc[k] = 0.0;
    auto stage_index = [&](int i) {                        // staged row: buf[i] = B[(i - M) mod ng]
        int x = (i - M) % ng;
        return x < 0 ? x + ng : x;
    };

    if (lpr_log2 >= 0) {
        // ---- LPR lanes per row (kXT * LPR >= ng, ng a multiple of kXT), 32 / LPR rows per warp and trip:
        //      register-resident, software-pipelined, no guards in the loop
        const int LPR = 1 << lpr_log2, RPW = 32 >> lpr_log2;
        const int sub = lane >> lpr_log2, lr = lane & (LPR - 1);
        const int blen = ng + 2 * M;                       // (even: 16-byte aligned rows)
        // 16-byte pieces are stored swizzled inside aligned groups of 8 (piece p at p ^ ((p >> 3) & 3)): the lanes of a
        // quarter-warp read pieces 4 apart, which would otherwise share two bank groups (4-way conflicts, measured).  This
        // mask makes the eight reads p = 4 lane + j conflict-free for every j (checked by enumeration; & 7 left half of them
        // 2-way), and keeps eight consecutive pieces -- what a copy instruction writes -- on eight bank groups.
        auto swz = [](int p) { return p ^ ((p >> 3) & 3); };
        const int blen_pad = (blen + 15) & ~15, slot = blen_pad + ((ng + 15) & ~15);   // one staged row pair: B with its halo, then A
        // B is staged in 16-byte pieces (M and ng are even, so a pair of slots never straddles the wrap): per lane
        // ceil((ng + 2M) / 2 / LPR) <= kXT / 2 + ceil(M / 8) of them
        constexpr int NST = kXT / 2 + (M + 7) / 8;
        // The lanes of a row group copy CONSECUTIVE pieces (lr, lr + LPR, ...) of B and of A: a cp.async writes shared memory
        // one wavefront per global line it receives, so lanes 64 bytes apart in global memory (each copying its own 8
        // points of A) cost 4x the wavefronts (measured); a piece past the end is not copied at all.
        int xs[NST], xg[NST];                              // first slot of each piece this lane fills, and the x of B it holds
        uint32_t bmask = 0, amask = 0;                     // which of its pieces exist
#pragma unroll                                             // (the same for every row)
        for (int t = 0; t < NST; t++) {
            const int pc = lr + LPR * t;
            if (2 * pc < blen) bmask |= 1u << t;
            xs[t] = min(2 * pc, blen - 2); xg[t] = stage_index(xs[t]); xs[t] = 2 * swz(xs[t] / 2);
        }
        uint32_t sa_off[kXT / 2];                          // A: byte offset of piece lr + LPR t inside the staged row pair
        int ga_off[kXT / 2];                               //    and the x it starts at
        // the lane's window: pieces xa / 2 + j of B and of A, at their swizzled places (byte offsets inside a staged row pair)
        uint32_t ob[WIN / 2], oa[kXT / 2];
        const bool live = kXT * lr < ng;
        const int xa = live ? kXT * lr : 0;
#pragma unroll
        for (int j = 0; j < WIN / 2; j++) ob[j] = 16u * (uint32_t)swz(xa / 2 + j);
#pragma unroll
        for (int k = 0; k < kXT / 2; k++) {
            oa[k] = 8u * (uint32_t)blen_pad + 16u * (uint32_t)swz(xa / 2 + k);
            const int pc = lr + LPR * k;
            if (2 * pc < ng) amask |= 1u << k;
            ga_off[k] = min(2 * pc, ng - 2);
            sa_off[k] = 8u * (uint32_t)blen_pad + 16u * (uint32_t)swz(ga_off[k] / 2);
        }
        // stage s of this lane's row group: rows_sm[((s * 8 + wid) * RPW + sub) * slot]
        auto stage_ptr = [&](int st) { return rows_sm + (((size_t)st * 8 + wid) * RPW + sub) * slot; };
        // rows r0 + wid * RPW + sub + 8 RPW it: (gz, gy) advanced without a division; the slab is a whole number of trips
        int gz = z0, gy = wid * RPW + sub;
        while (gy >= ng) { gy -= ng; gz++; }
        auto issue = [&](int st) {                         // cp.async: the row pair goes to shared memory without passing registers
            const int gzc = min(gz, ng - 1);               // (a row past the end of the slab is fetched and never used)
            int hy = gy + v.x, hz = gzc + v.y;
            hy += hy < 0 ? ng : (hy >= ng ? -ng : 0);
            hz += hz < 0 ? ng : (hz >= ng ? -ng : 0);
            const double *A = delta + ((size_t)gzc * ng + gy) * ng, *B = delta + ((size_t)hz * ng + hy) * ng;
            double *sb = stage_ptr(st);
            const uint32_t sa = (uint32_t)__cvta_generic_to_shared(sb);
#pragma unroll
            for (int t = 0; t < NST; t++)
                if (bmask & (1u << t))
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(sa + 8u * (uint32_t)xs[t]), "l"(B + xg[t]) : "memory");
#pragma unroll
            for (int k = 0; k < kXT / 2; k++)
                if (amask & (1u << k))
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(sa + sa_off[k]), "l"(A + ga_off[k]) : "memory");
            asm volatile("cp.async.commit_group;" ::: "memory");
            gy += 8 * RPW;
            while (gy >= ng) { gy -= ng; gz++; }
        };
        for (int st = 0; st < kStagesDG - 1; st++) issue(st);
        const int ntrips = (r1 - r0) / (8 * RPW);
        int st = 0;
        for (int it = 0; it < ntrips; it++) {
            issue((st + kStagesDG - 1) % kStagesDG);       // kStagesDG - 1 row pairs in flight while this one is computed
            asm volatile("cp.async.wait_group %0;" ::"n"(kStagesDG - 1) : "memory");
            __syncwarp();
            const unsigned char *sb = reinterpret_cast<const unsigned char *>(stage_ptr(st));
            double a[kXT], w[WIN];
#pragma unroll
            for (int k = 0; k < kXT / 2; k++) {
                const double2 t = *reinterpret_cast<const double2 *>(sb + oa[k]);
                a[2 * k] = live ? t.x : 0.0; a[2 * k + 1] = live ? t.y : 0.0;
            }
#pragma unroll
            for (int j = 0; j < WIN / 2; j++) { const double2 t = *reinterpret_cast<const double2 *>(sb + ob[j]); w[2 * j] = t.x; w[2 * j + 1] = t.y; }
#pragma unroll
            for (int i = 0; i < kXT; i++)                  // (i outermost: 2M + 1 independent multiply-adds between dependent ones)
#pragma unroll
                for (int k = 0; k < W; k++) acc[k] = fma(a[i], w[i + k], acc[k]);
            __syncwarp();
            st = st + 1 == kStagesDG ? 0 : st + 1;
        }
        asm volatile("cp.async.wait_group 0;" ::: "memory");
    } else {
        // ---- any other row length: the same scheme with 4 points per lane, segment by segment, without the register pipeline
        const int ngp = (ng + 3) & ~3, blen = ngp + 2 * M;
        double *buf = rows_sm + (size_t)wid * blen;
        for (int r = r0 + wid; r < r1; r += 8) {
            const int gz = r / ng, gy = r - gz * ng;
            int hy = gy + v.x, hz = gz + v.y;
            hy += hy < 0 ? ng : (hy >= ng ? -ng : 0);
            hz += hz < 0 ? ng : (hz >= ng ? -ng : 0);
            const double *A = delta + ((size_t)gz * ng + gy) * ng, *B = delta + ((size_t)hz * ng + hy) * ng;
            for (int i = lane; i < blen; i += 32) buf[i] = i < ng + 2 * M ? B[stage_index(i)] : 0.0;
            __syncwarp();
            for (int x0 = 4 * lane; x0 < ngp; x0 += 128) {
                double a[4], w[4 + 2 * M];
#pragma unroll
                for (int k = 0; k < 4; k++) a[k] = (x0 + k < ng) ? A[x0 + k] : 0.0;
                const double2 *b2 = reinterpret_cast<const double2 *>(buf + x0);
#pragma unroll
                for (int j = 0; j < 2 + M; j++) { const double2 t = b2[j]; w[2 * j] = t.x; w[2 * j + 1] = t.y; }
#pragma unroll
                for (int i = 0; i < 4; i++)
#pragma unroll
                    for (int k = 0; k < W; k++) acc[k] = fma(a[i], w[i + k], acc[k]);
            }
            __syncwarp();
        }
    }
    // ---- reduce the accumulators over the CTA and add them to their bins (acc[k]: vx = k - M)
#pragma unroll
    for (int k = 0; k < W; k++) {
        double t = acc[k];
        for (int o = 16; o; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (lane == 0) red[wid][k] = t;
    }
    __syncthreads();
    if (threadIdx.x < W) {
        const int vx = (int)threadIdx.x - M, Wm = 2 * m + 1;
        const bool half = v.y > 0 || v.x > 0 || vx > 0;    // the mirrored offset is met through this one
        if (abs(vx) <= m && half) {
            const int bin = binidx[((v.y + m) * Wm + (v.x + m)) * Wm + (vx + m)];
            if (bin >= 0) {
                double t = 0.0;
                for (int w8 = 0; w8 < 8; w8++) t += red[w8][threadIdx.x];
                atomicAdd(&sum_dd[bin], 2.0 * t);
            }
        }
    }
}

template <int M>
static cudaError_t launch_rows(const double *delta, int ng, int m, const int2 *vyz, int npairs, int npairs_all, const int *binidx, double *sum_dd,
                               cudaStream_t s)
{
    int zsplit = (8 * dg_sm_count() + npairs_all - 1) / npairs_all;   // (the launches of the classes run back to back: size the slabs for all of them)
    zsplit = zsplit < 1 ? 1 : (zsplit > ng ? ng : zsplit);
    // fast path: ng a multiple of 8, at most 256, and every slab a whole number of trips of 8 warps x (32 / LPR) rows
    int lpr_log2 = -1;
    if (ng % kXT == 0 && ng <= 32 * kXT && ng > 4 * kXT) {   // (8, 16 or 32 lanes per row: the staging below assumes >= 8)
        int l2 = 0;
        while ((kXT << l2) < ng) l2++;
        const int trip = 8 * (32 >> l2);
        while (zsplit > 1 && (ng % zsplit != 0 || ((ng / zsplit) * ng) % trip != 0)) zsplit--;
        if (ng % zsplit == 0 && ((ng / zsplit) * ng) % trip == 0) lpr_log2 = l2;
    }
    const size_t smem = lpr_log2 >= 0 ? (size_t)kStagesDG * 8 * (size_t)(32 >> lpr_log2) * ((size_t)((ng + 2 * M + 15) & ~15) + (size_t)((ng + 15) & ~15)) * sizeof(double)
                                      : (size_t)8 * ((size_t)((ng + 3) & ~3) + 2 * M) * sizeof(double);
    cudaError_t e = cudaFuncSetAttribute(k_grid_corr_rows<M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_grid_corr_rows<M><<<npairs * zsplit, 256, smem, s>>>(delta, ng, m, vyz, zsplit, binidx, sum_dd, lpr_log2);
    return cudaGetLastError();
}

// host: the offsets of Eq. 17 and their bins, once
static int find_bin_host(const std::vector<double> &e, int n, double lo, double hi, int lg, double v)
{
    if (!(v >= e[0]) || !(v < e[n])) return -1;
    double g = lg ? (double)n * log(v / lo) / log(hi / lo) : (double)n * (v - lo) / (hi - lo);
    int k = (int)floor(g);
    k = k < 0 ? 0 : (k > n - 1 ? n - 1 : k);
    while (k > 0 && v < e[k]) k--;
    while (k < n - 1 && v >= e[k + 1]) k++;
    return k;
}

} // namespace cute

using namespace cute;

extern "C" {

static size_t dg_align(size_t x) { return (x + 255) / 256 * 256; }

static int dg_max_offsets(int ng, const cute_bin_spec *bins, double L, int *m_out)
{
    const double h = L / (double)ng;
    int m = (int)floor(bins->hi1 / h);
    if (m > (ng - 1) / 2) m = (ng - 1) / 2;
    if (m_out) *m_out = m;
    return (2 * m + 1) * (2 * m + 1) * (2 * m + 1);
}

int cute_density_grid_workspace_bytes(int ng, const cute_bin_spec *bins, double L, size_t *bytes)
{
    if (!bins || bins->struct_size != sizeof(cute_bin_spec) || !bytes || ng < 3 || ng > 2048 || !(L > 0.0)) return CUTE_ERR_INVALID_ARG;
    if (bins->n1 < 1 || !(bins->lo1 < bins->hi1) || bins->hi1 > 0.5 * L || (bins->log1 && !(bins->lo1 > 0.0))) return CUTE_ERR_INVALID_ARG;
    const size_t ng3 = (size_t)ng * ng * ng;
    const size_t noff = (size_t)dg_max_offsets(ng, bins, L, nullptr);
    *bytes = 256 + dg_align(ng3 * 8) + dg_align(noff * 16) + dg_align(((size_t)bins->n1 + 1) * 4) + dg_align((size_t)bins->n1 * 8);
    return CUTE_OK;
}

int cute_density_grid_xi(const cute_catalog *cat, double L, int ng, const cute_bin_spec *bins, double *h_xi, double *h_sum_dd,
                         uint64_t *h_npairs, double *d_delta, void *d_workspace, size_t bytes, void *stream)
{
    size_t need = 0;
    int rc = cute_density_grid_workspace_bytes(ng, bins, L, &need);
    if (rc) return rc;
    if (!cat || cat->struct_size != sizeof(cute_catalog) || cat->coord != CUTE_COORD_XYZ || cat->n < 1 || cat->n > 0x7fffffff) return CUTE_ERR_INVALID_ARG;
    if ((cat->dtype != CUTE_F32 && cat->dtype != CUTE_F64) || !cat->c0 || !cat->c1 || !cat->c2 || cat->weight) return CUTE_ERR_INVALID_ARG;
    if (!h_xi || !d_workspace || ((uintptr_t)d_workspace & 255)) return CUTE_ERR_INVALID_ARG;
    if (bytes < need) return CUTE_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t s = (cudaStream_t)stream;
    const int nb = bins->n1;
    const size_t ng3 = (size_t)ng * ng * ng;
    const double h = L / (double)ng;
    // ---- offsets and their bins, sorted by bin
    std::vector<double> e((size_t)nb + 1);
    for (int k = 0; k <= nb; k++)
        e[k] = bins->log1 ? exp(log(bins->lo1) + (double)k * (log(bins->hi1) - log(bins->lo1)) / (double)nb)
                          : bins->lo1 + (bins->hi1 - bins->lo1) * (double)k / (double)nb;
    e[0] = bins->lo1; e[nb] = bins->hi1;
    int m = 0;
    dg_max_offsets(ng, bins, L, &m);
    std::vector<int4> offs;
    for (int dz = -m; dz <= m; dz++)
        for (int dy = -m; dy <= m; dy++)
            for (int dx = -m; dx <= m; dx++) {
                if (dx == 0 && dy == 0 && dz == 0) continue;
                const double r = h * sqrt((double)(dx * dx + dy * dy + dz * dz));
                const int k = find_bin_host(e, nb, bins->lo1, bins->hi1, bins->log1, r);
                if (k >= 0) offs.push_back(make_int4(dx, dy, dz, k));
            }
    std::stable_sort(offs.begin(), offs.end(), [](const int4 &a, const int4 &b) { return a.w < b.w; });
    std::vector<uint32_t> bstart((size_t)nb + 1, 0);
    for (const int4 &o : offs) bstart[(size_t)o.w + 1]++;
    for (int k = 0; k < nb; k++) bstart[k + 1] += bstart[k];

    unsigned char *w = (unsigned char *)d_workspace;
    uint32_t *d_status = (uint32_t *)w;
    double *rho = (double *)(w + 256);
    int4 *d_offs = (int4 *)(w + 256 + dg_align(ng3 * 8));
    uint32_t *d_bstart = (uint32_t *)((unsigned char *)d_offs + dg_align((size_t)dg_max_offsets(ng, bins, L, nullptr) * 16));
    double *d_sum = (double *)((unsigned char *)d_bstart + dg_align(((size_t)nb + 1) * 4));
    if (cudaMemsetAsync(d_status, 0, 256, s) != cudaSuccess || cudaMemsetAsync(rho, 0, ng3 * 8, s) != cudaSuccess ||
        cudaMemsetAsync(d_sum, 0, (size_t)nb * 8, s) != cudaSuccess)
        return CUTE_ERR_CUDA;
    const bool fast = m <= 16 && m >= 1 && (size_t)8 * (((ng + 3) & ~3) + 32) * 8 <= 200 * 1024;
    if (!offs.empty() && !fast && cudaMemcpyAsync(d_offs, offs.data(), offs.size() * 16, cudaMemcpyHostToDevice, s) != cudaSuccess) return CUTE_ERR_CUDA;
    if (cudaMemcpyAsync(d_bstart, bstart.data(), bstart.size() * 4, cudaMemcpyHostToDevice, s) != cudaSuccess) return CUTE_ERR_CUDA;
    k_tsc3<<<dg_sm_count() * 8, 256, 0, s>>>(cat->c0, cat->c1, cat->c2, cat->dtype, cat->n, (double)ng / L, ng, rho, d_status);
    k_overdensity<<<(unsigned)((ng3 + 255) / 256), 256, 0, s>>>(rho, (int64_t)ng3, (double)ng3 / (double)cat->n);
    if (d_delta && cudaMemcpyAsync(d_delta, rho, ng3 * 8, cudaMemcpyDeviceToDevice, s) != cudaSuccess) return CUTE_ERR_CUDA;
    if (!offs.empty() && fast) {
        // fast stencil: the table offset -> bin and the list of (vy, vz) of the half-space live where the sorted offsets were
        const int Wm = 2 * m + 1;
        std::vector<int> binidx((size_t)Wm * Wm * Wm, -1);
        for (const int4 &o : offs) binidx[((size_t)(o.z + m) * Wm + (size_t)(o.y + m)) * Wm + (size_t)(o.x + m)] = o.w;
        // (vy, vz) of the half-space, grouped by the largest |vx| that still falls in a bin: a pair outside the sphere of
        // radius r_max is not swept at all, one near its rim sweeps 9 or 17 lags instead of 2m + 1
        std::vector<int2> vyz[4];
        for (int vz = 0; vz <= m; vz++)
            for (int vy = (vz == 0 ? 0 : -m); vy <= m; vy++) {
                int mx = -1;
                for (int vx = -m; vx <= m; vx++)
                    if (binidx[((size_t)(vz + m) * Wm + (size_t)(vy + m)) * Wm + (size_t)(vx + m)] >= 0 && abs(vx) > mx) mx = abs(vx);
                if (mx < 0) continue;
                vyz[mx <= 4 ? 0 : mx <= 8 ? 1 : mx <= 12 ? 2 : 3].push_back(make_int2(vy, vz));
            }
        std::vector<int2> all;
        int first[5] = {0, 0, 0, 0, 0};
        for (int c = 0; c < 4; c++) { all.insert(all.end(), vyz[c].begin(), vyz[c].end()); first[c + 1] = (int)all.size(); }
        int *d_binidx = (int *)d_offs;
        int2 *d_vyz = (int2 *)((unsigned char *)d_offs + dg_align(binidx.size() * 4));
        if (cudaMemcpyAsync(d_binidx, binidx.data(), binidx.size() * 4, cudaMemcpyHostToDevice, s) != cudaSuccess ||
            (!all.empty() && cudaMemcpyAsync(d_vyz, all.data(), all.size() * 8, cudaMemcpyHostToDevice, s) != cudaSuccess) ||
            cudaStreamSynchronize(s) != cudaSuccess)
            return CUTE_ERR_CUDA;   // (the host vectors go out of scope below: the copies must have left them)
        cudaError_t e = cudaSuccess;
        const int total = (int)all.size();
        for (int c = 0; c < 4 && e == cudaSuccess; c++) {
            const int np = first[c + 1] - first[c];
            if (np == 0) continue;
            const int2 *pl = d_vyz + first[c];
            if (c == 0) e = launch_rows<4>(rho, ng, m, pl, np, total, d_binidx, d_sum, s);
            else if (c == 1) e = launch_rows<8>(rho, ng, m, pl, np, total, d_binidx, d_sum, s);
            else if (c == 2) e = launch_rows<12>(rho, ng, m, pl, np, total, d_binidx, d_sum, s);
            else e = launch_rows<16>(rho, ng, m, pl, np, total, d_binidx, d_sum, s);
            note_launches(1);
        }
        if (e != cudaSuccess) return CUTE_ERR_CUDA;
    } else if (!offs.empty()) {
        k_grid_corr<<<(unsigned)((ng3 + kCorrThreads - 1) / kCorrThreads), kCorrThreads, 0, s>>>(rho, ng, d_offs, d_bstart, nb, d_sum);
        note_launches(1);
    }
    note_launches(2);   // k_tsc, k_overdensity
    if (cudaGetLastError() != cudaSuccess) return CUTE_ERR_CUDA;
    std::vector<double> sums((size_t)nb);
    uint32_t st = 0;
    if (cudaMemcpyAsync(sums.data(), d_sum, (size_t)nb * 8, cudaMemcpyDeviceToHost, s) != cudaSuccess ||
        cudaMemcpyAsync(&st, d_status, 4, cudaMemcpyDeviceToHost, s) != cudaSuccess || cudaStreamSynchronize(s) != cudaSuccess)
        return CUTE_ERR_CUDA;
    if (st) return CUTE_ERR_POINT_OUT_OF_BOX;
    int warn = CUTE_OK;
    for (int k = 0; k < nb; k++) {
        const uint64_t np = (uint64_t)(bstart[k + 1] - bstart[k]) * (uint64_t)ng3;
        if (h_npairs) h_npairs[k] = np;
        if (h_sum_dd) h_sum_dd[k] = sums[k];
        if (np == 0) { h_xi[k] = 0.0; warn = CUTE_WARN_EMPTY_BIN; }
        else h_xi[k] = sums[k] / (double)np;
    }
    return warn;
}

} // extern "C"
