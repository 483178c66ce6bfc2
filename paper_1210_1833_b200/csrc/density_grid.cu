// density_grid.cu -- the density-grid monopole of CUTE_box:
// "the particle content of the catalog is first interpolated to a grid and the overdensity field delta is
// estimated at every grid point using a TSC algorithm.  Then pairs of grid points are correlated, and a weight
// delta_i delta_j is given to each pair.  The correlation function is estimated as
//        xi(r) = < delta(x) delta(x + r) >                                                        (Eq. 17)
// ... since the relative distances between neighboring points are the same everywhere, these relative
// distances only have to be calculated once."
// Readings D1-D4: grid points = cell centres (g + 1/2) h; TSC = second-order B-spline per axis;
// delta = rho / (N / ng^3) - 1; every ordered pair (g, g + v), v != 0 with the minimum image, r = h |v|, half-open bins.
// Three kernels: TSC scatter (float64 atomics into the L2-resident grid; HBM-bound on the particle read),
// overdensity (elementwise), and the offset-stencil correlation: the offsets are found, binned and sorted by bin ONCE on
// the host; every thread owns one grid point and sweeps the offsets of a bin with one float64 accumulator, the block
// reduces it and adds it to the bin's global sum.  All arithmetic float64 (the grid fits L2; this path is not the
// float32 pair kernel), so the result differs from a serial float64 loop only by the order of the additions.
#include "cute_internal.h"
#include <math.h>
#include <vector>
#include <algorithm>

namespace cute {

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

__global__ void __launch_bounds__(256) k_tsc(const void *x, const void *y, const void *z, int dtype, int64_t n, double inv_h, int ng,
                                             double *rho, uint32_t *status)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
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
    if (bad) { atomicExch(status, 1u); return; }
    int gx[3], gy[3], gz[3];
#pragma unroll
    for (int k = 0; k < 3; k++) { gx[k] = wrap(g0[0] + k, ng); gy[k] = wrap(g0[1] + k, ng); gz[k] = wrap(g0[2] + k, ng); }
#pragma unroll
    for (int a = 0; a < 3; a++)
#pragma unroll
        for (int b = 0; b < 3; b++)
#pragma unroll
            for (int c = 0; c < 3; c++)
                atomicAdd(&rho[((size_t)gz[a] * ng + gy[b]) * ng + gx[c]], w[0][c] * w[1][b] * w[2][a]);
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
    if (!offs.empty() && cudaMemcpyAsync(d_offs, offs.data(), offs.size() * 16, cudaMemcpyHostToDevice, s) != cudaSuccess) return CUTE_ERR_CUDA;
    if (cudaMemcpyAsync(d_bstart, bstart.data(), bstart.size() * 4, cudaMemcpyHostToDevice, s) != cudaSuccess) return CUTE_ERR_CUDA;
    k_tsc<<<(unsigned)((cat->n + 255) / 256), 256, 0, s>>>(cat->c0, cat->c1, cat->c2, cat->dtype, cat->n, (double)ng / L, ng, rho, d_status);
    k_overdensity<<<(unsigned)((ng3 + 255) / 256), 256, 0, s>>>(rho, (int64_t)ng3, (double)ng3 / (double)cat->n);
    if (d_delta && cudaMemcpyAsync(d_delta, rho, ng3 * 8, cudaMemcpyDeviceToDevice, s) != cudaSuccess) return CUTE_ERR_CUDA;
    if (!offs.empty()) k_grid_corr<<<(unsigned)((ng3 + kCorrThreads - 1) / kCorrThreads), kCorrThreads, 0, s>>>(rho, ng, d_offs, d_bstart, nb, d_sum);
    note_launches(3);
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
