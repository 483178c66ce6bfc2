// peaks.cu -- microbenchmarks of the units the pair kernel's roofline is made of (SURVEY.md 8(d) R2:
// "issue rate, MUFU, F2I, shared-atomic throughput vs multiplicity ... microbenchmarked, not taken on
// faith").  Each test runs one persistent 512-thread CTA per SM (the pair kernel's launch shape), times
// a loop of one instruction kind with clock64() inside the kernel, and reports LANE-operations per clock
// per SM (a packed f32x2 instruction counts as 2 lane-operations per lane).  cute_measure_peaks() is
// what bench.py calls to get its roofline denominator on the box it runs on.
#include "cute_internal.h"

namespace cute {

enum PeakOp {
    P_FFMA = 0, P_FADD, P_FFMA2, P_FADD2, P_FADD_RM, P_FADD2_RM, P_FMNMX, P_IADD, P_LOP3, P_IMAD,
    P_MUFU_SQRT, P_MUFU_LG2, P_MUFU_RSQ,
    P_ATOMS_INC_M1, P_ATOMS_INC_M2, P_ATOMS_INC_M4, P_ATOMS_INC_M8, P_ATOMS_INC_M32, P_ATOMS_ADD_M1,
    P_ATOMS_COLS8, P_ATOMS_COLS32, P_LDS128_BCAST,
    P_MIX_FFMA_FMNMX, P_MIX_FFMA2_FMNMX, P_MIX_FFMA2_MUFU_FMNMX, P_MIX_FFMA_IADD, P_MIX_FFMA2_FFMA,
    P_DFMA,      // float64 multiply-add: the density-grid stencil's roofline (density_grid.cu)
    P_COUNT
};

static const char *kPeakNames[P_COUNT] = {
    "ffma", "fadd", "ffma2", "fadd2", "fadd_rm", "fadd2_rm", "fmnmx", "iadd", "lop3", "imad",
    "mufu_sqrt", "mufu_lg2", "mufu_rsq",
    "atoms_inc_same1", "atoms_inc_same2", "atoms_inc_same4", "atoms_inc_same8", "atoms_inc_same32", "atoms_add_same1",
    "atoms_inc_cols8_random_bins", "atoms_inc_cols32_random_bins", "lds128_broadcast",
    "mix_ffma+fmnmx", "mix_ffma2+fmnmx", "mix_2ffma2+mufu+fmnmx", "mix_ffma+iadd", "mix_ffma2+ffma",
    "dfma"
};

constexpr int kPeakThreads = 512;
constexpr int kChains = 8;

// lane-operations one loop iteration of one thread performs
__host__ __device__ constexpr int ops_per_iter(int op)
{
    return (op == P_FFMA2 || op == P_FADD2 || op == P_FADD2_RM) ? 2 * kChains
         : (op == P_MIX_FFMA_FMNMX || op == P_MIX_FFMA_IADD) ? 2 * kChains
         : (op == P_MIX_FFMA2_FMNMX) ? 3 * kChains
         : (op == P_MIX_FFMA2_MUFU_FMNMX) ? 6 * kChains
         : (op == P_MIX_FFMA2_FFMA) ? 3 * kChains
         : (op == P_LDS128_BCAST) ? kChains
         : kChains;
}
// warp-instructions per thread per iteration (for the issue-rate view)
__host__ __device__ constexpr int instr_per_iter(int op)
{
    return (op == P_MIX_FFMA_FMNMX || op == P_MIX_FFMA_IADD || op == P_MIX_FFMA2_FMNMX || op == P_MIX_FFMA2_FFMA) ? 2 * kChains
         : (op == P_MIX_FFMA2_MUFU_FMNMX) ? 4 * kChains
         : kChains;
}

template <int OP>
__global__ void __launch_bounds__(kPeakThreads, 1) k_peak(unsigned long long *cyc, float *sink, int iters)
{
    __shared__ uint32_t sh[48 * 32 + 64];
    __shared__ unsigned long long tmax;
    const int lane = threadIdx.x & 31;
    for (int k = threadIdx.x; k < 48 * 32 + 64; k += blockDim.x) sh[k] = k;
    if (threadIdx.x == 0) tmax = 0;
    float a[kChains];
    unsigned long long a2[kChains];
    uint32_t u[kChains];
    double d[kChains];
    const double db = 1.0 + 1e-9 * (double)threadIdx.x, dc = 1e-12 * (double)(threadIdx.x & 31);
    const float b = 1.0f + 1e-7f * (float)threadIdx.x, c = 1e-9f * (float)lane;
    unsigned long long b2, c2;
    asm volatile("mov.b64 %0, {%1, %1};" : "=l"(b2) : "f"(b));
    asm volatile("mov.b64 %0, {%1, %1};" : "=l"(c2) : "f"(c));
#pragma unroll
    for (int k = 0; k < kChains; k++) {
        a[k] = 1.0f + 0.01f * (float)(k + lane);
        asm volatile("mov.b64 %0, {%1, %1};" : "=l"(a2[k]) : "f"(a[k]));
        u[k] = (uint32_t)(k * 7 + threadIdx.x);
        d[k] = 1.0 + 0.01 * (double)(k + lane);
    }
    // shared-atomic address patterns
    uint32_t base = (uint32_t)__cvta_generic_to_shared(sh);
    int mult = OP == P_ATOMS_INC_M2 ? 2 : OP == P_ATOMS_INC_M4 ? 4 : OP == P_ATOMS_INC_M8 ? 8 : OP == P_ATOMS_INC_M32 ? 32 : 1;
    uint32_t addr = base + 4u * (uint32_t)(lane / mult);       // `mult` lanes share one address; groups on distinct banks
    uint32_t rnd = 1234567u * (uint32_t)(threadIdx.x + 1) + 89u;
    // [bin][column] layouts of the pair kernel with a pseudo-random bin (0..39) per lane and chain
    uint32_t hoff[kChains];
#pragma unroll
    for (int k = 0; k < kChains; k++) {
        rnd = rnd * 1664525u + 1013904223u;
        const uint32_t bin = (rnd >> 16) % 40u;
        hoff[k] = base + 4u * (OP == P_ATOMS_COLS8 ? (bin * 8u + (uint32_t)(lane & 7)) : (bin * 32u + (uint32_t)lane));
    }
    __syncthreads();
    const long long t0 = clock64();
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int k = 0; k < kChains; k++) {
            if (OP == P_FFMA) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[k]) : "f"(b), "f"(c));
            else if (OP == P_DFMA) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[k]) : "d"(db), "d"(dc));
            else if (OP == P_FADD) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(a[k]) : "f"(c));
            else if (OP == P_FFMA2) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a2[k]) : "l"(b2), "l"(c2));
            else if (OP == P_FADD2) asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(a2[k]) : "l"(c2));
            else if (OP == P_FADD_RM) asm volatile("add.rm.f32 %0, %0, %1;" : "+f"(a[k]) : "f"(c));
            else if (OP == P_FADD2_RM) asm volatile("add.rm.f32x2 %0, %0, %1;" : "+l"(a2[k]) : "l"(c2));
            else if (OP == P_FMNMX) asm volatile("min.f32 %0, %0, %1;" : "+f"(a[k]) : "f"(b));
            else if (OP == P_IADD) asm volatile("add.s32 %0, %0, %1;" : "+r"(u[k]) : "r"(rnd));
            else if (OP == P_LOP3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u[k]) : "r"(rnd), "r"(base));
            else if (OP == P_IMAD) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(u[k]) : "r"(rnd), "r"(base));
            else if (OP == P_MUFU_SQRT) asm volatile("sqrt.approx.ftz.f32 %0, %0;" : "+f"(a[k]));
            else if (OP == P_MUFU_LG2) asm volatile("lg2.approx.ftz.f32 %0, %0;" : "+f"(a[k]));
            else if (OP == P_MUFU_RSQ) asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(a[k]));
            else if (OP >= P_ATOMS_INC_M1 && OP <= P_ATOMS_INC_M32)
                asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(addr + 128u * (uint32_t)k) : "memory");
            else if (OP == P_ATOMS_ADD_M1)
                asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr + 128u * (uint32_t)k), "r"(u[0]) : "memory");
            else if (OP == P_ATOMS_COLS8 || OP == P_ATOMS_COLS32)
                asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(hoff[k]) : "memory");
            else if (OP == P_LDS128_BCAST) {
                float4 v;
                asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                             : "r"(base + 16u * (uint32_t)((it + k) & 63)) : "memory");
                a[k] += v.x;
            } else if (OP == P_MIX_FFMA_FMNMX) {
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[k]) : "f"(b), "f"(c));
                asm volatile("min.f32 %0, %0, %1;" : "+f"(*reinterpret_cast<float *>(&u[k])) : "f"(b));
            } else if (OP == P_MIX_FFMA_IADD) {
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[k]) : "f"(b), "f"(c));
                asm volatile("add.s32 %0, %0, %1;" : "+r"(u[k]) : "r"(rnd));
            } else if (OP == P_MIX_FFMA2_FMNMX) {
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a2[k]) : "l"(b2), "l"(c2));
                asm volatile("min.f32 %0, %0, %1;" : "+f"(a[k]) : "f"(b));
            } else if (OP == P_MIX_FFMA2_FFMA) {
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a2[k]) : "l"(b2), "l"(c2));
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[k]) : "f"(b), "f"(c));
            } else if (OP == P_MIX_FFMA2_MUFU_FMNMX) {
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a2[k]) : "l"(b2), "l"(c2));
                asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(a2[k]) : "l"(c2));
                asm volatile("sqrt.approx.ftz.f32 %0, %0;" : "+f"(a[k]));
                asm volatile("min.f32 %0, %0, %1;" : "+f"(*reinterpret_cast<float *>(&u[k])) : "f"(b));
            }
        }
    }
    const long long t1 = clock64();
    atomicMax(&tmax, (unsigned long long)(t1 - t0));
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kChains; k++) s += a[k] + (float)(a2[k] & 0xffu) + (float)(u[k] & 0xffu) + (float)d[k];
    __syncthreads();
    if (threadIdx.x == 0) cyc[blockIdx.x] = tmax;
    if (s == 12345.678f) sink[threadIdx.x] = s + (float)sh[lane];   // never true: keeps the chains alive
}

template <int OP>
static cudaError_t run_one(unsigned long long *d_cyc, float *d_sink, int blocks, int iters, cudaStream_t s)
{
    k_peak<OP><<<blocks, kPeakThreads, 0, s>>>(d_cyc, d_sink, iters);
    note_launches(1);
    return cudaGetLastError();
}

template <int OP>
static cudaError_t run_all(unsigned long long *d_cyc, float *d_sink, int blocks, int iters, cudaStream_t s)
{
    cudaError_t e = run_one<OP>(d_cyc + (size_t)OP * 1024, d_sink, blocks, iters, s);
    if (e != cudaSuccess) return e;
    if constexpr (OP + 1 < P_COUNT) return run_all<OP + 1>(d_cyc, d_sink, blocks, iters, s);
    return cudaSuccess;
}

} // namespace cute

using namespace cute;

extern "C" {

int cute_peak_count(void) { return P_COUNT; }

const char *cute_peak_name(int idx) { return (idx >= 0 && idx < P_COUNT) ? kPeakNames[idx] : ""; }

int cute_measure_peaks(double *lane_ops_per_clk_sm, double *instr_per_clk_sm, int n, void *d_tmp, size_t bytes, void *stream)
{
    if (!lane_ops_per_clk_sm || n < P_COUNT || !d_tmp || ((uintptr_t)d_tmp & 255)) return CUTE_ERR_INVALID_ARG;
    const size_t need = (size_t)P_COUNT * 1024 * 8 + 4096;
    if (bytes < need) return CUTE_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t s = (cudaStream_t)stream;
    int dev = 0, blocks = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&blocks, cudaDevAttrMultiProcessorCount, dev);
    if (blocks > 1024) blocks = 1024;
    unsigned long long *d_cyc = (unsigned long long *)d_tmp;
    float *d_sink = (float *)((unsigned char *)d_tmp + (size_t)P_COUNT * 1024 * 8);
    const int iters = 2048;
    for (int rep = 0; rep < 2; rep++)   // the first pass warms the instruction cache and the clocks
        if (run_all<0>(d_cyc, d_sink, blocks, iters, s) != cudaSuccess) return CUTE_ERR_CUDA;
    static unsigned long long h[P_COUNT * 1024];
    if (cudaMemcpyAsync(h, d_cyc, sizeof(h), cudaMemcpyDeviceToHost, s) != cudaSuccess || cudaStreamSynchronize(s) != cudaSuccess)
        return CUTE_ERR_CUDA;
    for (int op = 0; op < P_COUNT; op++) {
        // median over the SMs of the slowest warp's cycles
        unsigned long long v[1024];
        for (int b = 0; b < blocks; b++) v[b] = h[(size_t)op * 1024 + b];
        for (int i = 1; i < blocks; i++) { unsigned long long x = v[i]; int j = i - 1; while (j >= 0 && v[j] > x) { v[j + 1] = v[j]; j--; } v[j + 1] = x; }
        const double cycles = (double)v[blocks / 2];
        const double lanes = (double)kPeakThreads * (double)iters;
        lane_ops_per_clk_sm[op] = cycles > 0 ? lanes * ops_per_iter(op) / cycles : 0.0;
        if (instr_per_clk_sm) instr_per_clk_sm[op] = cycles > 0 ? lanes / 32.0 * instr_per_iter(op) / cycles : 0.0;
    }
    return CUTE_OK;
}

} // extern "C"
