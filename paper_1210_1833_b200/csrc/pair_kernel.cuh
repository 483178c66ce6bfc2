// pair_kernel.cuh -- the pair kernel, device side.  Instantiated per kind in
// pair_kind*.cu (so that the kinds compile in parallel); planned and launched from pair_count.cu.
//
// What is computed (sec. III.A): for every pair of objects "calculating the distance
// between each pair of objects, determining the bin corresponding to that distance and increasing
// the histogram count on that bin", Eq. 11.  The paper's CUDA kernel
// lets every thread stride over j for one i and atomicAdd into one shared histogram per block; it
// names the histogram update "the bottleneck of any algorithm involving histograms in CUDA"
// (PAPER.md:192).  That design is prior art; this one is organised for sm_100a:
//
//  * every WARP is an independent worker: it pops a work item (<=128 cell-sorted i-points of one
//    cell row, 4 per lane, held in registers) from a global queue and streams the contiguous
//    j-ranges of the neighbouring cell rows ("Neighbors ... are only searched for in the gray
//    region") through its own double-buffered shared-memory tiles, filled by
//    1-D TMA bulk copies (cp.async.bulk + mbarrier) issued by lane 0.  No __syncthreads in the loop.
//  * each j is read once per warp as a broadcast LDS.128 and meets 128 i-points.
//  * separations in float32 with PACKED f32x2 arithmetic (FADD2 / FMUL2 / FFMA2, new on sm_100): a lane's
//    four i-points live in registers as two packed pairs, the j-point is the broadcast scalar operand, so
//    one instruction slot does the work of two pairs.  Measured (cute_measure_peaks): FFMA2 keeps the
//    full 128 lane-operations per clock per SM in HALF the issue slots, and issue slots are what this
//    kernel runs out of.  Squared comoving distance (monopole, r-mu) or squared chord on unit vectors
//    (angular; PAPER.md:233 without the arccos of PAPER.md:235-239).  The float32 chord carries the absolute
//    rounding of the unit vectors (~2e-7), so pairs closer than a theta_min chosen on the host go to float64
//    together with the pairs near a bin edge (measured: the hi/lo-corrected chord of round 1 made the angular
//    kernel FP32-pipe-bound, 12 lane-operations per pair for the separation instead of 6).
//  * bin map without division or compare chains: t = S*g(q) + O - 1/2 with g = MUFU sqrt or log2; ONE
//    round-to-nearest add of 1.5*2^23 leaves floor(t + 1/2) in the mantissa, and d = t - rint(t) is the
//    distance of the pair from the centre of its bin in units of bins.  The float32 bin is certain iff
//    |d| <= 1/2 - tau (tau = a proven bound on the float32 error); otherwise the lane queues its BLOCK of
//    pairs, the warp re-examines queued blocks 32 at a time, recomputes their uncertain pairs in float64 (the
//    definition) and moves a provisional count whose float64 cell differs ("the rare path" below), so the
//    histogram equals the float64 definition except at float64-rounding distance of an edge.
//  * histogram: per-warp private uint32 copies in shared memory, [bin][column] (8 columns per warp;
//    a 2-D histogram too large for that is kept once per CTA), with one row (2-D: a border) of dump
//    cells on either side: out-of-range pairs are CLAMPED into the border instead of being predicated
//    off (FMNMX + LEA + ATOMS.POPC.INC per pair, no compare, no select).  Flushed to the uint64 global
//    histogram with 64-bit atomics before 2^32 increments can accumulate and at the end.
#pragma once
#include "cute_internal.h"
#include <math.h>

namespace cute {

// ------------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}
// 1-D TMA bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ float fast_sqrt(float x)
{
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float fast_rsqrt(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float fast_lg2(float x)
{
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// shared-memory increment without a return value (value 1: ATOMS.POPC.INC, which merges lanes that hit one address)
__device__ __forceinline__ void red_shared(uint32_t addr)
{
    asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(addr) : "memory");
}
__device__ __forceinline__ void red_shared_add(uint32_t addr, uint32_t v)
{
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// ---- packed float32 pairs: one FADD2 / FMUL2 / FFMA2 does two lanes' worth of work per thread in one issue slot.
// A pair built from one scalar (bc) is folded by ptxas into the instruction's broadcast operand form (R.F32).
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk(float a, float b)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ f32x2 bc(float a) { return pk(a, a); }
__device__ __forceinline__ void unpk(f32x2 v, float &a, float &b)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

#define CUTE_MAGIC_F 12582912.0f        /* 1.5 * 2^23: adding it (round to nearest) leaves rint(t) in the mantissa */
#define CUTE_MAGIC_BITS 0x4B400000u

// kernel variants (template FLAGS)
enum : int {
    PK_FIXCS = 1,      // the histogram column count is the kind's default (compile-time shift): 8 columns, or 1 for the 2-D kinds
    PK_SIMPLE = 2,     // linear bins starting at 0 on every axis (no lower clamp), constant-folded |l|^-2 term for r-mu
    PK_ALWAYS = 4,     // every candidate pair goes to float64 (RADIAL, force_refine)
    PK_WEIGHTED = 8    // pairs count w_i * w_j (pixel maps)
};

__host__ __device__ constexpr bool kind_is_2d(int kind) { return kind == CUTE_RMU || kind == CUTE_PISIGMA || kind == CUTE_RADIAL; }
__host__ __device__ constexpr int fixed_colshift(int kind) { return kind_is_2d(kind) ? 0 : 3; }

// ------------------------------------------------------------------------------- float64 definition
// The refine path: the pair's binned variable(s) exactly as the paper defines them, in IEEE float64
// with explicit round-to-nearest operations (no FMA contraction), and the bin looked up in the edge
// array (the sole authority on edges).
__device__ __forceinline__ int find_bin64(const double *e, int n, double lo, double hi, int lg, int closed_top, double v)
{
    if (!(v >= e[0])) return -1;
    if (!(v < e[n])) return (closed_top && v == e[n]) ? n - 1 : -1;
    double g = lg ? (double)n * log(v / lo) / log(hi / lo) : (double)n * (v - lo) / (hi - lo);
    int k = (int)floor(g);
    k = k < 0 ? 0 : (k > n - 1 ? n - 1 : k);
    while (k > 0 && v < e[k]) k--;
    while (k < n - 1 && v >= e[k + 1]) k++;
    return k;
}

__device__ __forceinline__ double norm2_64(double x, double y, double z)
{
    return __dadd_rn(__dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y)), __dmul_rn(z, z));
}

__device__ __forceinline__ void load64(const GridView &g, uint32_t idx, double v[4], int nload)
{
    if (g.p64) {
        for (int d = 0; d < nload; d++) v[d] = g.p64[4 * (size_t)idx + d];
    } else {   // float32 catalogue: the float32 values ARE the input
        float4 h = g.hi[idx];
        v[0] = h.x; v[1] = h.y; v[2] = h.z; v[3] = h.w;
    }
}

template <int KIND>
__device__ __noinline__ int refine_cell(const PairParams &p, uint32_t i_idx, uint32_t j_idx)
{
    double a[4], b[4];
    load64(p.g1, i_idx, a, KIND == CUTE_RADIAL ? 4 : 3);
    load64(p.g2, j_idx, b, KIND == CUTE_RADIAL ? 4 : 3);
    double dx = __dsub_rn(a[0], b[0]), dy = __dsub_rn(a[1], b[1]), dz = __dsub_rn(a[2], b[2]);
    double v1, v2 = 0.0;
    if (KIND == CUTE_MONOPOLE) {
        if (p.L > 0.0) {   // periodic box: minimum image
            dx = __dsub_rn(dx, __dmul_rn(p.L, rint(__ddiv_rn(dx, p.L))));
            dy = __dsub_rn(dy, __dmul_rn(p.L, rint(__ddiv_rn(dy, p.L))));
            dz = __dsub_rn(dz, __dmul_rn(p.L, rint(__ddiv_rn(dz, p.L))));
        }
        v1 = __dsqrt_rn(norm2_64(dx, dy, dz));
    } else if (KIND == CUTE_ANGULAR || KIND == CUTE_RADIAL) {
        double h = __dmul_rn(0.5, __dsqrt_rn(norm2_64(dx, dy, dz)));   // theta = 2 asin(chord/2)
        if (h > 1.0) h = 1.0;
        double th = __dmul_rn(2.0, asin(h));
        if (KIND == CUTE_ANGULAR) v1 = th;
        else {
            if (!(th < p.aperture)) return -1;                          // strict
            v1 = __dmul_rn(0.5, __dadd_rn(a[3], b[3]));
            v2 = fabs(__dsub_rn(a[3], b[3]));
        }
    } else {   // RMU, PISIGMA: mid-point line of sight l = x_i + x_j (Eq. 9)
        double lx = __dadd_rn(a[0], b[0]), ly = __dadd_rn(a[1], b[1]), lz = __dadd_rn(a[2], b[2]);
        double r = __dsqrt_rn(norm2_64(dx, dy, dz)), l = __dsqrt_rn(norm2_64(lx, ly, lz));
        double mu = 0.0;
        if (r > 0.0 && l > 0.0) {
            double dot = __dadd_rn(__dadd_rn(__dmul_rn(dx, lx), __dmul_rn(dy, ly)), __dmul_rn(dz, lz));
            mu = __ddiv_rn(fabs(dot), __dmul_rn(r, l));
        }
        if (mu > 1.0) mu = 1.0;
        v1 = r; v2 = mu;
        if (KIND == CUTE_PISIGMA) {   // Eq. 2: pi = r mu, sigma = sqrt(r^2 - pi^2)
            const double pi = __dmul_rn(r, mu), s2 = __dsub_rn(__dmul_rn(r, r), __dmul_rn(pi, pi));
            v1 = pi; v2 = s2 > 0.0 ? __dsqrt_rn(s2) : 0.0;
        }
    }
    int k1 = find_bin64(p.edges1, p.n1, p.lo1, p.hi1, p.logbins, 0, v1);
    if (k1 < 0) return -1;
    if (p.n2 > 0) {
        int k2 = find_bin64(p.edges2, p.n2, p.lo2, p.hi2, 0, p.closed_top2, v2);
        if (k2 < 0) return -1;
        return k1 * p.n2 + k2;
    }
    return k1;
}

// ------------------------------------------------------------------------------- per-warp state
constexpr int R = kIPerLane;
constexpr uint32_t kTileBytes = kTile * 16;

struct WarpSmem {          // pointers into this warp's slice of dynamic shared memory
    float4 *thi, *tlo;     // [kStages][kTile]
    uint4 *segs;           // [kSegSlots] {j_begin, j_end, code, -}
    uint4 *rq;             // [kRefineCap] flagged blocks {idx0, j, meta, i_last} (see flag_block)
    uint4 *pq;             // [kPairCap] uncertain pairs {i, j, provisional address, weight}
    uint32_t *rq_count, *pq_count;
    uint32_t *hist;        // [nhist_pad << colshift]
    uint32_t bar[kStages]; // shared-space addresses of the mbarriers
};

template <bool NEEDLO>
__device__ __forceinline__ WarpSmem carve(unsigned char *ws)
{
    WarpSmem s;
    s.thi = reinterpret_cast<float4 *>(ws);
    ws += kStages * kTileBytes;
    s.tlo = reinterpret_cast<float4 *>(ws);
    if (NEEDLO) ws += kStages * kTileBytes;
    s.segs = reinterpret_cast<uint4 *>(ws);
    ws += kSegSlots * 16;
    s.rq = reinterpret_cast<uint4 *>(ws);
    ws += kRefineCap * 16;
    s.pq = reinterpret_cast<uint4 *>(ws);
    ws += kPairCap * 16;
    for (int k = 0; k < kStages; k++) s.bar[k] = smem_u32(ws + 8 * k);
    s.rq_count = reinterpret_cast<uint32_t *>(ws + 8 * kStages);
    s.pq_count = s.rq_count + 1;
    ws += 32;
    s.hist = reinterpret_cast<uint32_t *>(ws);
    return s;
}

// The shared-memory histogram is PADDED: one dump row below and above (1-D), a border of dump cells (2-D).
// padded index of real cell c = k1 * n2eff + k2:
__device__ __forceinline__ uint32_t pad_cell(const PairParams &p, uint32_t cell)
{
    if (p.n2 > 0) return (cell / (uint32_t)p.n2 + 1u) * (uint32_t)p.n2p + cell % (uint32_t)p.n2 + 1u;
    return cell + 1u;
}

// P5: add this warp's private histogram to the global uint64 histogram and clear it.
// Lanes own cells; the column index is rotated by the lane so that the 32 reads hit 32 banks.
__device__ __forceinline__ void flush_hist(const PairParams &p, const WarpSmem &s, int lane)
{
    __syncwarp();
    const int C = 1 << p.colshift;
    for (uint32_t c = lane; c < (uint32_t)p.nhist_pad; c += 32) {
        const uint32_t k1p = p.n2 > 0 ? c / (uint32_t)p.n2p : c, k2p = p.n2 > 0 ? c % (uint32_t)p.n2p : 1u;
        unsigned long long sum = 0;
        uint32_t *row = s.hist + ((size_t)c << p.colshift);
        for (int k = 0; k < C; k++) {
            int col = (k + lane) & (C - 1);
            if (p.hist_shared) sum += atomicExch(row + col, 0u);   // other warps keep adding: read-and-clear in one step
            else {
                // the epoch bound keeps every private counter far below 2^31: one above it means increments were lost
                if (row[col] >= 0x80000000u) atomicOr(p.status, 2u);
                sum += row[col]; row[col] = 0;
            }
        }
        // border cells hold the clamped out-of-range pairs: dropped
        const bool real = k1p >= 1u && k1p <= (uint32_t)p.n1 && k2p >= 1u && (p.n2 == 0 || k2p <= (uint32_t)p.n2);
        // a column can hold a count moved away before it arrived as 2^32 - 1: the sum over the columns is taken modulo 2^32
        if (!p.hist_shared) sum &= 0xffffffffull;
        else sum = (unsigned long long)(long long)(int)(uint32_t)sum;   // shared copy: a moved count may follow another warp's flush
        if (real && sum) atomicAdd(p.hist + ((k1p - 1u) * (uint32_t)p.n2eff + (p.n2 > 0 ? k2p - 1u : 0u)), sum);
    }
    __syncwarp();
}

// weight of a pair: w_i * w_j for weighted catalogues (pixel maps), else 1.  The integer weight travels as
// a bit pattern in hi.w (RA/Dec catalogues) or in lo.x (xyz catalogues, whose hi.w holds |x|^2)
__device__ __forceinline__ uint32_t pair_weight(const PairParams &p, uint32_t i, uint32_t j)
{
    if (!p.weighted) return 1u;
    if (p.weight_in_lo) return __float_as_uint(p.g1.lo[i].x) * __float_as_uint(p.g2.lo[j].x);
    return __float_as_uint(p.g1.hi[i].w) * __float_as_uint(p.g2.hi[j].w);
}

// ------------------------------------------------------------------------------- the per-pair body
struct IPoints {           // the R = 4 i-points of this lane as two packed pairs (points 0,1 and 2,3)
    f32x2 X[2], Y[2], Z[2];      // hi (already shifted by the segment's periodic image)
    f32x2 X0[2], Y0[2], Z0[2];   // hi, unshifted (periodic cell lists re-derive X, Y, Z per segment)
    f32x2 W[2], LW[2];           // RMU / PISIGMA: |x|^2 hi, |x|^2 lo
    float w[R];                  // RADIAL: z; WEIGHTED: weight bit patterns
    uint32_t idx0;               // cell-sorted index of i-point 0 (point r is idx0 + 32 r)
};

struct Consts {            // loop constants held in registers (not re-read from the constant bank)
    float q_hi, q_small, dz_hi, Lf, invL;   // q_small: ANGULAR, pairs closer than theta_min always go to float64
    float q_mid, thr_mid, tau_a, tau_b;     // ANGULAR log bins: tau = tau_a + tau_b / chord; thr1 holds for q >= q_mid
    float S1, O1h, thr1, top1, tauw1, c1, c2, c3, c4;   // O1h = O - 1/2, thr1 = 1/2 - tau, top1 = MAGIC + n1
    float S2, O2h, top2, tv2, tauw2, cc2;               // tv2 = tau2 - 1/2
    uint32_t n2p;
};

template <int KIND>
__device__ __forceinline__ Consts load_consts(const PairParams &p)
{
    Consts c;
    c.q_hi = p.q_hi; c.q_small = p.q_small; c.dz_hi = p.dz_hi;
    c.q_mid = p.q_mid; c.thr_mid = 0.5f - p.tau_mid; c.tau_a = p.tau_a; c.tau_b = p.tau_b; c.Lf = p.Lf; c.invL = p.Lf > 0.f ? 1.0f / p.Lf : 0.f;
    c.S1 = p.a1.S; c.O1h = p.a1.O - 0.5f; c.thr1 = 0.5f - p.a1.tau; c.top1 = CUTE_MAGIC_F + (float)p.n1; c.tauw1 = p.a1.tau_w;
    c.c1 = p.a1.c1; c.c2 = p.a1.c2; c.c3 = p.a1.c3; c.c4 = p.a1.c4;
    c.S2 = p.a2.S; c.O2h = p.a2.O - 0.5f; c.top2 = CUTE_MAGIC_F + (float)p.n2; c.tv2 = p.a2.tau - 0.5f; c.tauw2 = p.a2.tau_w;
    c.cc2 = p.a1.c1;
    if (KIND == CUTE_RMU) {
        // the kernel works with w' = sqrt(2) / (r |l|) (it forms q * |l|^2 / 2) and tests d^2 > 1/4 - tau2
        c.S2 = p.a2.S * 0.70710678f; c.tauw2 = p.a2.tau_w * 0.70710678f; c.cc2 = p.a1.c1 * 0.5f; c.tv2 = p.a2.tau - 0.25f;
    }
    c.n2p = (uint32_t)p.n2p;
    return c;
}

// rint and distance from it, two pairs at a time: r = MAGIC + rint(t), d = t - rint(t) in [-1/2, 1/2]  (t = S g + Oh)
__device__ __forceinline__ void axis_round(f32x2 g, float S, float Oh, f32x2 &r, f32x2 &d)
{
    const f32x2 t = fma2(g, bc(S), bc(Oh));
    r = add2(t, bc(CUTE_MAGIC_F));
    d = sub2(t, sub2(r, bc(CUTE_MAGIC_F)));   // both subtractions are exact
}

// P2: squared separations of the lane's four i-points from one j-point, as two packed pairs
template <int KIND, bool MINIMG>
__device__ __forceinline__ void separations(const Consts &c, const IPoints &ip, const float4 pj, f32x2 q2[2])
{
#pragma unroll
    for (int h = 0; h < 2; h++) {
        f32x2 dx = sub2(ip.X[h], bc(pj.x)), dy = sub2(ip.Y[h], bc(pj.y)), dz = sub2(ip.Z[h], bc(pj.z));
        if (MINIMG) {
            // periodic brute force: minimum image.  Only d^2 is needed and the coordinates lie in [0, L) (checked
            // when the grid is made), so |d'| = min(|d|, L - |d|): one packed add on the float32 pipe and two FMNMX on the ALU
            // pipe per axis, instead of three packed operations for d - L rint(d / L) -- this kernel is float32-pipe-bound.
            const f32x2 Lp = bc(c.Lf);
            float a0, a1, b0, b1;
            // (the absolute values are written on the scalars: ptxas folds them into the |.| operand modifiers)
            unpk(dx, a0, a1); unpk(sub2(Lp, pk(fabsf(a0), fabsf(a1))), b0, b1); dx = pk(fminf(fabsf(a0), b0), fminf(fabsf(a1), b1));
            unpk(dy, a0, a1); unpk(sub2(Lp, pk(fabsf(a0), fabsf(a1))), b0, b1); dy = pk(fminf(fabsf(a0), b0), fminf(fabsf(a1), b1));
            unpk(dz, a0, a1); unpk(sub2(Lp, pk(fabsf(a0), fabsf(a1))), b0, b1); dz = pk(fminf(fabsf(a0), b0), fminf(fabsf(a1), b1));
        }
        q2[h] = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
    }
}

// P3: the float32 bin map of the four pairs (lane's i-points x one j).  r1 (r2) = MAGIC + bin as a float;
// va = |d| of axis 1 (uncertain iff > thr1), vb = pair-dependent margin (uncertain iff > 0); returns "some pair uncertain".
template <int KIND, bool LOGB, bool SIMPLE>
__device__ __forceinline__ bool bin_map(const PairParams &p, const Consts &c, const IPoints &ip, const f32x2 q2[2], const float q[R],
                                        float wj, float lwj, float r1[R], float r2[R], float va[R], float vb[R])
{
    bool flag = false;
#pragma unroll
    for (int r = 0; r < R; r++) { r1[r] = 0.f; r2[r] = 0.f; va[r] = 0.f; vb[r] = -1.f; }
    if constexpr (KIND == CUTE_MONOPOLE || KIND == CUTE_ANGULAR || KIND == CUTE_RMU) {
        f32x2 g2[2];
        float w1[R];
        if constexpr (KIND == CUTE_ANGULAR) {
            // theta^2 = q P(q) (log bins) or theta = sqrt(q) P(q) (linear), P a cubic fitted on the host
#pragma unroll
            for (int h = 0; h < 2; h++) {
                const f32x2 poly = fma2(q2[h], fma2(q2[h], fma2(q2[h], bc(c.c4), bc(c.c3)), bc(c.c2)), bc(c.c1));
                float a, b;
                // (q = 0: lg2 = -inf, the pair is clamped into the lower dump row, as it must: theta = 0 < lo)
                if (LOGB) { unpk(mul2(q2[h], poly), a, b); g2[h] = pk(fast_lg2(a), fast_lg2(b)); }
                else g2[h] = mul2(pk(fast_sqrt(q[2 * h]), fast_sqrt(q[2 * h + 1])), poly);
            }
        } else if constexpr (LOGB) {
            // log bins in r: the absolute float32 error e_r of r is e_r / r in ln r, so tau = a + b / r
#pragma unroll
            for (int r = 0; r < R; r++) w1[r] = fmaxf(q[r], 1.0e-30f);
#pragma unroll
            for (int h = 0; h < 2; h++) g2[h] = pk(fast_lg2(w1[2 * h]), fast_lg2(w1[2 * h + 1]));
#pragma unroll
            for (int r = 0; r < R; r++) w1[r] = fast_rsqrt(w1[r]);
        } else {
#pragma unroll
            for (int h = 0; h < 2; h++) g2[h] = pk(fast_sqrt(q[2 * h]), fast_sqrt(q[2 * h + 1]));
        }
        float d[R];
#pragma unroll
        for (int h = 0; h < 2; h++) {
            f32x2 rr, dd;
            axis_round(g2[h], c.S1, c.O1h, rr, dd);
            unpk(rr, r1[2 * h], r1[2 * h + 1]);
            unpk(dd, d[2 * h], d[2 * h + 1]);
        }
        if constexpr (KIND == CUTE_MONOPOLE && LOGB) {
#pragma unroll
            for (int r = 0; r < R; r++) vb[r] = fabsf(d[r]) + fmaf(w1[r], c.tauw1, -c.thr1);
            flag = fmaxf(fmaxf(vb[0], vb[1]), fmaxf(vb[2], vb[3])) > 0.f;
        } else {
#pragma unroll
            for (int r = 0; r < R; r++) va[r] = fabsf(d[r]);
            flag = fmaxf(fmaxf(va[0], va[1]), fmaxf(va[2], va[3])) > c.thr1;
        }
        if constexpr (KIND == CUTE_RMU) {
            // mu = |s.l| / (|s||l|), s.l = |x_i|^2 - |x_j|^2 (hi/lo squares: no cancellation),
            // |l|^2 / 2 = |x_i|^2 + |x_j|^2 - q / 2   (mid-point line of sight, Eq. 9)
            f32x2 v2[2];
#pragma unroll
            for (int h = 0; h < 2; h++) {
                const f32x2 pn = add2(sub2(ip.W[h], bc(wj)), sub2(ip.LW[h], bc(lwj)));
                const f32x2 mh = fma2(q2[h], bc(-0.5f), add2(ip.W[h], bc(wj)));
                // q |l|^2 / 2, kept away from 0: q = 0 or |l| = 0 then give a huge but finite w, hence a huge tau2 and an
                // uncertain pair (SIMPLE: the catalogue is far from the origin, |l|^2 cannot round to a negative number)
                float qa, qb;
                if (SIMPLE) unpk(fma2(q2[h], mh, bc(1.0e-30f)), qa, qb);
                else { unpk(mul2(q2[h], mh), qa, qb); qa = fmaxf(qa, 1.0e-30f); qb = fmaxf(qb, 1.0e-30f); }
                const f32x2 w = pk(fast_rsqrt(qa), fast_rsqrt(qb));        // sqrt(2) / (r |l|)
                float ma, mb;
                unpk(mul2(pn, w), ma, mb);
                f32x2 rr, dd;
                axis_round(pk(fabsf(ma), fabsf(mb)), c.S2, c.O2h, rr, dd);
                // tau2 - 1/4 = a + b/(r|l|) [+ c/|l|^2, folded into a when the catalogue is far from the origin];
                // uncertain iff d^2 > 1/4 - tau2 (a little more than |d| > 1/2 - tau2)
                f32x2 tv = fma2(w, bc(c.tauw2), bc(c.tv2));
                if (!SIMPLE) tv = fma2(mul2(mul2(w, w), q2[h]), bc(c.cc2), tv);
                v2[h] = fma2(dd, dd, tv);
                unpk(rr, r2[2 * h], r2[2 * h + 1]);
            }
            unpk(v2[0], vb[0], vb[1]);
            unpk(v2[1], vb[2], vb[3]);
            flag = flag || (fmaxf(fmaxf(vb[0], vb[1]), fmaxf(vb[2], vb[3])) > 0.f);
        }
    } else if constexpr (KIND == CUTE_PISIGMA) {
        // pi = |s.l| / |l|, sigma = sqrt(q - pi^2)  (Eq. 2); both taus depend on the pair
        float wi[R], lwi[R];
        unpk(ip.W[0], wi[0], wi[1]); unpk(ip.W[1], wi[2], wi[3]);
        unpk(ip.LW[0], lwi[0], lwi[1]); unpk(ip.LW[1], lwi[2], lwi[3]);
#pragma unroll
        for (int r = 0; r < R; r++) {
            const float pn = (wi[r] - wj) + (lwi[r] - lwj);
            const float m = fmaf(2.0f, wi[r] + wj, -q[r]);
            const float w1 = fast_rsqrt(fmaxf(m, 1.0e-30f));               // clamps: no NaN/inf, a huge tau instead
            const float pi = fabsf(pn) * w1;
            const float epi = fmaf(w1 * w1, c.c1, c.c2);                   // absolute error bound of pi for this pair
            const float t1 = fmaf(pi, c.S1, c.O1h), tau1 = fmaf(epi, c.S1, p.a1.tau);
            r1[r] = t1 + CUTE_MAGIC_F;
            const float d1 = t1 - (r1[r] - CUTE_MAGIC_F);
            const float s2 = fmaxf(fmaf(-pi, pi, q[r]), 1.0e-30f);
            const float w2 = fast_rsqrt(s2);
            const float t2 = fmaf(s2 * w2, c.S2, c.O2h), tau2 = fmaf(w2, fmaf(epi, c.c3, c.tauw2), p.a2.tau);
            r2[r] = t2 + CUTE_MAGIC_F;
            const float d2 = t2 - (r2[r] - CUTE_MAGIC_F);
            vb[r] = fmaxf(fabsf(d1) + tau1, fabsf(d2) + tau2) - 0.5f;
            flag = flag || (vb[r] > 0.f);
        }
    }
    return flag;
}

// ------------------------------------------------------------------------------- one guarded block
// A BLOCK is two j-points against the lane's four i-points (eight pairs per lane, 256 per warp).  The same three
// functions serve the hot loop (compute_tile) and the deferred re-examination of a flagged block (process_entry),
// so that both see bit-identical float32 results.

// Segment code: bits 0-1 / 2-3 / 4-5 = periodic image along x / y / z (0: none, 1: the i-points are one box length BELOW
// the j-points, 2: above); bit 8: same cell row in an auto-correlation (count j > i only).
// The image is applied by subtracting L from the LARGER coordinate, which is exact in float32 (Sterbenz: L/2 <= x <= 2L for a
// point in the top cells of the box): code 2 shifts the i-points (registers, once per segment), code 1 shifts the j-points
// (in the shared-memory tile, once per tile).  Adding L to the smaller coordinate would round at ulp(2L).
__device__ __forceinline__ float image_shift_i(uint32_t code, int axis, float L)
{
    return ((code >> (2 * axis)) & 3u) == 2u ? -L : 0.f;
}
__device__ __forceinline__ float image_shift_j(uint32_t code, int axis, float L)
{
    return ((code >> (2 * axis)) & 3u) == 1u ? -L : 0.f;
}

// The lane's i-points: cell-sorted indices idx0 + 32 r (r < 4) up to i_last, padding points beyond it.  The packed pairs
// are BORN in an aligned register pair by a packed add (of the segment's image shift, or of +0): ptxas otherwise keeps the
// scalars of the LDG.128 results and re-assembles every pair with two MOVs before each packed use inside the loop
// (measured: 18 % of C3's issue slots).
template <int KIND, int FLAGS>
__device__ __forceinline__ void load_ipoints(const GridView &g1, uint32_t idx0, uint32_t i_last, float sx, float sy, float sz,
                                             IPoints &ip, float &xmin, float &xmax)
{
    constexpr bool NEEDLO = (KIND == CUTE_RMU || KIND == CUTE_PISIGMA || ((FLAGS & PK_WEIGHTED) && KIND != CUTE_ANGULAR));
    float bx[R], by[R], bz[R], bw[R], lw[R];
    ip.idx0 = idx0;
    xmin = 3.0e38f; xmax = -3.0e38f;
#pragma unroll
    for (int r = 0; r < R; r++) {
        const uint32_t k = idx0 + 32u * r;
        float4 h = make_float4(kSentinel, kSentinel, kSentinel, 0.f);
        lw[r] = 0.f;
        float wbits = 0.f;
        if (k <= i_last) {
            h = g1.hi[k];
            if (NEEDLO) { const float4 l = g1.lo[k]; lw[r] = l.w; wbits = l.x; }
            xmin = fminf(xmin, h.x); xmax = fmaxf(xmax, h.x);
        }
        bx[r] = h.x; by[r] = h.y; bz[r] = h.z; bw[r] = h.w;
        ip.w[r] = ((FLAGS & PK_WEIGHTED) && KIND != CUTE_ANGULAR) ? wbits : h.w;
    }
    const f32x2 z2 = bc(0.f);
#pragma unroll
    for (int h = 0; h < 2; h++) {
        ip.X0[h] = add2(pk(bx[2 * h], bx[2 * h + 1]), z2); ip.Y0[h] = add2(pk(by[2 * h], by[2 * h + 1]), z2);
        ip.Z0[h] = add2(pk(bz[2 * h], bz[2 * h + 1]), z2);
        ip.W[h] = add2(pk(bw[2 * h], bw[2 * h + 1]), z2);
        ip.LW[h] = add2(pk(lw[2 * h], lw[2 * h + 1]), z2);
        ip.X[h] = add2(ip.X0[h], bc(sx)); ip.Y[h] = add2(ip.Y0[h], bc(sy)); ip.Z[h] = add2(ip.Z0[h], bc(sz));
    }
}

// P2 for a block; returns the lane's smallest q.  masked: auto-correlation, only j > i counts (j = index of the first j-point)
template <int KIND, bool MINIMG>
__device__ __forceinline__ float block_separations(const Consts &c, const IPoints &ip, const float4 pj[2], bool masked, uint32_t j,
                                                   f32x2 q2[2][2], float q[2][R])
{
#pragma unroll
    for (int u = 0; u < 2; u++) {
        separations<KIND, MINIMG>(c, ip, pj[u], q2[u]);
        unpk(q2[u][0], q[u][0], q[u][1]);
        unpk(q2[u][1], q[u][2], q[u][3]);
        if (masked) {
#pragma unroll
            for (int r = 0; r < R; r++) q[u][r] = (j + u > ip.idx0 + 32u * r) ? q[u][r] : 3.0e38f;
            q2[u][0] = pk(q[u][0], q[u][1]);
            q2[u][1] = pk(q[u][2], q[u][3]);
        }
    }
    return fminf(fminf(fminf(q[0][0], q[0][1]), fminf(q[0][2], q[0][3])), fminf(fminf(q[1][0], q[1][1]), fminf(q[1][2], q[1][3])));
}

// RADIAL / always-refine: the pairs that pass the coarse float32 test (bit 4 u + r)
template <int KIND>
__device__ __forceinline__ uint32_t block_candidates(const Consts &c, const IPoints &ip, const float4 pj[2], const float q[2][R])
{
    uint32_t need = 0;
#pragma unroll
    for (int u = 0; u < 2; u++)
#pragma unroll
        for (int r = 0; r < R; r++) {
            bool in = q[u][r] < c.q_hi;
            if (KIND == CUTE_RADIAL) in = in && (fabsf(ip.w[r] - pj[u].w) < c.dz_hi);
            if (in) need |= 1u << (4 * u + r);
        }
    return need;
}

// P3 + the addresses of P4 for a block: addr = shared-memory address of the pair's (clamped) padded histogram cell in
// column hoff; returns "some pair of this lane may be uncertain" (then block_uncertain says which).
// Padded cell (k1 + 1) [* n2p + (k2 + 1)] of column hoff lives at hb + ((bits(r1) [* n2p + bits(r2)]) << sh): the
// magic-number bits are folded into the base (all arithmetic modulo 2^32).
template <int KIND>
__device__ __forceinline__ uint32_t hist_base(const WarpSmem &s, const Consts &c, uint32_t hoff, uint32_t sh)
{
    constexpr uint32_t MB1 = CUTE_MAGIC_BITS - 1u;
    return smem_u32(s.hist + hoff) - ((kind_is_2d(KIND) ? MB1 * (c.n2p + 1u) : MB1) << sh);
}

template <int KIND, bool LOGB, int FLAGS>
__device__ __forceinline__ bool block_bins(const PairParams &p, const Consts &c, const IPoints &ip, const f32x2 q2[2][2], const float q[2][R],
                                           float qm, const float4 pj[2], const float4 pl[2], uint32_t hb, uint32_t sh,
                                           uint32_t addr[2][R], float va[2][R], float vb[2][R])
{
    constexpr bool SIMPLE = (FLAGS & PK_SIMPLE) != 0;
    constexpr bool TWO_D = kind_is_2d(KIND);
    const float bot = CUTE_MAGIC_F - 1.0f;
    float r1[2][R], r2[2][R];
    bool flag[2];
#pragma unroll
    for (int u = 0; u < 2; u++)
        flag[u] = bin_map<KIND, LOGB, SIMPLE>(p, c, ip, q2[u], q[u], pj[u].w, pl[u].w, r1[u], r2[u], va[u], vb[u]);
    // clamp into the padded histogram (no compare, no select)
#pragma unroll
    for (int u = 0; u < 2; u++) {
#pragma unroll
        for (int r = 0; r < R; r++) {
            float a = fminf(r1[u][r], c.top1);
            if (!SIMPLE) a = fmaxf(a, bot);
            uint32_t cell = __float_as_uint(a);
            if (TWO_D) {
                float b = fminf(r2[u][r], c.top2);
                if (!SIMPLE) b = fmaxf(b, bot);
                cell = cell * c.n2p + __float_as_uint(b);
            }
            addr[u][r] = hb + (cell << sh);
        }
    }
    // ANGULAR, log bins: the error of log(theta) grows as 1 / theta.  thr1 is sized for chords above sqrt(q_mid)
    // (nearly every pair); a block that holds a closer pair is examined with the loose threshold of the
    // closest allowed chord, and the pairs are then decided one by one with their own tau = a + b / chord.
    bool near_flag = false;
    if (KIND == CUTE_ANGULAR && LOGB && qm < c.q_mid) {
        float am = 0.f;
#pragma unroll
        for (int u = 0; u < 2; u++)
#pragma unroll
            for (int r = 0; r < R; r++) am = fmaxf(am, va[u][r]);
        near_flag = am > c.thr_mid;
    }
    return flag[0] || flag[1] || near_flag || (KIND == CUTE_ANGULAR && qm < c.q_small);
}

// the in-range pairs of a flagged block whose float32 bin is not certain (bit 4 u + r)
template <int KIND, bool LOGB>
__device__ __forceinline__ uint32_t block_uncertain(const Consts &c, const float q[2][R], const float va[2][R], const float vb[2][R])
{
    uint32_t need = 0;
#pragma unroll
    for (int u = 0; u < 2; u++)
#pragma unroll
        for (int r = 0; r < R; r++) {
            bool unc = va[u][r] > c.thr1 || vb[u][r] > 0.f || (KIND == CUTE_ANGULAR && q[u][r] < c.q_small);
            if (KIND == CUTE_ANGULAR && LOGB)   // the pair's own tau (q_mid > 0 only for log bins)
                unc = q[u][r] < c.q_small || va[u][r] > 0.5f - fmaf(c.tau_b, fast_rsqrt(fmaxf(q[u][r], 1.0e-30f)), c.tau_a);
            if (unc && q[u][r] < c.q_hi) need |= 1u << (4 * u + r);
        }
    return need;
}

// ------------------------------------------------------------------------------- the rare path
// A lane whose block holds a pair that float32 cannot decide does NOT deal with it in the hot loop (measured on C3: the
// per-pair undo-and-queue code ran with one lane of 32 active and took 28 % of all issue slots).  It queues the BLOCK:
// {idx0, first j, meta, i_last}, meta = lane | masked << 5 | (second j is padding) << 6 | image code << 8.  When 32 blocks
// are queued (and before every flush) the warp re-examines them one per lane (examine_entry): the same float32 arithmetic
// on the same inputs gives the same bins and the same uncertain pairs, which go to a second queue {i, j, provisional
// address, weight}.  That queue is emptied 32 pairs at a time, one per lane, all lanes busy (settle_pair): the pair is
// recomputed in float64 with the paper's definition (refine_cell), and if the float64 cell is not the provisional one the
// count is moved.
__device__ __forceinline__ void settle_pair(const PairParams &p, const WarpSmem &s, uint32_t cs, int cell, uint4 pe, int lane)
{
    const uint32_t hb = smem_u32(s.hist);
    const uint32_t col = pe.z ? ((pe.z - hb) >> 2) & ((1u << cs) - 1u) : (uint32_t)lane & ((1u << cs) - 1u);
    const uint32_t na = cell >= 0 ? hb + 4u * ((pad_cell(p, (uint32_t)cell) << cs) + col) : 0u;
    if (na != pe.z) {                      // move the provisional count (same column: exact)
        if (pe.z) red_shared_add(pe.z, 0u - pe.w);
        if (na) red_shared_add(na, pe.w);
    }
}

template <int KIND, bool MINIMG, bool LOGB, int FLAGS>
__device__ __forceinline__ uint32_t examine_entry(const PairParams &p, const WarpSmem &s, const Consts &c, uint4 en, int lane)
{
    constexpr bool ALWAYS = (FLAGS & PK_ALWAYS) != 0 || KIND == CUTE_RADIAL, WEIGHTED = (FLAGS & PK_WEIGHTED) != 0;
    constexpr bool FIXCS = (FLAGS & PK_FIXCS) != 0;
    constexpr bool NEEDLW = (KIND == CUTE_RMU || KIND == CUTE_PISIGMA);
    constexpr bool XYZW = WEIGHTED && KIND != CUTE_ANGULAR;
    const uint32_t idx0 = en.x, j = en.y, meta = en.z, i_last = en.w, code = meta >> 8;
    const bool masked = (meta & 32u) != 0, pad2 = (meta & 64u) != 0;
    const uint32_t cs = FIXCS ? (uint32_t)fixed_colshift(KIND) : (uint32_t)p.colshift, sh = cs + 2u;
    const uint32_t hoff = (meta & 31u) & ((1u << cs) - 1u);
    float sx = 0.f, sy = 0.f, sz = 0.f, jsx = 0.f, jsy = 0.f, jsz = 0.f;
    if (KIND == CUTE_MONOPOLE && !MINIMG && p.periodic) {
        sx = image_shift_i(code, 0, p.Lf); sy = image_shift_i(code, 1, p.Lf); sz = image_shift_i(code, 2, p.Lf);
        jsx = image_shift_j(code, 0, p.Lf); jsy = image_shift_j(code, 1, p.Lf); jsz = image_shift_j(code, 2, p.Lf);
    }
    IPoints ip;
    float xmin, xmax;
    load_ipoints<KIND, FLAGS>(p.g1, idx0, i_last, sx, sy, sz, ip, xmin, xmax);
    float4 pj[2], pl[2];
    uint32_t wj[2];
#pragma unroll
    for (int u = 0; u < 2; u++) {
        pl[u] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (u == 1 && pad2) pj[u] = make_float4(-kSentinel, -kSentinel, -kSentinel, 0.f);
        else {
            pj[u] = p.g2.hi[j + u];
            if (jsx != 0.f || jsy != 0.f || jsz != 0.f) { pj[u].x += jsx; pj[u].y += jsy; pj[u].z += jsz; }
            if (NEEDLW || XYZW) pl[u] = p.g2.lo[j + u];
        }
        wj[u] = WEIGHTED ? __float_as_uint(XYZW ? pl[u].x : pj[u].w) : 1u;
    }
    f32x2 q2[2][2];
    float q[2][R];
    const float qm = block_separations<KIND, MINIMG>(c, ip, pj, masked, j, q2, q);
    uint32_t need, addr[2][R];
    if (ALWAYS) {
        need = block_candidates<KIND>(c, ip, pj, q);
#pragma unroll
        for (int u = 0; u < 2; u++)
#pragma unroll
            for (int r = 0; r < R; r++) addr[u][r] = 0u;
    } else {
        float va[2][R], vb[2][R];
        block_bins<KIND, LOGB, FLAGS>(p, c, ip, q2, q, qm, pj, pl, hist_base<KIND>(s, c, hoff, sh), sh, addr, va, vb);
        need = block_uncertain<KIND, LOGB>(c, q, va, vb);
    }
    uint32_t inline_done = 0;
#pragma unroll
    for (int u = 0; u < 2; u++)
#pragma unroll
        for (int r = 0; r < R; r++) {
            if (!(need & (1u << (4 * u + r)))) continue;
            const uint4 pe = make_uint4(idx0 + 32u * r, j + u, addr[u][r], WEIGHTED ? __float_as_uint(ip.w[r]) * wj[u] : 1u);
            const uint32_t slot = atomicAdd(s.pq_count, 1u);
            if (slot < (uint32_t)kPairCap) s.pq[slot] = pe;
            else {   // queue full (only the test modes that send every pair to float64 get here)
                settle_pair(p, s, cs, refine_cell<KIND>(p, pe.x, pe.y), pe, lane);
                inline_done++;
            }
        }
    return inline_done;
}

// empties the block queue; the pair queue is emptied in groups of 32 (all of it when `all`)
template <int KIND, bool MINIMG, bool LOGB, int FLAGS>
__device__ __noinline__ uint32_t drain_flagged(const PairParams &p, const WarpSmem &s, const Consts &c, int lane, bool all)
{
    const uint32_t cs = (FLAGS & PK_FIXCS) ? (uint32_t)fixed_colshift(KIND) : (uint32_t)p.colshift;
    __syncwarp();
    uint32_t n = *s.rq_count;
    n = n < (uint32_t)kRefineCap ? n : (uint32_t)kRefineCap;
    uint32_t done = 0;
    for (uint32_t e0 = 0; e0 < n || all; e0 += 32) {
        if (e0 + lane < n) done += examine_entry<KIND, MINIMG, LOGB, FLAGS>(p, s, c, s.rq[e0 + lane], lane);
        __syncwarp();
        uint32_t m = *s.pq_count;
        m = m < (uint32_t)kPairCap ? m : (uint32_t)kPairCap;
        const bool last = e0 + 32 >= n;
        while (m >= 32u || (all && last && m > 0u)) {
            const uint32_t take = m < 32u ? m : 32u;
            if ((uint32_t)lane < take) {
                const uint4 pe = s.pq[m - take + lane];
                settle_pair(p, s, cs, refine_cell<KIND>(p, pe.x, pe.y), pe, lane);
            }
            m -= take; done += (uint32_t)lane < take ? 1u : 0u;
        }
        __syncwarp();
        if (lane == 0) *s.pq_count = m;
        __syncwarp();
        if (last) break;
    }
    if (lane == 0) *s.rq_count = 0;
    __syncwarp();
    return done;
}

// block queue full (test modes only): the lane examines its block at once
template <int KIND, bool MINIMG, bool LOGB, int FLAGS>
__device__ __noinline__ uint32_t examine_overflow(const PairParams &p, const WarpSmem &s, const Consts &c, uint4 en, int lane)
{
    return examine_entry<KIND, MINIMG, LOGB, FLAGS>(p, s, c, en, lane);
}

// One tile of j-points against the lane's i-points, two j-points (eight pairs per lane) per guarded block: the pair
// of independent chains is what hides the LDS / MUFU / packed-FMA latencies with four warps per scheduler.
// An odd tile is padded with a sentinel j-point (never in range) by the caller.  meta0 = lane | masked << 5 | code << 8.
template <int KIND, bool MINIMG, bool LOGB, int FLAGS, bool MASK>
__device__ __forceinline__ void compute_tile(const PairParams &p, const WarpSmem &s, const Consts &c, const IPoints &ip,
                                             const float4 *th, const float4 *tl, uint32_t t_cnt, uint32_t j0, uint32_t meta0,
                                             uint32_t i_last, int lane, uint32_t &refined_inline)
{
    constexpr bool FIXCS = (FLAGS & PK_FIXCS) != 0;
    constexpr bool ALWAYS = (FLAGS & PK_ALWAYS) != 0 || KIND == CUTE_RADIAL, WEIGHTED = (FLAGS & PK_WEIGHTED) != 0;
    constexpr bool NEEDLW = (KIND == CUTE_RMU || KIND == CUTE_PISIGMA);
    constexpr bool XYZW = WEIGHTED && KIND != CUTE_ANGULAR;   // weights of xyz catalogues: lo.x
    const uint32_t cs = FIXCS ? (uint32_t)fixed_colshift(KIND) : (uint32_t)p.colshift;
    const uint32_t sh = cs + 2u;
    const uint32_t hoff = (uint32_t)lane & ((1u << cs) - 1u);
    const uint32_t hb = hist_base<KIND>(s, c, hoff, sh);
    const uint32_t cnt2 = (t_cnt + 1u) >> 1;
    // Measured: reading the NEXT block's j-points before this block's guarded bin path is worth 4 % on the short monopole body
    // (with four copies of the body, C5) and 1 % on the angular one (two copies, C2); it costs 8 % on the r-mu body (registers).
    constexpr bool PREFETCH = (KIND == 1 /* CUTE_MONOPOLE */ || KIND == 0 /* CUTE_ANGULAR */) && !WEIGHTED;
    constexpr int kUnroll = KIND == 1 ? 4 : 2;
    float4 nx[2];
    if (PREFETCH) { nx[0] = th[0]; nx[1] = th[1]; }
#pragma unroll kUnroll
    for (uint32_t jp = 0; jp < cnt2; jp++) {
        const uint32_t jj = 2u * jp;
        float4 pj[2], pl[2];
        f32x2 q2[2][2];
        float q[2][R];
        uint32_t wj[2];
#pragma unroll
        for (int u = 0; u < 2; u++) {
            pj[u] = PREFETCH ? nx[u] : th[jj + u];
            pl[u] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (NEEDLW) pl[u].w = tl[jj + u].w;
            wj[u] = WEIGHTED ? __float_as_uint(XYZW ? tl[jj + u].x : pj[u].w) : 1u;
        }
        if (PREFETCH) {
            const uint32_t jn = min(jj + 2u, (uint32_t)kTile - 2u);   // (the last block re-reads inside the tile buffer)
            nx[0] = th[jn]; nx[1] = th[jn + 1];
        }
        const float qm = block_separations<KIND, MINIMG>(c, ip, pj, MASK, j0 + jj, q2, q);
        if (qm < c.q_hi) {
            bool flagged;
            if (ALWAYS) flagged = block_candidates<KIND>(c, ip, pj, q) != 0u;
            else {
                uint32_t addr[2][R];
                float va[2][R], vb[2][R];
                flagged = block_bins<KIND, LOGB, FLAGS>(p, c, ip, q2, q, qm, pj, pl, hb, sh, addr, va, vb);
                // ---- P4: increment (an uncertain pair is counted provisionally like any other)
#pragma unroll
                for (int u = 0; u < 2; u++)
#pragma unroll
                    for (int r = 0; r < R; r++) {
                        if (WEIGHTED) red_shared_add(addr[u][r], __float_as_uint(ip.w[r]) * wj[u]);
                        else red_shared(addr[u][r]);
                    }
            }
            if (flagged) {   // rare: queue the block for re-examination (process_entry)
                const uint4 en = make_uint4(ip.idx0, j0 + jj, meta0 | (jj + 1u >= t_cnt ? 64u : 0u), i_last);
                const uint32_t slot = atomicAdd(s.rq_count, 1u);
                if (slot < (uint32_t)kRefineCap) s.rq[slot] = en;
                else refined_inline += examine_overflow<KIND, MINIMG, LOGB, FLAGS>(p, s, c, en, lane);
            }
        }
    }
}

// ------------------------------------------------------------------------------- G4: neighbour schedule
// Lane `nb` expands neighbour row number nb of the chunk into <= 3 contiguous ranges of the
// cell-sorted j array ("we only correlate C_i with the cells inside a cube of 2k+1 cells per side
// around it", with k = ceil(Rmax/a) -- DESIGN.md reading G3; on the sphere the rows
// and the RA window of the repaired Eq. 16).
__device__ __forceinline__ void expand_row(const PairParams &p, const Chunk &ch, float xmin, float xmax, int nb, int nrows_nb,
                                           uint32_t part, uint4 *out)
{
    uint4 none = make_uint4(0u, 0u, 0u, 0u);
    out[0] = out[1] = out[2] = none;
    if (nb >= nrows_nb || (uint32_t)nb % p.nsplit != part) return;   // this row belongs to another item of the chunk
    const GridView &g = p.g2;
    const int ncx = g.ncx, ncy = g.ncy, ncz = g.ncz;
    const int cy = (int)(ch.row % (uint32_t)ncy), cz = (int)(ch.row / (uint32_t)ncy);
    const int cx0 = (int)(ch.cx01 & 0xffffu), cx1 = (int)(ch.cx01 >> 16);
    int y, z = cz, kx = p.kx;
    uint32_t code = 0;
    bool same_row, wrapx;
    int lo_x = -0x40000000, hi_x = 0x40000000;   // cells reached by [xmin - w, xmax + w] (BOX3D)
    if (p.mode == CUTE_GRID_SPHERE) {
        y = p.g1.row_ylo[cy] + nb;
        if (p.is_auto && y < cy) return;
        kx = p.g1.row_kx[cy];
        same_row = (y == cy);
        wrapx = p.ring != 0;
    } else {
        const int wy = 2 * p.ky + 1;
        const int dy = nb % wy - p.ky, dz = nb / wy - p.kz;
        if (p.is_auto && !(dz > 0 || (dz == 0 && dy >= 0))) return;
        // prune rows that cannot hold a pair within rmax
        const float my = (float)max(0, abs(dy) - 1) * p.ay, mz = (float)max(0, abs(dz) - 1) * p.az;
        if (my * my + mz * mz > p.rmax2) return;
        // ... and trim the row's cells the same way: only x within w = sqrt(rmax^2 - my^2 - mz^2) of the chunk's
        // own x-extent can hold a pair (rmax2 is padded by 0.1 %; trim_pad covers the float32 rounding of the trim)
        const float w = sqrtf(p.rmax2 - (my * my + mz * mz)) + p.trim_pad;
        lo_x = (int)floorf((xmin - w - p.ox) * p.inv_ax);
        hi_x = (int)floorf((xmax + w - p.ox) * p.inv_ax);
        y = cy + dy; z = cz + dz;
        if (p.periodic) {
            if (y >= ncy) { y -= ncy; code |= 2u << 2; } else if (y < 0) { y += ncy; code |= 1u << 2; }
            if (z >= ncz) { z -= ncz; code |= 2u << 4; } else if (z < 0) { z += ncz; code |= 1u << 4; }
        } else if (y < 0 || y >= ncy || z < 0 || z >= ncz) return;
        same_row = (dy == 0 && dz == 0);
        wrapx = p.periodic != 0;
    }
    const uint32_t rb = (uint32_t)(z * ncy + y) * (uint32_t)ncx;
    const uint32_t *cs = g.cell_start + rb;
    int lo = max(cx0 - kx, lo_x), hi = min(cx1 + kx, hi_x);
    const bool self = p.is_auto && same_row;
    if (p.mode == CUTE_GRID_SPHERE && wrapx && hi - lo + 1 >= ncx) { lo = 0; hi = ncx - 1; wrapx = false; }
    const int a0 = max(lo, 0), a1 = min(hi, ncx - 1);
    if (self) {
        const uint32_t je = cs[a1 + 1];
        if (ch.i_begin + 1 < je) out[0] = make_uint4(ch.i_begin + 1, je, code | 0x100u, 0u);
    } else if (a0 <= a1) {
        out[0] = make_uint4(cs[a0], cs[a1 + 1], code, 0u);
    }
    if (wrapx && self && p.mode == CUTE_GRID_SPHERE) {
        // Own row on a ring: a pair is the SAME chord whichever way round the ring it is found, so it must be met
        // exactly once -- by the chunk of its lower sorted index.  Besides the masked direct range above, that chunk
        // takes the cells near the END of the ring that reach its low cells through the seam (all later in sorted
        // order, hence unmasked), clipped to start after the direct range; no chunk looks backwards through the seam.
        // (Decided per pair, not per chunk: a chunk whose window covers the whole ring simply gets the rest of the row.)
        if (lo < 0) {
            const int s0 = max(lo + ncx, a1 + 1);
            if (s0 <= ncx - 1) out[1] = make_uint4(cs[s0], cs[ncx], code, 0u);
        }
    } else if (wrapx) {
        // BOX3D: the wrapped ranges are met through a periodic IMAGE (a different separation; at most one of the
        // images is within rmax because ncx >= 2k+1), so the direct and the wrapped range may hold the same point
        if (lo < 0 && !self) out[1] = make_uint4(cs[max(ncx + lo, 0)], cs[ncx], code | (p.mode == CUTE_GRID_SPHERE ? 0u : 1u), 0u);
        if (hi >= ncx) out[2] = make_uint4(cs[0], cs[min(hi - ncx, ncx - 1) + 1], code | (p.mode == CUTE_GRID_SPHERE ? 0u : 2u), 0u);
    }
}

// ------------------------------------------------------------------------------- the kernel
template <int KIND, bool MINIMG, bool LOGB, int FLAGS>
__global__ void __launch_bounds__(32 * kMaxWarps, 1) pair_kernel(const __grid_constant__ PairParams p)
{
    const Consts cst = load_consts<KIND>(p);
    // lo.w = low part of |x|^2 (r-mu, pi-sigma); lo.x = integer weight of an xyz catalogue
    constexpr bool NEEDLO = (KIND == CUTE_RMU || KIND == CUTE_PISIGMA || ((FLAGS & PK_WEIGHTED) && KIND != CUTE_ANGULAR));
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpSmem s = carve<NEEDLO>(smem_raw + (size_t)warp * p.smem_per_warp);
    if (p.hist_shared) {   // large (2-D) histograms: one copy per CTA, so that more warps fit
        s.hist = reinterpret_cast<uint32_t *>(smem_raw + (size_t)p.warps * p.smem_per_warp);
        for (uint32_t k = threadIdx.x; k < (uint32_t)p.nhist_pad; k += blockDim.x) s.hist[k] = 0;
        __syncthreads();   // the only block-wide barrier of the kernel, before any work
    }

    if (!p.hist_shared)
        for (uint32_t k = lane; k < ((uint32_t)p.nhist_pad << p.colshift); k += 32) s.hist[k] = 0;
    if (lane == 0) {
        for (int k = 0; k < kStages; k++) mbar_init(s.bar[k], 1);
        *s.rq_count = 0; *s.pq_count = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncwarp();

    uint32_t phase = 0;           // bit k = parity to wait for on stage k
    uint32_t stage = 0;
    uint32_t jepoch = 0;
    unsigned long long evaluated = 0, refined = 0, items = 0, flushes = 0;
    uint32_t refined_inline = 0;
    const GridView &g1 = p.g1, &g2 = p.g2;

    for (;;) {
        uint32_t item = 0;
        if (lane == 0) item = atomicAdd(p.queue, 1u) + p.item_begin;
        item = __shfl_sync(0xffffffffu, item, 0);
        if (item >= p.item_end) break;
        items++;
        const uint32_t c = item / p.nsplit, sp = item % p.nsplit;
        const Chunk ch = g1.chunks[c];
        const uint32_t i_last = ch.i_begin + ch.i_count - 1;

        // ---- i-points into registers; x-extent of the chunk (the j-ranges are trimmed to it)
        IPoints ip;
        float xmin, xmax;
        load_ipoints<KIND, FLAGS>(g1, ch.i_begin + lane, i_last, 0.f, 0.f, 0.f, ip, xmin, xmax);
        for (int o = 16; o; o >>= 1) {
            xmin = fminf(xmin, __shfl_xor_sync(0xffffffffu, xmin, o));
            xmax = fmaxf(xmax, __shfl_xor_sync(0xffffffffu, xmax, o));
        }

        if ((FLAGS & PK_WEIGHTED) && p.is_auto && p.self_bin >= 0 && sp == 0) {
            // the w objects of one pixel are w (w - 1) / 2 pairs at zero separation (reading P2)
            unsigned long long self = 0;
#pragma unroll
            for (int r = 0; r < R; r++)
                if ((uint32_t)(lane + 32 * r) < ch.i_count) {
                    const unsigned long long w = __float_as_uint(ip.w[r]);
                    self += w * (w - 1ull) / 2ull;
                }
            for (int o = 16; o; o >>= 1) self += __shfl_xor_sync(0xffffffffu, self, o);
            if (lane == 0 && self) atomicAdd(p.hist + p.self_bin, self);
        }
        // ---- neighbour rows, 32 at a time
        int nrows_nb = 1;
        if (p.mode == CUTE_GRID_BOX3D) nrows_nb = (2 * p.ky + 1) * (2 * p.kz + 1);
        else if (p.mode == CUTE_GRID_SPHERE) {
            const int cy = (int)ch.row;
            nrows_nb = g1.row_yhi[cy] - g1.row_ylo[cy] + 1;
        }
        for (int nb0 = 0; nb0 < nrows_nb; nb0 += kSegBatch) {
            int nslots;
            __syncwarp();
            if (p.mode == CUTE_GRID_NONE) {
                uint32_t jb = sp * p.jsplit, je = min(g2.n, jb + p.jsplit);
                uint32_t code = 0;
                if (p.is_auto) { jb = max(jb, ch.i_begin + 1); code = 0x100u; }
                if (lane == 0) s.segs[0] = make_uint4(jb, max(jb, je), code, 0u);
                nslots = 1;
            } else {
                expand_row(p, ch, xmin, xmax, nb0 + lane, nrows_nb, sp, s.segs + 3 * lane);
                nslots = 3 * min(kSegBatch, nrows_nb - nb0);
            }
            __syncwarp();

            // ---- P1: stream the tiles of this batch, double-buffered
            int pslot = 0; uint32_t pj = 0;           // producer cursor
            uint32_t t_j0 = 0, t_cnt = 0; int t_slot = 0;
            auto next_tile = [&](uint32_t &o_j0, uint32_t &o_cnt, int &o_slot) -> bool {
                while (pslot < nslots) {
                    const uint4 sg = s.segs[pslot];
                    if (pj < sg.x) pj = sg.x;
                    if (pj < sg.y) {
                        o_j0 = pj; o_cnt = min((uint32_t)kTile, sg.y - pj); o_slot = pslot; pj += o_cnt;
                        return true;
                    }
                    pslot++; pj = 0;
                }
                return false;
            };
            auto issue = [&](uint32_t st, uint32_t j0, uint32_t cnt) {
                if (lane == 0) {
                    // (the buffer may hold a sentinel written through the generic proxy: order it before the bulk copy)
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    mbar_expect_tx(s.bar[st], cnt * 16u * (NEEDLO ? 2u : 1u));
                    bulk_g2s(smem_u32(s.thi + st * kTile), g2.hi + j0, cnt * 16u, s.bar[st]);
                    if (NEEDLO) bulk_g2s(smem_u32(s.tlo + st * kTile), g2.lo + j0, cnt * 16u, s.bar[st]);
                }
            };
            bool have = next_tile(t_j0, t_cnt, t_slot);
            if (have) issue(stage, t_j0, t_cnt);
            int active_slot = -1;
            bool seg_mask = false;
            float jsx = 0.f, jsy = 0.f, jsz = 0.f;   // image shift of this segment's j-points
            while (have) {
                uint32_t n_j0 = 0, n_cnt = 0; int n_slot = 0;
                const bool have_next = next_tile(n_j0, n_cnt, n_slot);
                if (have_next) issue(stage ^ 1u, n_j0, n_cnt);
                mbar_wait(s.bar[stage], (phase >> stage) & 1u);
                phase ^= 1u << stage;
                if (t_slot != active_slot) {
                    active_slot = t_slot;
                    const uint32_t code = s.segs[t_slot].z;
                    seg_mask = (code & 0x100u) != 0;
                    if (KIND == CUTE_MONOPOLE && !MINIMG && p.periodic) {
                        const float sx = image_shift_i(code, 0, p.Lf), sy = image_shift_i(code, 1, p.Lf), sz = image_shift_i(code, 2, p.Lf);
                        jsx = image_shift_j(code, 0, p.Lf); jsy = image_shift_j(code, 1, p.Lf); jsz = image_shift_j(code, 2, p.Lf);
#pragma unroll
                        for (int h = 0; h < 2; h++) {
                            ip.X[h] = add2(ip.X0[h], bc(sx)); ip.Y[h] = add2(ip.Y0[h], bc(sy)); ip.Z[h] = add2(ip.Z0[h], bc(sz));
                        }
                    }
                }
                float4 *th = s.thi + stage * kTile, *tl = s.tlo + stage * kTile;
                if (KIND == CUTE_MONOPOLE && !MINIMG && (jsx != 0.f || jsy != 0.f || jsz != 0.f)) {
                    for (uint32_t k = lane; k < t_cnt; k += 32) {   // this tile's j-points take the image (exact, see above)
                        float4 v = th[k];
                        v.x += jsx; v.y += jsy; v.z += jsz;
                        th[k] = v;
                    }
                    __syncwarp();
                }
                if (t_cnt & 1u) {   // odd tile: pad with a sentinel j-point (never in range); the tile has room (t_cnt < kTile)
                    if (lane == 0) {
                        // (-kSentinel: the padding I-points sit at +kSentinel and must not meet the padding j at distance 0)
                        th[t_cnt] = make_float4(-kSentinel, -kSentinel, -kSentinel, 0.f);
                        if (NEEDLO) tl[t_cnt] = make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                    __syncwarp();
                }
                const uint32_t meta0 = (uint32_t)lane | ((s.segs[t_slot].z & 0x3fu) << 8);
                if (seg_mask && t_j0 <= i_last) {
                    compute_tile<KIND, MINIMG, LOGB, FLAGS, true>(p, s, cst, ip, th, tl, t_cnt, t_j0, meta0 | 32u, i_last, lane, refined_inline);
#pragma unroll
                    for (int r = 0; r < R; r++) {
                        if (ip.idx0 + 32u * r <= i_last) {
                            const uint32_t b = max(t_j0, ip.idx0 + 32u * r + 1), e = t_j0 + t_cnt;
                            if (b < e) evaluated += e - b;
                        }
                    }
                } else {
                    compute_tile<KIND, MINIMG, LOGB, FLAGS, false>(p, s, cst, ip, th, tl, t_cnt, t_j0, meta0, i_last, lane, refined_inline);
                    if (lane == 0) evaluated += (unsigned long long)ch.i_count * t_cnt;
                }
                __syncwarp();
                if (*s.rq_count >= 32u) refined += drain_flagged<KIND, MINIMG, LOGB, FLAGS>(p, s, cst, lane, false);
                jepoch += t_cnt;
                if (jepoch >= p.epoch_j) {
                    refined += drain_flagged<KIND, MINIMG, LOGB, FLAGS>(p, s, cst, lane, true);   // (a provisional increment and its correction stay in one epoch)
                    flush_hist(p, s, lane); flushes++; jepoch = 0;
                }
                stage ^= 1u;
                t_j0 = n_j0; t_cnt = n_cnt; t_slot = n_slot; have = have_next;
            }
            if (p.mode == CUTE_GRID_NONE) break;
        }
        if (p.flush_items && (items % p.flush_items) == 0) {
            refined += drain_flagged<KIND, MINIMG, LOGB, FLAGS>(p, s, cst, lane, true);
            flush_hist(p, s, lane); flushes++; jepoch = 0;
        }
    }
    refined += drain_flagged<KIND, MINIMG, LOGB, FLAGS>(p, s, cst, lane, true);
    flush_hist(p, s, lane);
    flushes++;
    refined += refined_inline;
    for (int o = 16; o; o >>= 1) {
        evaluated += __shfl_xor_sync(0xffffffffu, evaluated, o);
        refined += __shfl_xor_sync(0xffffffffu, refined, o);
    }
    if (lane == 0) {
        atomicAdd(p.stats + 0, evaluated);
        atomicAdd(p.stats + 1, refined);
        atomicAdd(p.stats + 2, items);
        atomicAdd(p.stats + 3, flushes);
    }
}

template <int KIND, bool MINIMG, bool LOGB, int FLAGS>
static cudaError_t launch_k(const PairParams &p, int blocks, size_t smem, cudaStream_t s)
{
    auto kern = pair_kernel<KIND, MINIMG, LOGB, FLAGS>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<blocks, 32 * p.warps, smem, s>>>(p);
    note_launches(1);
    return cudaGetLastError();
}

// variant selection shared by the per-kind launchers: `fast` = the kind's default column count and no testing options
template <int KIND, bool MINIMG, bool LOGB>
static cudaError_t launch_t(const PairParams &p, int blocks, size_t smem, cudaStream_t s)
{
    if (p.weighted) {   // integer weights (pixel maps PAPER.md:233, weighted objects): runtime column count
        if constexpr (KIND != CUTE_RADIAL) {
            if (p.always_refine) return launch_k<KIND, MINIMG, LOGB, PK_ALWAYS | PK_WEIGHTED>(p, blocks, smem, s);
            return launch_k<KIND, MINIMG, LOGB, PK_WEIGHTED>(p, blocks, smem, s);
        }
        return cudaErrorInvalidValue;
    }
    // the float64-everything variant (RADIAL, force_refine) is not performance critical: runtime column count
    if (p.always_refine) return launch_k<KIND, MINIMG, LOGB, PK_ALWAYS>(p, blocks, smem, s);
    if constexpr (KIND == CUTE_RADIAL) return cudaErrorInvalidValue;
    else {
        if (p.colshift != fixed_colshift(KIND)) return launch_k<KIND, MINIMG, LOGB, 0>(p, blocks, smem, s);
        if constexpr (!LOGB && KIND != CUTE_ANGULAR) {
            if (p.simple) return launch_k<KIND, MINIMG, LOGB, PK_FIXCS | PK_SIMPLE>(p, blocks, smem, s);
        }
        return launch_k<KIND, MINIMG, LOGB, PK_FIXCS>(p, blocks, smem, s);
    }
}

} // namespace cute
