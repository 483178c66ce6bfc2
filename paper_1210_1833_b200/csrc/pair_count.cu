// pair_count.cu -- the pair kernel.
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
//  * separations in float32: squared comoving distance (monopole, r-mu) or squared chord on hi/lo
//    unit vectors (angular; PAPER.md:233 without the arccos of PAPER.md:235-239).
//  * bin map without division: t = S*g(q)+O with g = MUFU sqrt or log2; floor by a round-down add of
//    1.5*2^23.  The bin is taken from float32 only if floor(t-tau) == floor(t+tau), tau = a bound on
//    the float32 error; otherwise the pair is queued and recomputed in float64 (the definition), so
//    the histogram equals the float64 definition except at float64-rounding distance of an edge.
//  * histogram: per-warp private uint32 copies in shared memory, [bin][column] with 8, 32 or 1 columns per
//    warp (a 2-D histogram too large for that is kept once per CTA), flushed to the uint64 global
//    histogram with 64-bit atomics before 2^32 increments can accumulate and at the end.
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

// shared-memory increment without a return value
__device__ __forceinline__ void red_shared(uint32_t addr)
{
    asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(addr) : "memory");
}

__device__ __forceinline__ void red_shared_add(uint32_t addr, uint32_t v)
{
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

#define CUTE_MAGIC_F 12582912.0f        /* 1.5 * 2^23: adding it with round-down leaves floor(t) in the mantissa */
#define CUTE_MAGIC_BITS 0x4B400000

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
        for (int d = 0; d < nload; d++) v[d] = g.p64[(size_t)d * g.n_pad + idx];
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
    uint2 *rq;             // [kRefineCap] deferred (i, j)
    uint32_t *rq_count;
    uint32_t *hist;        // [nhist << colshift]
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
    s.rq = reinterpret_cast<uint2 *>(ws);
    ws += kRefineCap * 8;
    for (int k = 0; k < kStages; k++) s.bar[k] = smem_u32(ws + 8 * k);
    s.rq_count = reinterpret_cast<uint32_t *>(ws + 8 * kStages);
    ws += 32;
    s.hist = reinterpret_cast<uint32_t *>(ws);
    return s;
}

static inline uint32_t hist_bytes(int nhist, int colshift)
{
    return ((((uint32_t)(nhist + 1) << colshift) * 4 + 15) & ~15u);   // + one dump row
}

static inline uint32_t warp_smem_bytes(bool needlo, int nhist, int colshift, bool shared_hist)
{
    uint32_t b = kStages * kTileBytes * (needlo ? 2 : 1) + kSegSlots * 16 + kRefineCap * 8 + 32;
    if (!shared_hist) b += hist_bytes(nhist, colshift);
    return (b + 127) & ~127u;
}

// P5: add this warp's private histogram to the global uint64 histogram and clear it.
// Lanes own cells; the column index is rotated by the lane so that the 32 reads hit 32 banks.
__device__ __forceinline__ void flush_hist(const PairParams &p, const WarpSmem &s, int lane)
{
    __syncwarp();
    const int C = 1 << p.colshift;
    for (int c = lane; c < p.nhist; c += 32) {
        unsigned long long sum = 0;
        uint32_t *row = s.hist + ((size_t)c << p.colshift);
        for (int k = 0; k < C; k++) {
            int col = (k + lane) & (C - 1);
            if (p.hist_shared) sum += atomicExch(row + col, 0u);   // other warps keep adding: read-and-clear in one step
            else { sum += row[col]; row[col] = 0; }
        }
        if (sum) atomicAdd(p.hist + c, sum);
    }
    __syncwarp();
}

// weight of a pair: w_i * w_j for weighted catalogues (pixel maps; bit patterns in hi.w), else 1
__device__ __forceinline__ uint32_t pair_weight(const PairParams &p, uint32_t i, uint32_t j)
{
    return p.weighted ? __float_as_uint(p.g1.hi[i].w) * __float_as_uint(p.g2.hi[j].w) : 1u;
}

// deferred float64 recomputation of the queued pairs, one per lane
template <int KIND>
__device__ __forceinline__ uint32_t drain_refine(const PairParams &p, const WarpSmem &s, int lane)
{
    __syncwarp();
    uint32_t n = *s.rq_count;
    n = n < (uint32_t)kRefineCap ? n : (uint32_t)kRefineCap;
    uint32_t done = 0;
    for (uint32_t e = lane; e < n; e += 32) {
        uint2 ij = s.rq[e];
        int cell = refine_cell<KIND>(p, ij.x, ij.y);
        if (cell >= 0) atomicAdd(s.hist + (((uint32_t)cell << p.colshift) + (lane & ((1 << p.colshift) - 1))), pair_weight(p, ij.x, ij.y));
        done++;
    }
    __syncwarp();
    if (lane == 0) *s.rq_count = 0;
    __syncwarp();
    return done;
}

// ------------------------------------------------------------------------------- the per-pair body
struct IPoints {           // the R i-points of this lane (float32 fast path)
    float x[R], y[R], z[R], w[R];      // hi (x,y,z already shifted by the segment's periodic image), w
    float lx[R], ly[R], lz[R], lw[R];  // lo parts (ANGULAR) / lo of |x|^2 in lw (RMU)
    uint32_t idx0;                     // cell-sorted index of i-point 0 (point r is idx0 + 32 r)
};

struct Consts {            // loop constants held in registers (not re-read from the constant bank)
    float q_hi, dz_hi, Lf;
    float S1, Oa1, Ob1, c1, c2, c3, c4;
    float O1, tau1, tauw1;     // PISIGMA: the pi axis has a pair-dependent tau too
    float S2, O2, tau2, tauw2;
    uint32_t n1, n2;
};

__device__ __forceinline__ Consts load_consts(const PairParams &p)
{
    Consts c;
    c.q_hi = p.q_hi; c.dz_hi = p.dz_hi; c.Lf = p.Lf;
    c.S1 = p.a1.S; c.Oa1 = p.a1.Oa; c.Ob1 = p.a1.Ob; c.c1 = p.a1.c1; c.c2 = p.a1.c2; c.c3 = p.a1.c3; c.c4 = p.a1.c4;
    c.O1 = p.a1.O; c.tau1 = p.a1.tau; c.tauw1 = p.a1.tau_w;
    c.S2 = p.a2.S; c.O2 = p.a2.O; c.tau2 = p.a2.tau; c.tauw2 = p.a2.tau_w;
    c.n1 = (uint32_t)p.n1; c.n2 = (uint32_t)p.n2;
    return c;
}

// rare path: queue the pairs of this lane whose float32 bin is not certain (bit r of `need`)
template <int KIND>
__device__ __noinline__ void push_refine(const PairParams &p, const WarpSmem &s, uint32_t need, uint32_t idx0, uint32_t j,
                                         uint32_t hoff, uint32_t &refined_inline)
{
    for (int r = 0; r < R; r++) {
        if (!(need & (1u << r))) continue;
        const uint32_t i = idx0 + 32u * r;
        const uint32_t slot = atomicAdd(s.rq_count, 1u);
        if (slot < (uint32_t)kRefineCap) s.rq[slot] = make_uint2(i, j);
        else {
            const int cell = refine_cell<KIND>(p, i, j);
            refined_inline++;
            if (cell >= 0) atomicAdd(s.hist + (((uint32_t)cell << p.colshift) + hoff), pair_weight(p, i, j));
        }
    }
}

struct BinOut { uint32_t kb; uint32_t unsure; bool inr; };   // kb = cell + MAGIC_BITS

// P3: the float32 bin map of one pair.  t = S*g + O is evaluated at t - tau and t + tau and floored by a
// round-down add of 1.5*2^23; `unsure` = floor(t+tau) - floor(t-tau) (+ the same for mu), 0 when the bin is certain.
template <int KIND, bool LOGB>
__device__ __forceinline__ BinOut bin_of(const Consts &c, float q, float wi, float lwi, float wj, float lwj)
{
    BinOut o;
    if (KIND == CUTE_PISIGMA) {
        // pi = |s.l| / |l| (s.l = |x_i|^2 - |x_j|^2 from the hi/lo squares, |l|^2 = 2|x_i|^2 + 2|x_j|^2 - q),
        // sigma = sqrt(q - pi^2)  (Eq. 2); both taus depend on the pair (1/|l| and 1/sigma)
        const float pn = (wi - wj) + (lwi - lwj);
        const float m = fmaf(2.0f, wi + wj, -q);
        const float w1 = fast_rsqrt(fmaxf(m, 1.0e-30f));               // clamps: no NaN/inf, a huge tau instead
        const float pi = fabsf(pn) * w1;
        const float epi = fmaf(w1 * w1, c.c1, c.c2);                   // absolute error bound of pi for this pair
        const float t1 = fmaf(pi, c.S1, c.O1), tau1 = fmaf(epi, c.S1, c.tau1);
        const float fa = __fadd_rd(t1 - tau1, CUTE_MAGIC_F), fb = __fadd_rd(t1 + tau1, CUTE_MAGIC_F);
        const float s2 = fmaxf(fmaf(-pi, pi, q), 1.0e-30f);
        const float w2 = fast_rsqrt(s2);
        const float t2 = fmaf(s2 * w2, c.S2, c.O2), tau2 = fmaf(w2, fmaf(epi, c.c3, c.tauw2), c.tau2);
        const float f2a = __fadd_rd(t2 - tau2, CUTE_MAGIC_F), f2b = __fadd_rd(t2 + tau2, CUTE_MAGIC_F);
        const uint32_t k1 = __float_as_uint(fa) - (uint32_t)CUTE_MAGIC_BITS, k2 = __float_as_uint(f2a) - (uint32_t)CUTE_MAGIC_BITS;
        o.unsure = min((__float_as_uint(fb) - __float_as_uint(fa)) | (__float_as_uint(f2b) - __float_as_uint(f2a)), 15u);
        o.inr = (k1 < c.n1) && (k2 < c.n2);
        o.kb = k1 * c.n2 + k2 + (uint32_t)CUTE_MAGIC_BITS;
        return o;
    }
    if (KIND == CUTE_MONOPOLE && LOGB) {
        // log bins in r: the absolute float32 error e_r of r is an error e_r / r in ln r, so tau depends on the pair:
        // tau = a + b / r  (with a fixed tau sized for r = lo every pair would be uncertain when lo << e_r)
        const float g = fast_lg2(q), w = fast_rsqrt(q);
        const float t = fmaf(g, c.S1, c.O1), tau = fmaf(w, c.tauw1, c.tau1);
        const float fa = __fadd_rd(t - tau, CUTE_MAGIC_F), fb = __fadd_rd(t + tau, CUTE_MAGIC_F);
        o.kb = __float_as_uint(fa);
        o.unsure = min(__float_as_uint(fb) - __float_as_uint(fa), 15u);   // q = 0: NaN bits, clamped into the byte
        o.inr = (o.kb - (uint32_t)CUTE_MAGIC_BITS) < c.n1;
        return o;
    }
    float g;
    if (KIND == CUTE_ANGULAR) {
        const float poly = fmaf(q, fmaf(q, fmaf(q, c.c4, c.c3), c.c2), c.c1);   // cubic fitted on the host over [0, q_hi]
        if (LOGB) g = fast_lg2(q * poly);                      // log2(theta^2), theta^2 = q (1 + q/12 + ...)
        else { const float h = fast_sqrt(q); g = h * poly; }   // theta = c (1 + q/24 + ...)
    } else g = LOGB ? fast_lg2(q) : fast_sqrt(q);
    const float fa = __fadd_rd(fmaf(g, c.S1, c.Oa1), CUTE_MAGIC_F);
    const float fb = __fadd_rd(fmaf(g, c.S1, c.Ob1), CUTE_MAGIC_F);
    o.kb = __float_as_uint(fa);
    o.unsure = __float_as_uint(fb) - __float_as_uint(fa);
    o.inr = (o.kb - (uint32_t)CUTE_MAGIC_BITS) < c.n1;
    if (KIND == CUTE_RMU) {
        // mu = |s.l| / (|s||l|), s.l = |x_i|^2 - |x_j|^2 (hi/lo), |l|^2 = 2|x_i|^2 + 2|x_j|^2 - q
        const float pn = (wi - wj) + (lwi - lwj);
        const float m = fmaf(2.0f, wi + wj, -q);
        // clamped away from 0: q = 0 or |l| = 0 then give a huge but finite w, hence a huge tau2 and an uncertain pair
        const float w = fast_rsqrt(fmaxf(q * m, 1.0e-30f));
        const float t2 = fmaf(fabsf(pn) * w, c.S2, c.O2);
        const float tau2 = fmaf(w * w * q, c.c1, fmaf(w, c.tauw2, c.tau2));   // a + b/(r|l|) + c/|l|^2
        const float f2a = __fadd_rd(t2 - tau2, CUTE_MAGIC_F), f2b = __fadd_rd(t2 + tau2, CUTE_MAGIC_F);
        const uint32_t k2 = __float_as_uint(f2a) - (uint32_t)CUTE_MAGIC_BITS;
        // (clamped: tau2 grows without bound as r -> 0, and the caller keeps one byte per pair)
        o.unsure += min(__float_as_uint(f2b) - __float_as_uint(f2a), 15u);
        o.inr = o.inr && (k2 < c.n2);
        o.kb = (o.kb - (uint32_t)CUTE_MAGIC_BITS) * c.n2 + k2 + (uint32_t)CUTE_MAGIC_BITS;
    }
    return o;
}

// COLS32: one histogram column per lane (compile-time shift); ALWAYS: every candidate pair goes to float64
template <int KIND, bool MINIMG, bool LOGB, bool MASK, bool COLS32, bool ALWAYS, bool WEIGHTED>
__device__ __forceinline__ void compute_tile(const PairParams &p, const WarpSmem &s, const Consts &c, const IPoints &ip,
                                             const float4 *th, const float4 *tl, uint32_t cnt, uint32_t j0,
                                             int lane, uint32_t &refined_inline)
{
    const uint32_t cs = COLS32 ? 5u : (uint32_t)p.colshift;
    const uint32_t hoff = (uint32_t)lane & ((1u << cs) - 1u);
    // bin k of column hoff lives at hbase[(k << cs)]; the magic-number bits are folded into the base
    const uint32_t dump_s = smem_u32(s.hist + (((uint32_t)p.nhist << cs) + hoff));
    const uint32_t hbase_s = smem_u32(s.hist + hoff) - ((uint32_t)CUTE_MAGIC_BITS << (cs + 2u));   // shared-space byte address
#pragma unroll ((KIND == 2 || KIND == 4) ? 2 : 4)   /* RMU, PISIGMA: the bin path is long, 4 copies cost more than they hide */
    for (uint32_t jj = 0; jj < cnt; jj++) {
        const float4 pj = th[jj];
        float4 pl = make_float4(0.f, 0.f, 0.f, 0.f);
        if (KIND == CUTE_ANGULAR) pl = tl[jj];
        float q[R];
#pragma unroll
        for (int r = 0; r < R; r++) {
            float dx = ip.x[r] - pj.x, dy = ip.y[r] - pj.y, dz = ip.z[r] - pj.z;
            if (KIND == CUTE_ANGULAR) {      // hi/lo unit vectors: chord stays precise at tiny theta
                dx += ip.lx[r] - pl.x; dy += ip.ly[r] - pl.y; dz += ip.lz[r] - pl.z;
            }
            if (MINIMG) {                    // periodic brute force: minimum image
                dx = fminf(fabsf(dx), c.Lf - fabsf(dx));
                dy = fminf(fabsf(dy), c.Lf - fabsf(dy));
                dz = fminf(fabsf(dz), c.Lf - fabsf(dz));
            }
            q[r] = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            if (MASK) q[r] = (j0 + jj > ip.idx0 + 32u * r) ? q[r] : 3.0e38f;   // auto-correlation: j > i only
        }
        const float qm = fminf(fminf(q[0], q[1]), fminf(q[2], q[3]));
        if (qm < c.q_hi) {
            float nlo = 0.f;
            if (KIND == CUTE_RMU || KIND == CUTE_PISIGMA) nlo = tl[jj].w;
            if (ALWAYS || KIND == CUTE_RADIAL) {
                uint32_t need = 0;
#pragma unroll
                for (int r = 0; r < R; r++) {
                    bool in = q[r] < c.q_hi;
                    if (KIND == CUTE_RADIAL) in = in && (fabsf(ip.w[r] - pj.w) < c.dz_hi);
                    if (in) need |= 1u << r;
                }
                if (need) push_refine<KIND>(p, s, need, ip.idx0, j0 + jj, hoff, refined_inline);
            } else {
                // acc packs, one byte per pair, floor(t+tau) - floor(t-tau) (>= 0): non-zero <=> some bin is not certain
                uint32_t acc = 0;
#pragma unroll
                for (int r = 0; r < R; r++) {
                    BinOut o = bin_of<KIND, LOGB>(c, q[r], ip.w[r], ip.lw[r], pj.w, nlo);
                    acc += o.unsure << (8 * r);   // one byte per pair (unsure <= 5)
                    // P4: private column, no conflict.  A pair that is out of range or uncertain increments the
                    // column's dump row instead: one SEL + one ATOMS, no branch.
                    const uint32_t addr = (o.unsure == 0u && o.inr) ? hbase_s + (o.kb << (cs + 2u)) : dump_s;
                    if (WEIGHTED) red_shared_add(addr, __float_as_uint(ip.w[r]) * __float_as_uint(pj.w));
                    else red_shared(addr);
                }
                if (acc) {   // rare: queue the uncertain pairs for float64
                    uint32_t need = 0;
#pragma unroll
                    for (int r = 0; r < R; r++)
                        if (((acc >> (8 * r)) & 0xffu) && q[r] < c.q_hi) need |= 1u << r;
                    if (need) push_refine<KIND>(p, s, need, ip.idx0, j0 + jj, hoff, refined_inline);
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------- G4: neighbour schedule
// Segment code: bits 0-1 / 2-3 / 4-5 = periodic image of the i-points along x / y / z
// (0: none, 1: +L, 2: -L); bit 8: same cell row in an auto-correlation (count j > i only).
__device__ __forceinline__ float image_shift(uint32_t code, int axis, float L)
{
    uint32_t c = (code >> (2 * axis)) & 3u;
    return c == 1u ? L : (c == 2u ? -L : 0.f);
}

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
        // own x-extent can hold a pair (rmax2 is padded by 0.1 %, far above the float32 rounding here)
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
template <int KIND, bool MINIMG, bool LOGB, bool COLS32, bool ALWAYS, bool WEIGHTED>
__global__ void __launch_bounds__(32 * kMaxWarps, 1) pair_kernel(const __grid_constant__ PairParams p)
{
    const Consts cst = load_consts(p);
    constexpr bool NEEDLO = (KIND == CUTE_ANGULAR || KIND == CUTE_RMU || KIND == CUTE_PISIGMA);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpSmem s = carve<NEEDLO>(smem_raw + (size_t)warp * p.smem_per_warp);
    if (p.hist_shared) {   // large (2-D) histograms: one copy per CTA, so that more warps fit
        s.hist = reinterpret_cast<uint32_t *>(smem_raw + (size_t)p.warps * p.smem_per_warp);
        for (uint32_t k = threadIdx.x; k < (uint32_t)(p.nhist + 1); k += blockDim.x) s.hist[k] = 0;
        __syncthreads();   // the only block-wide barrier of the kernel, before any work
    }

    if (!p.hist_shared)
        for (uint32_t k = lane; k < ((uint32_t)(p.nhist + 1) << p.colshift); k += 32) s.hist[k] = 0;
    if (lane == 0) {
        for (int k = 0; k < kStages; k++) mbar_init(s.bar[k], 1);
        *s.rq_count = 0;
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

        // ---- i-points into registers
        IPoints ip;
        ip.idx0 = ch.i_begin + lane;
        float bx[R], by[R], bz[R];
#pragma unroll
        for (int r = 0; r < R; r++) {
            const uint32_t k = lane + 32 * r;
            float4 h = make_float4(kSentinel, kSentinel, kSentinel, 0.f), l = make_float4(0.f, 0.f, 0.f, 0.f);
            if (k < ch.i_count) {
                h = g1.hi[ch.i_begin + k];
                if (NEEDLO) l = g1.lo[ch.i_begin + k];
            }
            bx[r] = ip.x[r] = h.x; by[r] = ip.y[r] = h.y; bz[r] = ip.z[r] = h.z; ip.w[r] = h.w;
            ip.lx[r] = l.x; ip.ly[r] = l.y; ip.lz[r] = l.z; ip.lw[r] = l.w;
        }

        if (WEIGHTED && p.is_auto && p.self_bin >= 0 && sp == 0) {
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
        // x-extent of the chunk (the j-ranges are trimmed to it)
        float xmin = 3.0e38f, xmax = -3.0e38f;
#pragma unroll
        for (int r = 0; r < R; r++)
            if ((uint32_t)(lane + 32 * r) < ch.i_count) { xmin = fminf(xmin, bx[r]); xmax = fmaxf(xmax, bx[r]); }
        for (int o = 16; o; o >>= 1) {
            xmin = fminf(xmin, __shfl_xor_sync(0xffffffffu, xmin, o));
            xmax = fmaxf(xmax, __shfl_xor_sync(0xffffffffu, xmax, o));
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
                    mbar_expect_tx(s.bar[st], cnt * 16u * (NEEDLO ? 2u : 1u));
                    bulk_g2s(smem_u32(s.thi + st * kTile), g2.hi + j0, cnt * 16u, s.bar[st]);
                    if (NEEDLO) bulk_g2s(smem_u32(s.tlo + st * kTile), g2.lo + j0, cnt * 16u, s.bar[st]);
                }
            };
            bool have = next_tile(t_j0, t_cnt, t_slot);
            if (have) issue(stage, t_j0, t_cnt);
            int active_slot = -1;
            bool seg_mask = false;
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
                        const float sx = image_shift(code, 0, p.Lf), sy = image_shift(code, 1, p.Lf), sz = image_shift(code, 2, p.Lf);
#pragma unroll
                        for (int r = 0; r < R; r++) { ip.x[r] = bx[r] + sx; ip.y[r] = by[r] + sy; ip.z[r] = bz[r] + sz; }
                    }
                }
                const float4 *th = s.thi + stage * kTile, *tl = s.tlo + stage * kTile;
                if (seg_mask && t_j0 <= i_last) {
                    compute_tile<KIND, MINIMG, LOGB, true, COLS32, ALWAYS, WEIGHTED>(p, s, cst, ip, th, tl, t_cnt, t_j0, lane, refined_inline);
#pragma unroll
                    for (int r = 0; r < R; r++) {
                        if (ip.idx0 + 32u * r <= i_last) {
                            const uint32_t b = max(t_j0, ip.idx0 + 32u * r + 1), e = t_j0 + t_cnt;
                            if (b < e) evaluated += e - b;
                        }
                    }
                } else {
                    compute_tile<KIND, MINIMG, LOGB, false, COLS32, ALWAYS, WEIGHTED>(p, s, cst, ip, th, tl, t_cnt, t_j0, lane, refined_inline);
                    if (lane == 0) evaluated += (unsigned long long)ch.i_count * t_cnt;
                }
                __syncwarp();
                if (*s.rq_count >= 32u) refined += drain_refine<KIND>(p, s, lane);
                jepoch += t_cnt;
                if (jepoch >= p.epoch_j) { flush_hist(p, s, lane); flushes++; jepoch = 0; }
                stage ^= 1u;
                t_j0 = n_j0; t_cnt = n_cnt; t_slot = n_slot; have = have_next;
            }
            if (p.mode == CUTE_GRID_NONE) break;
        }
        if (p.flush_items && (items % p.flush_items) == 0) {
            refined += drain_refine<KIND>(p, s, lane);
            flush_hist(p, s, lane); flushes++; jepoch = 0;
        }
    }
    refined += drain_refine<KIND>(p, s, lane);
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

// ------------------------------------------------------------------------------- host side
static constexpr int kSmemBudget = 227 * 1024;

int plan_pair_kernel(PairParams &p, int want_warps, int want_cols)
{
    // Warps hide the latency of the dependent MUFU/FFMA chains and ncu shows throughput growing with the warp
    // count up to 16, while the number of private histogram columns (32, 8, 1) makes no measurable difference
    // (ATOMS.POPC.INC merges lanes that hit one address): default = 8 columns, as many warps as fit.  A histogram
    // too large for 8 warps with private copies (the 2-D kinds) becomes ONE copy per CTA shared by all its warps.
    const bool needlo = (p.kind == CUTE_ANGULAR || p.kind == CUTE_RMU || p.kind == CUTE_PISIGMA);
    p.hist_shared = 0;
    const int clist[] = {3, 0, 5};
    for (int ci = 0; ci < 3; ci++) {
        if (want_cols > 0 && (1 << clist[ci]) != want_cols) continue;
        const uint32_t per = warp_smem_bytes(needlo, p.nhist, clist[ci], false);
        int w = (int)((size_t)kSmemBudget / per);
        if (w > kMaxWarps) w = kMaxWarps;
        if (want_warps > 0) { if (want_warps > w) continue; w = want_warps; }
        else if (want_cols <= 0 && w < kMaxWarps && clist[ci] != 5) continue;   // would cost warps: share instead
        else if (want_cols <= 0 && clist[ci] == 5) continue;
        if (w < 1) continue;
        p.colshift = clist[ci]; p.warps = w; p.smem_per_warp = per;
        return (int)(per * (uint32_t)w);
    }
    if (want_cols > 0) return -1;
    {   // shared copy, one column
        const uint32_t per = warp_smem_bytes(needlo, p.nhist, 0, true), hb = hist_bytes(p.nhist, 0);
        if ((size_t)hb + per > (size_t)kSmemBudget) return -1;
        int w = (int)(((size_t)kSmemBudget - hb) / per);
        if (w > kMaxWarps) w = kMaxWarps;
        if (want_warps > 0) { if (want_warps > w) return -1; w = want_warps; }
        p.hist_shared = 1; p.colshift = 0; p.warps = w; p.smem_per_warp = per;
        return (int)(per * (uint32_t)w + hb);
    }
}

template <int KIND, bool MINIMG, bool LOGB, bool COLS32, bool ALWAYS, bool WEIGHTED>
static cudaError_t launch_k(const PairParams &p, int blocks, cudaStream_t s)
{
    const size_t smem = (size_t)p.smem_per_warp * p.warps + (p.hist_shared ? hist_bytes(p.nhist, 0) : 0);
    auto kern = pair_kernel<KIND, MINIMG, LOGB, COLS32, ALWAYS, WEIGHTED>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<blocks, 32 * p.warps, smem, s>>>(p);
    note_launches(1);
    return cudaGetLastError();
}

template <int KIND, bool MINIMG, bool LOGB>
static cudaError_t launch_t(const PairParams &p, int blocks, cudaStream_t s)
{
    if (p.weighted) {   // pixel maps: ANGULAR only, runtime column count
        if constexpr (KIND == CUTE_ANGULAR) {
            if (p.always_refine) return launch_k<KIND, MINIMG, LOGB, false, true, true>(p, blocks, s);
            return launch_k<KIND, MINIMG, LOGB, false, false, true>(p, blocks, s);
        }
        return cudaErrorInvalidValue;
    }
    // the float64-everything variant (RADIAL, force_refine) is not performance critical: one column layout
    if (p.always_refine) return launch_k<KIND, MINIMG, LOGB, false, true, false>(p, blocks, s);
    if (KIND == CUTE_RADIAL) return cudaErrorInvalidValue;
    return p.colshift == 5 ? launch_k<KIND, MINIMG, LOGB, true, false, false>(p, blocks, s)
                           : launch_k<KIND, MINIMG, LOGB, false, false, false>(p, blocks, s);
}

cudaError_t launch_pair_kernel(const PairParams &p, int blocks, cudaStream_t s)
{
    const bool minimg = (p.kind == CUTE_MONOPOLE && p.mode == CUTE_GRID_NONE && p.L > 0.0);
    const bool lg = p.logbins != 0;
    switch (p.kind) {
    case CUTE_MONOPOLE:
        if (minimg) return lg ? launch_t<CUTE_MONOPOLE, true, true>(p, blocks, s) : launch_t<CUTE_MONOPOLE, true, false>(p, blocks, s);
        return lg ? launch_t<CUTE_MONOPOLE, false, true>(p, blocks, s) : launch_t<CUTE_MONOPOLE, false, false>(p, blocks, s);
    case CUTE_ANGULAR:
        return lg ? launch_t<CUTE_ANGULAR, false, true>(p, blocks, s) : launch_t<CUTE_ANGULAR, false, false>(p, blocks, s);
    case CUTE_RMU:
        return launch_t<CUTE_RMU, false, false>(p, blocks, s);
    case CUTE_RADIAL:
        return launch_t<CUTE_RADIAL, false, false>(p, blocks, s);
    case CUTE_PISIGMA:
        return launch_t<CUTE_PISIGMA, false, false>(p, blocks, s);
    }
    return cudaErrorInvalidValue;
}

} // namespace cute
