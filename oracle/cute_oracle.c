/*
 * cute_oracle.c -- the ORACLE for the CUTE pair-counting hot path (arXiv 1210.1833).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or helper with the CUDA path under paper_1210_1833_b200/csrc and
 * neither includes the other.
 *
 * What it is: the plain definition, written out.  The method (cell lists, pixels, GPU
 * histograms) reaches EXACTLY the result of the two nested loops of the serial algorithm
 *   "one loop over each catalog and performing 3 operations in each iteration: calculating
 *    the distance between each pair of objects, determining the bin corresponding to that
 *    distance and increasing the histogram count on that bin"     (sec. III.A)
 * i.e. Eq. 11   N_p(r) dr = sum_i sum_{j != i} Theta(r-dr/2 < |x_i-x_j| < r+dr/2),
 * so the oracle is those two loops in IEEE float64 (compile with -ffp-contract=off, never
 * -ffast-math).  Parallelised exactly like the paper's OpenMP version (PAPER.md:126-151,
 * sec. III.B.1): one private histogram per thread, outer loop split over threads, partial
 * histograms added under `omp critical`.
 *
 * Readings of the paper where it is silent:
 *   S1  bins are half-open [e_k, e_{k+1}); out-of-range pairs are dropped; the edge ARRAY is the
 *       sole authority (arithmetic guess + fix-up compare);
 *   S2  auto-correlation counts UNORDERED pairs i<j, cross-correlation all N1*N2 pairs (forced
 *       by the coefficients of Eq. 15);
 *   S4  self pairs skipped; distinct coincident points are a pair with r = 0;
 *   S5  mu uses the mid-point line of sight l = x_i + x_j (pinned by Eq. 9);
 *   S6  mu = |cos|;  mu >= 1 goes to the last mu bin when hi2 >= 1; r = 0 => mu := 0;
 *   P1  pixelised catalogues: pixels with constant limits in (sin dec, RA); a pixel is
 *       represented by its centre in those coordinates and weighted by its number of objects;
 *   P2  weighted pairs: pair (i,j) counts w_i w_j; in an auto-correlation the w_i objects of one pixel count as
 *       w_i (w_i - 1)/2 pairs at zero separation, so that weights are exactly equivalent to repeated objects;
 *   N1  (pi,sigma): pi = r mu with the mu of S5/S6, sigma = sqrt(max(0, r^2 - pi^2)) (Eq. 2); first
 *       variable pi (major index), second sigma;
 *   S7  radial: zbar = (z_i+z_j)/2 (major index), dz = |z_i - z_j|;
 *   S8  radial aperture test is strict: theta < aperture;
 *   S12 the angular distance measure is theta itself, computed as
 *       theta = 2 asin(|n_i - n_j| / 2), which equals arccos(n_i . n_j) (Eq. 7)
 *       but stays accurate for tiny theta;
 *   periodic box: minimum image d -= L*nearbyint(d/L).
 *
 * Besides the histogram the oracle reports, per pair, whether a binned variable lies within
 * relative 2^-20 of a bin edge (or of the radial aperture); `amb_cell[c]` counts, for every
 * histogram cell c (and one extra "virtual" out-of-range cell at index ncell), the flagged pairs
 * that could land in c if the flagged variable(s) crossed their edge.  The parity rule of the
 * north star ("GPU histograms must match the oracle exactly ... except for pairs the oracle
 * flags as lying within relative 2^-20 of a bin edge") is then
 *      |gpu[c] - oracle[c]| <= amb_cell[c]  for every c,   |sum gpu - sum oracle| <= amb_cell[ncell].
 *
 * Pins: tests/test_oracle_pins.py (V1..V11 of SURVEY.md 8(c), the 2-D composition of amb_cell, the density-grid
 * functions); no function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <omp.h>

#define ORC_ANGULAR 0
#define ORC_MONOPOLE 1
#define ORC_RMU 2
#define ORC_RADIAL 3
#define ORC_PISIGMA 4 /* xi(pi,sigma): v = (pi, sigma), pi = r mu, sigma = sqrt(r^2 - pi^2), Eq. 2 */

#define ORC_OK 0
#define ORC_EINVAL (-1)
#define ORC_ENOMEM (-2)

static const double ORC_PI = 3.14159265358979323846264338327950288;
static const double ORC_BAND = 1.0 / 1048576.0; /* 2^-20 */

typedef struct {
    int n1; double lo1, hi1; int log1;   /* first variable: theta [rad] | r | r | zbar            */
    int n2; double lo2, hi2;             /* second variable (n2 = 0: none): mu | dz ; always linear */
    double aperture;                     /* RADIAL only: maximum angular separation [rad]          */
    double box_L;                        /* > 0: periodic box side, minimum image (MONOPOLE only)  */
} orc_bins;

/* ------------------------------------------------------------------ edges (S1) */
/* linear e_k = lo + (hi-lo) k/n ; log e_k = exp(log lo + k (log hi - log lo)/n); ends forced exact */
int orc_edges(const orc_bins *b, int axis, double *e)
{
    int n = axis == 0 ? b->n1 : b->n2;
    double lo = axis == 0 ? b->lo1 : b->lo2, hi = axis == 0 ? b->hi1 : b->hi2;
    int lg = axis == 0 ? b->log1 : 0;
    if (n < 1 || !(lo < hi) || (lg && !(lo > 0.0))) return ORC_EINVAL;
    for (int k = 0; k <= n; k++) {
        if (lg) e[k] = exp(log(lo) + (double)k * (log(hi) - log(lo)) / (double)n);
        else e[k] = lo + (hi - lo) * (double)k / (double)n;
    }
    e[0] = lo; e[n] = hi;
    return ORC_OK;
}

typedef struct {
    int n; int lg; int closed_top; double lo, hi; const double *e;
} axis_t;

/* half-open bin of v, -1 if outside; arithmetic guess then fix-up against the edge array */
static int find_bin(const axis_t *a, double v)
{
    int n = a->n;
    if (!(v >= a->e[0])) return -1;
    if (!(v < a->e[n])) return (a->closed_top && v == a->e[n]) ? n - 1 : -1;
    double g = a->lg ? (double)n * log(v / a->lo) / log(a->hi / a->lo) : (double)n * (v - a->lo) / (a->hi - a->lo);
    int k = (int)floor(g);
    if (k < 0) k = 0;
    if (k > n - 1) k = n - 1;
    while (k > 0 && v < a->e[k]) k--;
    while (k < n - 1 && v >= a->e[k + 1]) k++;
    return k;
}

/* nearest edge index (0..n) of v given its bin k (-1 outside) */
static int nearest_edge(const axis_t *a, double v, int k)
{
    if (k < 0) return (v < a->e[0]) ? 0 : a->n;
    return (v - a->e[k] <= a->e[k + 1] - v) ? k : k + 1;
}

/* is v within relative 2^-20 of edge j; if so *other = the bin on the other side of that edge */
static int edge_flag(const axis_t *a, double v, int k, int *edge, int *other)
{
    int j = nearest_edge(a, v, k);
    *edge = j;
    if (fabs(v - a->e[j]) <= ORC_BAND * fabs(a->e[j])) {
        int lower = j - 1, upper = (j < a->n) ? j : -1; /* bins below / above edge j */
        if (k < 0) *other = (j == 0) ? upper : lower;      /* v outside: the other side is the end bin */
        else *other = (k == lower) ? upper : lower;
        return 1;
    }
    return 0;
}

/* ------------------------------------------------------------------ per-point preparation */
typedef struct {
    int64_t n;
    const double *a, *b, *c; /* inputs: xyz | ra,dec[,z] */
    const uint32_t *w;       /* optional integer weights (NULL = 1): objects per pixel */
    double *ux, *uy, *uz;    /* unit vectors (ANGULAR/RADIAL), owned */
} cat_t;

static int prep_cat(int kind, cat_t *c)
{
    c->ux = c->uy = c->uz = NULL;
    if (kind == ORC_ANGULAR || kind == ORC_RADIAL) {
        size_t n = (size_t)(c->n > 0 ? c->n : 1);
        c->ux = (double *)malloc(n * sizeof(double));
        c->uy = (double *)malloc(n * sizeof(double));
        c->uz = (double *)malloc(n * sizeof(double));
        if (!c->ux || !c->uy || !c->uz) return ORC_ENOMEM;
        /* "projects all objects in the catalog into the unit sphere" */
        for (int64_t i = 0; i < c->n; i++) {
            double al = c->a[i] * (ORC_PI / 180.0), de = c->b[i] * (ORC_PI / 180.0);
            double cd = cos(de);
            c->ux[i] = cd * cos(al);
            c->uy[i] = cd * sin(al);
            c->uz[i] = sin(de);
        }
    }
    return ORC_OK;
}

static void free_cat(cat_t *c) { free(c->ux); free(c->uy); free(c->uz); c->ux = c->uy = c->uz = NULL; }

/* ------------------------------------------------------------------ the pair body */
typedef struct {
    int kind;
    axis_t ax1, ax2;
    int n2eff;       /* max(n2,1) */
    int ncell;       /* n1 * n2eff */
    double L;        /* periodic side or 0 */
    double aperture; /* rad */
    uint64_t *hist;  /* ncell      */
    uint64_t *amb_cell; /* ncell+1 */
    uint64_t *amb_e1;   /* n1+1    */
    uint64_t *amb_e2;   /* n2+2 : edges of variable 2, last = aperture flags */
    uint64_t npairs;    /* pairs evaluated */
} acc_t;

static inline double theta_of(const cat_t *c1, int64_t i, const cat_t *c2, int64_t j)
{
    double dx = c1->ux[i] - c2->ux[j], dy = c1->uy[i] - c2->uy[j], dz = c1->uz[i] - c2->uz[j];
    double h = 0.5 * sqrt(dx * dx + dy * dy + dz * dz);
    if (h > 1.0) h = 1.0;
    return 2.0 * asin(h);
}

/* wp = weight of the pair: w_i * w_j ("weighting each of them by the number of objects that fall inside it",
 * PAPER.md:233), or w_i (w_i - 1) / 2 for the objects of one pixel among themselves (j == i, zero separation) */
static inline void pair_eval(acc_t *A, const cat_t *c1, int64_t i, const cat_t *c2, int64_t j, uint64_t wp)
{
    double v1, v2 = 0.0;
    int in_ap = 1, ap_flag = 0;
    A->npairs++;
    switch (A->kind) {
    case ORC_MONOPOLE: {
        double dx = c1->a[i] - c2->a[j], dy = c1->b[i] - c2->b[j], dz = c1->c[i] - c2->c[j];
        if (A->L > 0.0) { /* periodic "wrapped around" sphere */
            dx -= A->L * nearbyint(dx / A->L);
            dy -= A->L * nearbyint(dy / A->L);
            dz -= A->L * nearbyint(dz / A->L);
        }
        v1 = sqrt(dx * dx + dy * dy + dz * dz);
    } break;
    case ORC_ANGULAR:
        v1 = theta_of(c1, i, c2, j);
        break;
    case ORC_RMU: {
        double sx = c1->a[i] - c2->a[j], sy = c1->b[i] - c2->b[j], sz = c1->c[i] - c2->c[j];
        double lx = c1->a[i] + c2->a[j], ly = c1->b[i] + c2->b[j], lz = c1->c[i] + c2->c[j];
        double r = sqrt(sx * sx + sy * sy + sz * sz), l = sqrt(lx * lx + ly * ly + lz * lz);
        double mu = 0.0;
        if (r > 0.0 && l > 0.0) mu = fabs(sx * lx + sy * ly + sz * lz) / (r * l);
        if (mu > 1.0) mu = 1.0;
        v1 = r; v2 = mu;
    } break;
    case ORC_PISIGMA: { /* Eq. 2: pi = r mu (along the mid-point line of sight), sigma = sqrt(r^2 - pi^2) */
        double sx = c1->a[i] - c2->a[j], sy = c1->b[i] - c2->b[j], sz = c1->c[i] - c2->c[j];
        double lx = c1->a[i] + c2->a[j], ly = c1->b[i] + c2->b[j], lz = c1->c[i] + c2->c[j];
        double r = sqrt(sx * sx + sy * sy + sz * sz), l = sqrt(lx * lx + ly * ly + lz * lz);
        double mu = 0.0;
        if (r > 0.0 && l > 0.0) mu = fabs(sx * lx + sy * ly + sz * lz) / (r * l);
        if (mu > 1.0) mu = 1.0;
        double pi = r * mu, s2 = r * r - pi * pi;
        v1 = pi; v2 = s2 > 0.0 ? sqrt(s2) : 0.0;
    } break;
    default: { /* ORC_RADIAL */
        double th = theta_of(c1, i, c2, j);
        in_ap = th < A->aperture;
        ap_flag = fabs(th - A->aperture) <= ORC_BAND * A->aperture;
        if (!in_ap && !ap_flag) return;
        v1 = 0.5 * (c1->c[i] + c2->c[j]);
        v2 = fabs(c1->c[i] - c2->c[j]);
    } break;
    }
    int k1 = find_bin(&A->ax1, v1), k2 = 0;
    int two = A->ax2.n > 0;
    if (two) k2 = find_bin(&A->ax2, v2);
    int cell = (in_ap && k1 >= 0 && k2 >= 0) ? k1 * A->n2eff + k2 : -1;
    if (cell >= 0) A->hist[cell] += wp;
    /* ambiguity flags */
    int e1, o1 = 0, e2 = 0, o2 = 0;
    int f1 = edge_flag(&A->ax1, v1, k1, &e1, &o1);
    int f2 = two ? edge_flag(&A->ax2, v2, k2, &e2, &o2) : 0;
    if (!(f1 || f2 || ap_flag)) return;
    if (f1) A->amb_e1[e1] += wp;
    if (f2) A->amb_e2[e2] += wp;
    if (ap_flag) A->amb_e2[A->ax2.n + 1] += wp;
    /* every cell the pair could land in: product of candidate bins, "out" -> virtual cell */
    int c1s[2] = {k1, o1}, c2s[2] = {k2, o2};
    int n1c = f1 ? 2 : 1, n2c = f2 ? 2 : 1, nap = ap_flag ? 2 : 1;
    int seen[9]; int ns = 0;
    for (int p = 0; p < nap; p++)
        for (int x = 0; x < n1c; x++)
            for (int y = 0; y < n2c; y++) {
                int inap = (nap == 2) ? p : in_ap;
                int kk1 = c1s[x], kk2 = c2s[y];
                int c = (inap && kk1 >= 0 && kk2 >= 0) ? kk1 * A->n2eff + kk2 : A->ncell;
                int dup = 0;
                for (int s = 0; s < ns; s++) if (seen[s] == c) dup = 1;
                if (!dup) { seen[ns++] = c; A->amb_cell[c] += wp; }
            }
}

static int acc_init(acc_t *A, int kind, const orc_bins *b, const double *e1, const double *e2)
{
    memset(A, 0, sizeof(*A));
    A->kind = kind;
    A->ax1.n = b->n1; A->ax1.lg = b->log1; A->ax1.lo = b->lo1; A->ax1.hi = b->hi1; A->ax1.e = e1; A->ax1.closed_top = 0;
    A->ax2.n = b->n2; A->ax2.lg = 0; A->ax2.lo = b->lo2; A->ax2.hi = b->hi2; A->ax2.e = e2;
    A->ax2.closed_top = (kind == ORC_RMU && b->n2 > 0 && b->hi2 >= 1.0); /* S6 */
    A->n2eff = b->n2 > 0 ? b->n2 : 1;
    A->ncell = b->n1 * A->n2eff;
    A->L = (kind == ORC_MONOPOLE) ? b->box_L : 0.0;
    A->aperture = b->aperture;
    A->hist = (uint64_t *)calloc((size_t)A->ncell, 8);
    A->amb_cell = (uint64_t *)calloc((size_t)A->ncell + 1, 8);
    A->amb_e1 = (uint64_t *)calloc((size_t)b->n1 + 1, 8);
    A->amb_e2 = (uint64_t *)calloc((size_t)b->n2 + 2, 8);
    if (!A->hist || !A->amb_cell || !A->amb_e1 || !A->amb_e2) return ORC_ENOMEM;
    return ORC_OK;
}
static void acc_free(acc_t *A) { free(A->hist); free(A->amb_cell); free(A->amb_e1); free(A->amb_e2); }

static int check_args(int kind, const orc_bins *b, int auto_)
{
    if (kind < 0 || kind > 4 || b->n1 < 1 || !(b->lo1 < b->hi1)) return ORC_EINVAL;
    if (b->log1 && !(b->lo1 > 0.0)) return ORC_EINVAL;
    if ((kind == ORC_RMU || kind == ORC_RADIAL || kind == ORC_PISIGMA) && (b->n2 < 1 || !(b->lo2 < b->hi2))) return ORC_EINVAL;
    if ((kind == ORC_ANGULAR || kind == ORC_MONOPOLE) && b->n2 != 0) return ORC_EINVAL;
    if (kind == ORC_RADIAL && !(b->aperture > 0.0)) return ORC_EINVAL;
    if (kind == ORC_MONOPOLE && b->box_L > 0.0 && b->hi1 > 0.5 * b->box_L) return ORC_EINVAL; /* S13 */
    (void)auto_;
    return ORC_OK;
}

/* ------------------------------------------------------------------ the oracle's own cell lists (mode "celled", O3) */
typedef struct {
    int kind3d;                /* 1: 3-D cells, 0: declination bands */
    int nc[3]; double org[3], inv[3];
    int64_t *start;            /* ncell+1 */
    int64_t *idx;              /* point indices sorted by cell (3-D) or by (band, RA) */
    int periodic;
    /* bands */
    int nband; double band_h;  /* band height in degrees of declination */
    double *ra_sorted;         /* RA of idx[] */
} cells_t;

static int cmp_ra(const void *p, const void *q)
{
    double a = ((const double *)p)[0], b = ((const double *)q)[0];
    return (a > b) - (a < b);
}

static int build_cells3d(cells_t *C, const cat_t *c, double rmax, double L)
{
    double lo[3], hi[3];
    const double *X[3] = {c->a, c->b, c->c};
    memset(C, 0, sizeof(*C));
    C->kind3d = 1; C->periodic = L > 0.0;
    for (int d = 0; d < 3; d++) {
        if (L > 0.0) { lo[d] = 0.0; hi[d] = L; }
        else {
            lo[d] = 1e300; hi[d] = -1e300;
            for (int64_t i = 0; i < c->n; i++) { if (X[d][i] < lo[d]) lo[d] = X[d][i]; if (X[d][i] > hi[d]) hi[d] = X[d][i]; }
            if (c->n == 0) { lo[d] = 0; hi[d] = 1; }
        }
        double ext = hi[d] - lo[d];
        int n = (int)floor(ext / rmax);      /* cell side >= rmax */
        if (n < 1) n = 1;
        if (n > 200) n = 200;
        C->nc[d] = n; C->org[d] = lo[d]; C->inv[d] = (ext > 0.0) ? (double)n / ext : 0.0;
    }
    int64_t ncell = (int64_t)C->nc[0] * C->nc[1] * C->nc[2];
    C->start = (int64_t *)calloc((size_t)ncell + 1, sizeof(int64_t));
    C->idx = (int64_t *)malloc((size_t)(c->n > 0 ? c->n : 1) * sizeof(int64_t));
    int64_t *cid = (int64_t *)malloc((size_t)(c->n > 0 ? c->n : 1) * sizeof(int64_t));
    if (!C->start || !C->idx || !cid) return ORC_ENOMEM;
    for (int64_t i = 0; i < c->n; i++) {
        int64_t k[3];
        for (int d = 0; d < 3; d++) {
            k[d] = (int64_t)floor((X[d][i] - C->org[d]) * C->inv[d]);
            if (k[d] < 0) k[d] = 0;
            if (k[d] >= C->nc[d]) k[d] = C->nc[d] - 1;
        }
        cid[i] = (k[2] * C->nc[1] + k[1]) * C->nc[0] + k[0];
        C->start[cid[i] + 1]++;
    }
    for (int64_t k = 0; k < ncell; k++) C->start[k + 1] += C->start[k];
    int64_t *cur = (int64_t *)malloc((size_t)ncell * sizeof(int64_t));
    if (!cur) return ORC_ENOMEM;
    memcpy(cur, C->start, (size_t)ncell * sizeof(int64_t));
    for (int64_t i = 0; i < c->n; i++) C->idx[cur[cid[i]]++] = i;
    free(cur); free(cid);
    return ORC_OK;
}

static int build_bands(cells_t *C, const cat_t *c, double thmax_rad)
{
    memset(C, 0, sizeof(*C));
    double h = thmax_rad * 180.0 / ORC_PI;  /* band height >= theta_max */
    int nb = (int)floor(180.0 / h);
    if (nb < 1) nb = 1;
    if (nb > 20000) nb = 20000;
    C->nband = nb; C->band_h = 180.0 / nb;
    C->start = (int64_t *)calloc((size_t)nb + 1, sizeof(int64_t));
    size_t n = (size_t)(c->n > 0 ? c->n : 1);
    C->idx = (int64_t *)malloc(n * sizeof(int64_t));
    C->ra_sorted = (double *)malloc(n * sizeof(double));
    double *tmp = (double *)malloc(n * 2 * sizeof(double));
    int *bd = (int *)malloc(n * sizeof(int));
    if (!C->start || !C->idx || !C->ra_sorted || !tmp || !bd) return ORC_ENOMEM;
    for (int64_t i = 0; i < c->n; i++) {
        int b = (int)floor((c->b[i] + 90.0) / C->band_h);
        if (b < 0) b = 0;
        if (b >= nb) b = nb - 1;
        bd[i] = b; C->start[b + 1]++;
    }
    for (int b = 0; b < nb; b++) C->start[b + 1] += C->start[b];
    int64_t *cur = (int64_t *)malloc((size_t)nb * sizeof(int64_t));
    if (!cur) return ORC_ENOMEM;
    memcpy(cur, C->start, (size_t)nb * sizeof(int64_t));
    for (int64_t i = 0; i < c->n; i++) {
        int64_t s = cur[bd[i]]++;
        double ra = fmod(c->a[i], 360.0); if (ra < 0) ra += 360.0;
        tmp[2 * s] = ra; tmp[2 * s + 1] = (double)i;
    }
    for (int b = 0; b < nb; b++)
        qsort(tmp + 2 * C->start[b], (size_t)(C->start[b + 1] - C->start[b]), 2 * sizeof(double), cmp_ra);
    for (int64_t s = 0; s < c->n; s++) { C->ra_sorted[s] = tmp[2 * s]; C->idx[s] = (int64_t)tmp[2 * s + 1]; }
    free(cur); free(tmp); free(bd);
    return ORC_OK;
}

static void free_cells(cells_t *C) { free(C->start); free(C->idx); free(C->ra_sorted); }

static int64_t lower_bound_d(const double *a, int64_t lo, int64_t hi, double v)
{
    while (lo < hi) { int64_t m = lo + (hi - lo) / 2; if (a[m] < v) lo = m + 1; else hi = m; }
    return lo;
}

/* ------------------------------------------------------------------ driver */
/*
 * orc_count: histogram of pairs (i in cat1[i_begin,i_end)) x (j in cat2), or i<j pairs of cat1
 * when a2 == NULL (auto).  mode 0 = plain O(N1 N2) loops (the definition), mode 1 = celled (the
 * same pair body behind the oracle's own cell list; identical results, proven by tests).
 * Outputs (caller-allocated, overwritten): hist[n1*max(n2,1)], amb_cell[ncell+1], amb_e1[n1+1],
 * amb_e2[n2+2] (may be NULL), *npairs = separations evaluated.
 * Angles: coordinates RA/Dec in DEGREES; bin limits and aperture in RADIANS.
 */
int orc_count_w(int kind, int mode,
                int64_t n1, const double *a1, const double *b1, const double *c1, const uint32_t *w1,
                int64_t n2, const double *a2, const double *b2, const double *c2, const uint32_t *w2,
                const orc_bins *bins, int64_t i_begin, int64_t i_end, int nthreads,
                uint64_t *hist, uint64_t *amb_cell, uint64_t *amb_e1, uint64_t *amb_e2, uint64_t *npairs)
{
    int auto_ = (a2 == NULL);
    int rc = check_args(kind, bins, auto_);
    if (rc) return rc;
    if (i_begin < 0) i_begin = 0;
    if (i_end < 0 || i_end > n1) i_end = n1;
    double *e1 = (double *)malloc(((size_t)bins->n1 + 1) * 8), *e2 = (double *)malloc(((size_t)bins->n2 + 2) * 8);
    if (!e1 || !e2) return ORC_ENOMEM;
    orc_edges(bins, 0, e1);
    if (bins->n2 > 0) orc_edges(bins, 1, e2);
    cat_t C1 = {n1, a1, b1, c1, w1, 0, 0, 0}, C2s = {n2, a2, b2, c2, w2, 0, 0, 0};
#define WPROD(i, j) ((uint64_t)(C1.w ? C1.w[i] : 1u) * (uint64_t)(C2->w ? C2->w[j] : 1u))
    if ((rc = prep_cat(kind, &C1))) return rc;
    cat_t *C2 = &C1;
    if (!auto_) { if ((rc = prep_cat(kind, &C2s))) return rc; C2 = &C2s; }
    acc_t G;
    if ((rc = acc_init(&G, kind, bins, e1, e2))) return rc;
    if (nthreads < 1) nthreads = omp_get_max_threads();

    cells_t cells; int have_cells = 0;
    double rmax = 0.0;
    if (mode == 1) {
        if (kind == ORC_MONOPOLE || kind == ORC_RMU || kind == ORC_PISIGMA) {
            rmax = bins->hi1 * (1.0 + 4.0 * ORC_BAND);
            if (kind == ORC_PISIGMA) rmax = sqrt(bins->hi1 * bins->hi1 + bins->hi2 * bins->hi2) * (1.0 + 4.0 * ORC_BAND);
            if ((rc = build_cells3d(&cells, C2, rmax, G.L))) return rc;
            have_cells = 1;
            /* a periodic grid with fewer than 3 cells per side would meet a cell through two images */
            if (G.L > 0.0 && (cells.nc[0] < 3 || cells.nc[1] < 3 || cells.nc[2] < 3)) { free_cells(&cells); have_cells = 0; mode = 0; }
        } else {
            rmax = (kind == ORC_ANGULAR ? bins->hi1 : bins->aperture) * (1.0 + 4.0 * ORC_BAND);
            if (rmax >= 0.5) mode = 0; /* wide angles: cell list pointless */
            else { if ((rc = build_bands(&cells, C2, rmax))) return rc; have_cells = 1; }
        }
    }

    int failed = 0;
#pragma omp parallel num_threads(nthreads)
    {
        acc_t T; /* one private histogram per thread */
        int ok = acc_init(&T, kind, bins, e1, e2) == ORC_OK;
        if (!ok) {
#pragma omp atomic write
            failed = 1;
        }
#pragma omp barrier
        if (!failed) {
#pragma omp for schedule(dynamic, 16)
            for (int64_t i = i_begin; i < i_end; i++) {
                /* the w_i objects of one pixel are w_i (w_i - 1) / 2 pairs at zero separation (reading P2) */
                if (auto_ && C1.w && C1.w[i] > 1)
                    pair_eval(&T, &C1, i, C2, i, (uint64_t)C1.w[i] * (uint64_t)(C1.w[i] - 1) / 2);
                if (mode == 0) {
                    for (int64_t j = auto_ ? i + 1 : 0; j < C2->n; j++) pair_eval(&T, &C1, i, C2, j, WPROD(i, j));
                } else if (cells.kind3d) {
                    const double *X[3] = {C1.a, C1.b, C1.c};
                    int k[3], lo[3], hi[3];
                    for (int d = 0; d < 3; d++) {
                        k[d] = (int)floor((X[d][i] - cells.org[d]) * cells.inv[d]);
                        lo[d] = k[d] - 1; hi[d] = k[d] + 1;
                        if (!cells.periodic) {
                            /* a point of cat1 may lie outside cat2's bounding box: widen by one cell */
                            if (lo[d] < 0) lo[d] = 0;
                            if (hi[d] > cells.nc[d] - 1) hi[d] = cells.nc[d] - 1;
                            if (k[d] < 0) { lo[d] = 0; hi[d] = 0; }
                            if (k[d] > cells.nc[d] - 1) { lo[d] = hi[d] = cells.nc[d] - 1; }
                        }
                    }
                    for (int z = lo[2]; z <= hi[2]; z++)
                        for (int y = lo[1]; y <= hi[1]; y++)
                            for (int x = lo[0]; x <= hi[0]; x++) {
                                int xx = x, yy = y, zz = z;
                                if (cells.periodic) {
                                    xx = ((x % cells.nc[0]) + cells.nc[0]) % cells.nc[0];
                                    yy = ((y % cells.nc[1]) + cells.nc[1]) % cells.nc[1];
                                    zz = ((z % cells.nc[2]) + cells.nc[2]) % cells.nc[2];
                                }
                                int64_t cidx = ((int64_t)zz * cells.nc[1] + yy) * cells.nc[0] + xx;
                                for (int64_t s = cells.start[cidx]; s < cells.start[cidx + 1]; s++) {
                                    int64_t j = cells.idx[s];
                                    if (auto_ && j <= i) continue;
                                    pair_eval(&T, &C1, i, C2, j, WPROD(i, j));
                                }
                            }
                } else {
                    /* declination bands +-1 and the RA window of the spherical cube that contains the
                     * cap of radius rmax about point i (repaired Eq. 16; G2):
                     * half-width asin(sin rmax / cos dec), full ring if the cap reaches a pole. */
                    double dec = C1.b[i], ra = fmod(C1.a[i], 360.0); if (ra < 0) ra += 360.0;
                    int b0 = (int)floor((dec + 90.0) / cells.band_h);
                    if (b0 < 0) b0 = 0;
                    if (b0 >= cells.nband) b0 = cells.nband - 1;
                    double decr = fabs(dec) * ORC_PI / 180.0, w;
                    if (decr + rmax >= 0.5 * ORC_PI * (1.0 - 1e-9)) w = 400.0;
                    else w = asin(sin(rmax) / cos(decr)) * 180.0 / ORC_PI * (1.0 + 1e-9) + 1e-12;
                    for (int b = b0 - 1; b <= b0 + 1; b++) {
                        if (b < 0 || b >= cells.nband) continue;
                        int64_t s0 = cells.start[b], s1 = cells.start[b + 1];
                        double wins[2][2]; int nw = 0;
                        if (w >= 180.0) { wins[0][0] = -1.0; wins[0][1] = 361.0; nw = 1; }
                        else {
                            double a0 = ra - w, a1 = ra + w;
                            if (a0 < 0.0) { wins[0][0] = a0 + 360.0; wins[0][1] = 361.0; wins[1][0] = -1.0; wins[1][1] = a1; nw = 2; }
                            else if (a1 >= 360.0) { wins[0][0] = a0; wins[0][1] = 361.0; wins[1][0] = -1.0; wins[1][1] = a1 - 360.0; nw = 2; }
                            else { wins[0][0] = a0; wins[0][1] = a1; nw = 1; }
                        }
                        for (int q = 0; q < nw; q++) {
                            int64_t p0 = lower_bound_d(cells.ra_sorted, s0, s1, wins[q][0]);
                            for (int64_t s = p0; s < s1 && cells.ra_sorted[s] <= wins[q][1]; s++) {
                                int64_t j = cells.idx[s];
                                if (auto_ && j <= i) continue;
                                pair_eval(&T, &C1, i, C2, j, WPROD(i, j));
                            }
                        }
                    }
                }
            }
#pragma omp critical
            { /* add private histograms */
                for (int c = 0; c < G.ncell; c++) G.hist[c] += T.hist[c];
                for (int c = 0; c <= G.ncell; c++) G.amb_cell[c] += T.amb_cell[c];
                for (int c = 0; c <= bins->n1; c++) G.amb_e1[c] += T.amb_e1[c];
                for (int c = 0; c < bins->n2 + 2; c++) G.amb_e2[c] += T.amb_e2[c];
                G.npairs += T.npairs;
            }
        }
        if (ok) acc_free(&T);
    }
    if (!failed) {
        memcpy(hist, G.hist, (size_t)G.ncell * 8);
        if (amb_cell) memcpy(amb_cell, G.amb_cell, ((size_t)G.ncell + 1) * 8);
        if (amb_e1) memcpy(amb_e1, G.amb_e1, ((size_t)bins->n1 + 1) * 8);
        if (amb_e2) memcpy(amb_e2, G.amb_e2, ((size_t)bins->n2 + 2) * 8);
        if (npairs) *npairs = G.npairs;
    }
    if (have_cells) free_cells(&cells);
    acc_free(&G);
    free_cat(&C1);
    if (!auto_) free_cat(&C2s);
    free(e1); free(e2);
    return failed ? ORC_ENOMEM : ORC_OK;
}

int orc_count(int kind, int mode,
              int64_t n1, const double *a1, const double *b1, const double *c1,
              int64_t n2, const double *a2, const double *b2, const double *c2,
              const orc_bins *bins, int64_t i_begin, int64_t i_end, int nthreads,
              uint64_t *hist, uint64_t *amb_cell, uint64_t *amb_e1, uint64_t *amb_e2, uint64_t *npairs)
{
    return orc_count_w(kind, mode, n1, a1, b1, c1, NULL, n2, a2, b2, c2, NULL, bins, i_begin, i_end, nthreads,
                       hist, amb_cell, amb_e1, amb_e2, npairs);
}

/* Pixel map of an angular catalogue ("create a pixel map from the catalog and then correlate the
 * pixels (weighting each of them by the number of objects that fall inside it)"), on pixels "with constant limits
 * in (cos theta, phi)": n_ra x n_u pixels over RA in [ra0, ra0+dra) (degrees, taken modulo 360
 * relative to ra0) and u = sin(dec) in [u0, u0+du).  Reading P1: a pixel is represented by its centre in (RA, u).
 * Outputs (caller-allocated, n_ra*n_u entries, only the first *npix used): centre RA, centre Dec [deg], count.
 * Non-empty pixels only, in pixel-index order (u-major).  Returns ORC_EINVAL if a point falls outside the map. */
int orc_pixelize(int64_t n, const double *ra, const double *dec, double ra0, double dra, double u0, double du,
                 int n_ra, int n_u, double *pra, double *pdec, uint32_t *pw, int64_t *npix)
{
    if (n < 0 || n_ra < 1 || n_u < 1 || !(dra > 0.0) || !(du > 0.0)) return ORC_EINVAL;
    int64_t np = (int64_t)n_ra * n_u;
    uint32_t *cnt = (uint32_t *)calloc((size_t)np, sizeof(uint32_t));
    if (!cnt) return ORC_ENOMEM;
    for (int64_t i = 0; i < n; i++) {
        double al = fmod(ra[i] - ra0, 360.0);
        if (al < 0.0) al += 360.0;
        double u = sin(dec[i] * (ORC_PI / 180.0)) - u0;
        if (al > dra || u < -1e-15 || u > du + 1e-15) { free(cnt); return ORC_EINVAL; }
        int kx = (int)floor(al * ((double)n_ra / dra)), ky = (int)floor(u * ((double)n_u / du));
        if (kx > n_ra - 1) kx = n_ra - 1;
        if (ky > n_u - 1) ky = n_u - 1;
        if (kx < 0) kx = 0;
        if (ky < 0) ky = 0;
        cnt[(int64_t)ky * n_ra + kx]++;
    }
    int64_t m = 0;
    for (int64_t p = 0; p < np; p++) {
        if (!cnt[p]) continue;
        int kx = (int)(p % n_ra), ky = (int)(p / n_ra);
        double r = ra0 + ((double)kx + 0.5) * (dra / (double)n_ra);
        double uc = u0 + ((double)ky + 0.5) * (du / (double)n_u);
        if (uc > 1.0) uc = 1.0;
        if (uc < -1.0) uc = -1.0;
        pra[m] = fmod(r, 360.0); pdec[m] = asin(uc) * (180.0 / ORC_PI); pw[m] = cnt[p];
        m++;
    }
    *npix = m;
    free(cnt);
    return ORC_OK;
}

/* ------------------------------------------------------------------ estimators (host arithmetic) */
/* Landy-Szalay, Eq. 15 exactly as printed:
 *   xi = [ Nr(Nr-1)/(Nd(Nd-1)) DD - (Nr-1)/Nd DR + RR ] / RR,  DD, RR unordered, DR all pairs.
 * Bins with RR = 0: xi = 0 and they are counted in the return value (paper silent; reading S9). */
int orc_landy_szalay(const uint64_t *dd, const uint64_t *dr, const uint64_t *rr, uint64_t nd, uint64_t nr, int n, double *xi)
{
    int empty = 0;
    double fdd = (double)nr * ((double)nr - 1.0) / ((double)nd * ((double)nd - 1.0));
    double fdr = ((double)nr - 1.0) / (double)nd;
    for (int k = 0; k < n; k++) {
        if (rr[k] == 0) { xi[k] = 0.0; empty++; continue; }
        xi[k] = (fdd * (double)dd[k] - fdr * (double)dr[k] + (double)rr[k]) / (double)rr[k];
    }
    return empty;
}

/* natural estimator, Eq. 14 */
int orc_natural(const uint64_t *dd, const uint64_t *rr, uint64_t nd, uint64_t nr, int n, double *xi)
{
    int empty = 0;
    double f = (double)nr * ((double)nr - 1.0) / ((double)nd * ((double)nd - 1.0));
    for (int k = 0; k < n; k++) {
        if (rr[k] == 0) { xi[k] = 0.0; empty++; continue; }
        xi[k] = f * (double)dd[k] / (double)rr[k] - 1.0;
    }
    return empty;
}

/* expected unordered random pairs in a periodic box: N(N-1)/2 * (4 pi/3)(e_{k+1}^3 - e_k^3) / L^3
 * (north star (a); the paper's Eqs. 12-13, with the exact shell volume and
 * N(N-1)/2 in place of N^2 v(r) ~ 4 pi r^2 dr -- reading S3) */
int orc_periodic_rr(uint64_t n, double L, const orc_bins *b, double *rr)
{
    double *e = (double *)malloc(((size_t)b->n1 + 1) * 8);
    if (!e) return ORC_ENOMEM;
    int rc = orc_edges(b, 0, e);
    if (rc == ORC_OK) {
        double np = 0.5 * (double)n * ((double)n - 1.0);
        for (int k = 0; k < b->n1; k++)
            rr[k] = np * (4.0 * ORC_PI / 3.0) * (e[k + 1] * e[k + 1] * e[k + 1] - e[k] * e[k] * e[k]) / (L * L * L);
    }
    free(e);
    return rc;
}

/* Multipoles of xi(r,mu), Eq. 3-4: xi(r,mu) = sum_l xi_l(r) P_l(mu), so
 * xi_l(r) = (2l+1)/2 int_{-1}^{1} xi(r,mu) P_l(mu) dmu = (2l+1) int_0^1 ... for the even l of a pair-symmetric xi;
 * the monopole is Eq. 4.  The integral over the mu bins is the mid-point rule (reading M1 in DESIGN.md).
 * xi: [n_r][n_mu] over mu in [0,1]; out: [3][n_r] for l = 0, 2, 4. */
int orc_multipoles(const double *xi, int n_r, int n_mu, double *out)
{
    if (n_r < 1 || n_mu < 1) return ORC_EINVAL;
    for (int k = 0; k < n_r; k++) {
        double a0 = 0.0, a2 = 0.0, a4 = 0.0;
        for (int m = 0; m < n_mu; m++) {
            double mu = ((double)m + 0.5) / (double)n_mu, x = xi[(size_t)k * n_mu + m];
            double p2 = 0.5 * (3.0 * mu * mu - 1.0), p4 = (35.0 * mu * mu * mu * mu - 30.0 * mu * mu + 3.0) / 8.0;
            a0 += x; a2 += x * p2; a4 += x * p4;
        }
        out[k] = a0 / (double)n_mu;
        out[n_r + k] = 5.0 * a2 / (double)n_mu;
        out[2 * n_r + k] = 9.0 * a4 / (double)n_mu;
    }
    return ORC_OK;
}

/* ------------------------------------------------------------------ density-grid monopole (CUTE_box)
 * "the particle content of the catalog is first interpolated to a grid and the overdensity field delta is estimated at
 *  every grid point using a TSC algorithm.  Then pairs of grid points are correlated, and a weight delta_i delta_j is
 *  given to each pair.  The correlation function is estimated as xi(r) = < delta(x) delta(x + r) >  (Eq. 17), where the
 *  average is taken over all pairs of grid points separated by a distance r."
 * Readings (the paper gives no formulas here):
 *   D1  the grid points are the CENTRES of the ng^3 cubic cells of side h = L/ng: x_g = (g + 1/2) h, periodic;
 *   D2  TSC = triangular-shaped cloud, the standard second-order B-spline per axis, s = |x - x_g| / h:
 *           W(s) = 3/4 - s^2  (s <= 1/2),   (3/2 - s)^2 / 2  (1/2 < s <= 3/2),   0 otherwise;
 *       a particle feeds the 3 x 3 x 3 grid points around its cell with the product of the three axis weights;
 *   D3  delta_g = rho_g / rho_bar - 1 with rho_bar = N / ng^3 (the weights of one particle sum to 1);
 *   D4  "pairs of grid points separated by a distance r": every ORDERED pair (g, g + v) with v != 0 an integer offset
 *       taken with the minimum image, r = h |v|, binned half-open like every other separation (S1);
 *       xi_k = sum over those pairs of delta_g delta_{g+v} / number of those pairs; a bin no offset falls in has
 *       xi = 0 and is reported empty;  the offsets and their bins are found once, not per grid point.
 * Plain float64 loops. */
static double tsc_w(double s)
{
    s = fabs(s);
    if (s <= 0.5) return 0.75 - s * s;
    if (s <= 1.5) return 0.5 * (1.5 - s) * (1.5 - s);
    return 0.0;
}

/* rho[ng^3] (z-major: index = (gz * ng + gy) * ng + gx) = TSC-assigned particle number per grid point */
int orc_tsc_assign(int64_t n, const double *x, const double *y, const double *z, double L, int ng, double *rho)
{
    if (n < 0 || ng < 3 || !(L > 0.0)) return ORC_EINVAL;
    const double h = L / (double)ng;
    for (int64_t c = 0; c < (int64_t)ng * ng * ng; c++) rho[c] = 0.0;
    for (int64_t i = 0; i < n; i++) {
        const double p[3] = {x[i], y[i], z[i]};
        int g0[3]; double w[3][3];
        for (int d = 0; d < 3; d++) {
            double u = p[d] / h;                       /* position in units of cells */
            int c = (int)floor(u);                     /* the particle's own cell    */
            g0[d] = c - 1;
            for (int k = 0; k < 3; k++) w[d][k] = tsc_w(u - ((double)(c - 1 + k) + 0.5));
        }
        for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++)
                for (int c = 0; c < 3; c++) {
                    int gx = ((g0[0] + c) % ng + ng) % ng, gy = ((g0[1] + b) % ng + ng) % ng, gz = ((g0[2] + a) % ng + ng) % ng;
                    rho[((int64_t)gz * ng + gy) * ng + gx] += w[0][c] * w[1][b] * w[2][a];
                }
    }
    return ORC_OK;
}

/* delta = rho / (n / ng^3) - 1 */
int orc_overdensity(int64_t n, int ng, const double *rho, double *delta)
{
    if (n <= 0 || ng < 1) return ORC_EINVAL;
    const double mean = (double)n / ((double)ng * ng * ng);
    for (int64_t c = 0; c < (int64_t)ng * ng * ng; c++) delta[c] = rho[c] / mean - 1.0;
    return ORC_OK;
}

/* Eq. 17 on a periodic grid: sum_dd[k] = sum of delta_g delta_{g+v} over ordered pairs with h|v| in bin k,
 * npairs[k] = their number, xi[k] = sum_dd / npairs (0 when npairs = 0; the return value counts such bins) */
int orc_grid_correlation(const double *delta, int ng, double L, const orc_bins *b, double *xi, double *sum_dd, uint64_t *npairs)
{
    if (ng < 3 || !(L > 0.0) || b->n1 < 1 || !(b->lo1 < b->hi1) || b->hi1 > 0.5 * L) return ORC_EINVAL;
    double *e = (double *)malloc(((size_t)b->n1 + 1) * 8);
    if (!e) return ORC_ENOMEM;
    int rc = orc_edges(b, 0, e);
    if (rc) { free(e); return rc; }
    axis_t ax = {b->n1, b->log1, 0, b->lo1, b->hi1, e};
    const double h = L / (double)ng;
    int m = (int)floor(b->hi1 / h);
    if (m > (ng - 1) / 2) m = (ng - 1) / 2;
    for (int k = 0; k < b->n1; k++) { sum_dd[k] = 0.0; npairs[k] = 0; }
    const int64_t ng3 = (int64_t)ng * ng * ng;
    for (int dz = -m; dz <= m; dz++)
        for (int dy = -m; dy <= m; dy++)
            for (int dx = -m; dx <= m; dx++) {
                if (dx == 0 && dy == 0 && dz == 0) continue;
                const double r = h * sqrt((double)(dx * dx + dy * dy + dz * dz));
                const int k = find_bin(&ax, r);
                if (k < 0) continue;
                double s = 0.0;
#pragma omp parallel for reduction(+ : s) schedule(static)
                for (int gz = 0; gz < ng; gz++) {
                    const int hz = (gz + dz + ng) % ng;
                    for (int gy = 0; gy < ng; gy++) {
                        const int hy = (gy + dy + ng) % ng;
                        const double *r0 = delta + ((int64_t)gz * ng + gy) * ng, *r1 = delta + ((int64_t)hz * ng + hy) * ng;
                        for (int gx = 0; gx < ng; gx++) s += r0[gx] * r1[(gx + dx + ng) % ng];
                    }
                }
                sum_dd[k] += s;
                npairs[k] += (uint64_t)ng3;
            }
    int empty = 0;
    for (int k = 0; k < b->n1; k++) {
        if (npairs[k] == 0) { xi[k] = 0.0; empty++; }
        else xi[k] = sum_dd[k] / (double)npairs[k];
    }
    free(e);
    return empty;
}

int orc_max_threads(void) { return omp_get_max_threads(); }
