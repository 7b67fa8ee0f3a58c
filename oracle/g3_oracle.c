/*
 * g3_oracle.c -- plain CPU oracle for the triplet correlation function g(3).
 *
 * THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and the
 * `cpu_baseline` / `--impl reference` legs of bench.py may build, link, import
 * or call anything under oracle/.  The product (paper_1708_08619_b200/) never
 * does, and shares no code, header, table or constant generator with this file.
 *
 * What it computes follows arxiv 1708.08619, section 3.2:
 *   - Eq. 3: definition of g(3) and its rho^3 normalisation;
 *   - PAPER.md:407-409: "3D histogram binning of distances", two distances
 *     inside one cut-off and the third inside twice that;
 *   - Algorithm 6: per frame, minimum-image pair distances,
 *     "store new coordinates of neighbour particles", then for a centre i the
 *     pairs (j,k) of its neighbours, the j-k distance "using updated positions",
 *     and the histogram update;
 *   - Algorithm 7: the same with one thread per neighbour j
 *     looping over all neighbours k of i  ->  ORDERED pairs (j,k), j != k.
 * Where the paper is silent the readings S1-S5 / Q1-Q16 of SURVEY.md section 8(c),
 * restated in DESIGN.md ("Readings of the paper"), are taken.  The method reaches
 * exactly a plain definition (a histogram of integer-valued squared distances),
 * so this file IS that definition written out: no cell list in the reference
 * routine, no blocking, no fusion, no symmetry tricks.
 *
 * Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`): brute-force O(N^3)
 * enumeration in exact Python integers; the hand-computed 4x4x4 lattice values
 * of SURVEY.md 8(c) (tests/golden/lattice_4x4x4.txt); hand cases (three in a
 * line, equilateral triangle, pair across the periodic boundary); the count
 * invariant sum_i k_i (k_i - 1); r12<->r13 symmetry; triangle-inequality support;
 * shell marginals; metamorphic invariances; thresholds against exact rational
 * arithmetic; bin volumes against closed-form row sums, the total, the interior
 * closed form, the sphere-sphere lens volume and adaptive quadrature; ideal-gas
 * g3 = (1-1/N)(1-2/N).  No function here is "parity unpinned".
 *
 * Arithmetic: integers for everything that decides a bin (exact), fp64 with one
 * IEEE rounding per operation elsewhere.  Compile with -ffp-contract=off.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define G3O_GRID_BITS 20
#define G3O_GRID ((int64_t)1 << G3O_GRID_BITS)

/* ------------------------------------------------------------------------- */
/* S1  threshold tables (bin edges uniform in r, half-open,
 *     compared in squared integer grid units, reading Q7).                   */
/* T_r has n_r + 1 entries, T_t has n_t + 1 entries.                          */
void g3o_thresholds(double box, double r_max, int32_t n_r, int32_t n_t,
                    uint64_t *T_r, uint64_t *T_t)
{
    double inv_g = 1048576.0 / box;
    double w = (r_max / (double)n_r) * inv_g;
    double wt = ((2.0 * r_max) / (double)n_t) * inv_g;
    for (int32_t b = 0; b <= n_r; ++b) {
        double e = (double)b * w;
        T_r[b] = (uint64_t)ceil(e * e);
    }
    for (int32_t c = 0; c <= n_t; ++c) {
        double e = (double)c * wt;
        T_t[c] = (uint64_t)ceil(e * e);
    }
}

/* bin(T, q) = the largest b in [0, n] with T[b] <= q   (T[0] = 0 <= q always). */
static int32_t bin_of(const uint64_t *T, int32_t n, uint64_t q)
{
    int32_t lo = 0, hi = n;            /* invariant: T[lo] <= q; answer in [lo, hi] */
    while (lo < hi) {
        int32_t mid = lo + (hi - lo + 1) / 2;
        if (T[mid] <= q) lo = mid; else hi = mid - 1;
    }
    return lo;
}

/* ------------------------------------------------------------------------- */
/* S2  snap positions to the box/2^20 grid and wrap into the box.             */
void g3o_quantise(const double *pos, int64_t n, double box, int32_t *m)
{
    double inv_g = 1048576.0 / box;
    for (int64_t p = 0; p < 3 * n; ++p)
        m[p] = (int32_t)(llrint(pos[p] * inv_g) & (G3O_GRID - 1));
}

/* minimum-image component in grid units: ((d + 2^19) mod 2^20) - 2^19  (S3). */
static int64_t wrap(int64_t d)
{
    return (((d + (G3O_GRID >> 1)) % G3O_GRID + G3O_GRID) % G3O_GRID) - (G3O_GRID >> 1);
}

/* ------------------------------------------------------------------------- */
/* S3 + S4 for ONE centre i, given the candidate list `cand` (indices of the
 * particles to test as neighbours; the reference routine passes all of them).
 * Stores the minimum-image vectors of the neighbours ("store new coordinates
 * of neighbour particles"; Alg. 7 CUDA_g2), then
 * loops over ordered pairs (j,k), j != k (Alg. 7 CUDA_g3),
 * taking the j-k distance from the stored vectors with no second wrap
 * (reading Q3).  Returns k_i.                             */
typedef struct { int64_t dx, dy, dz; int32_t a; } nb_t;

static int64_t centre(const int32_t *m, int64_t i, const int64_t *cand, int64_t ncand,
                      const uint64_t *T_r, int32_t n_r, const uint64_t *T_t, int32_t n_t,
                      nb_t *nb, uint64_t *H, uint64_t *overflow)
{
    int64_t k_i = 0;
    for (int64_t q = 0; q < ncand; ++q) {
        int64_t j = cand ? cand[q] : q;
        if (j == i) continue;                                   /* Q10: j != i by index */
        int64_t dx = wrap((int64_t)m[3 * j + 0] - (int64_t)m[3 * i + 0]);
        int64_t dy = wrap((int64_t)m[3 * j + 1] - (int64_t)m[3 * i + 1]);
        int64_t dz = wrap((int64_t)m[3 * j + 2] - (int64_t)m[3 * i + 2]);
        uint64_t d2 = (uint64_t)(dx * dx + dy * dy + dz * dz);
        if (d2 < T_r[n_r]) {                                    /* r_ij < r_max */
            nb[k_i].dx = dx; nb[k_i].dy = dy; nb[k_i].dz = dz;
            nb[k_i].a = bin_of(T_r, n_r, d2);
            ++k_i;
        }
    }
    for (int64_t j = 0; j < k_i; ++j) {
        for (int64_t k = 0; k < k_i; ++k) {
            if (k == j) continue;                               /* Q5 */
            int64_t ex = nb[k].dx - nb[j].dx;
            int64_t ey = nb[k].dy - nb[j].dy;
            int64_t ez = nb[k].dz - nb[j].dz;
            uint64_t t2 = (uint64_t)(ex * ex + ey * ey + ez * ez);
            int32_t c = bin_of(T_t, n_t, t2);
            if (c < n_t)
                H[((int64_t)nb[j].a * n_r + nb[k].a) * n_t + c] += 1;
            else
                *overflow += 1;                                 /* Q12 */
        }
    }
    return k_i;
}

/* ------------------------------------------------------------------------- */
/* One frame, reference routine: every centre tests all N particles
 * (Alg. 6 loop 3 / Alg. 7 CUDA_g2 loop 3).  H [n_r][n_r][n_t] (c fastest) and
 * stats = {frames, sum_i k_i (k_i - 1), overflow} are ADDED to.
 * OpenMP splits the centres over threads with one private histogram each
 * (PAPER.md:717-721 parallelises the CPU code by splitting the work and
 * merging results); integer sums make the result independent of the split.   */
static void frame_generic(const int32_t *m, int64_t n,
                          const int64_t *cell_start, const int64_t *cell_items, int32_t ncell,
                          const uint64_t *T_r, int32_t n_r, const uint64_t *T_t, int32_t n_t,
                          uint64_t *H, uint64_t *stats)
{
    int64_t nbins = (int64_t)n_r * n_r * n_t;
    uint64_t pairs = 0, overflow = 0;
#pragma omp parallel reduction(+ : pairs, overflow)
    {
        uint64_t *Hl = (uint64_t *)calloc((size_t)nbins, sizeof(uint64_t));
        nb_t *nb = (nb_t *)malloc((size_t)n * sizeof(nb_t));
        int64_t *cand = cell_start ? (int64_t *)malloc((size_t)n * sizeof(int64_t)) : NULL;
#pragma omp for schedule(dynamic, 16)
        for (int64_t i = 0; i < n; ++i) {
            int64_t ncand = n;
            if (cell_start) {
                /* candidates = particles of the 27 cells around the centre's cell */
                int64_t cx = ((int64_t)m[3 * i + 0] * ncell) >> G3O_GRID_BITS;
                int64_t cy = ((int64_t)m[3 * i + 1] * ncell) >> G3O_GRID_BITS;
                int64_t cz = ((int64_t)m[3 * i + 2] * ncell) >> G3O_GRID_BITS;
                ncand = 0;
                for (int64_t ox = -1; ox <= 1; ++ox)
                    for (int64_t oy = -1; oy <= 1; ++oy)
                        for (int64_t oz = -1; oz <= 1; ++oz) {
                            int64_t c = (((cx + ox + ncell) % ncell) * ncell
                                         + (cy + oy + ncell) % ncell) * ncell
                                        + (cz + oz + ncell) % ncell;
                            for (int64_t q = cell_start[c]; q < cell_start[c + 1]; ++q)
                                cand[ncand++] = cell_items[q];
                        }
            }
            uint64_t ov = 0;
            int64_t k_i = centre(m, i, cand, ncand, T_r, n_r, T_t, n_t, nb, Hl, &ov);
            pairs += (uint64_t)(k_i * (k_i - 1));
            overflow += ov;
        }
#pragma omp critical
        for (int64_t b = 0; b < nbins; ++b) H[b] += Hl[b];
        free(Hl); free(nb); free(cand);
    }
    stats[0] += 1;
    stats[1] += pairs;
    stats[2] += overflow;
}

void g3o_frame_allpairs(const int32_t *m, int64_t n,
                        const uint64_t *T_r, int32_t n_r, const uint64_t *T_t, int32_t n_t,
                        uint64_t *H, uint64_t *stats)
{
    frame_generic(m, n, NULL, NULL, 0, T_r, n_r, T_t, n_t, H, stats);
}

/* One frame with a plain cell grid in front of the same per-centre routine:
 * ncell = floor(2^20 / ceil(sqrt(T_r[n_r]))) cells per edge, each at least one
 * cut-off wide, so all neighbours of a centre lie in the 27 cells around it.
 * Only a candidate pre-filter; used for the large configs and the timed CPU
 * baseline.  Falls back to the reference routine when ncell < 3 (config 1).
 * Pinned against g3o_frame_allpairs in tests/test_oracle_pins.py.            */
void g3o_frame_cells(const int32_t *m, int64_t n,
                     const uint64_t *T_r, int32_t n_r, const uint64_t *T_t, int32_t n_t,
                     uint64_t *H, uint64_t *stats)
{
    int64_t reach = (int64_t)ceil(sqrt((double)T_r[n_r])) + 1;   /* > any neighbour |component| */
    int32_t ncell = (int32_t)(G3O_GRID / reach);
    if (ncell < 3) { g3o_frame_allpairs(m, n, T_r, n_r, T_t, n_t, H, stats); return; }
    if (ncell > 64) ncell = 64;
    /* cell c covers grid coordinates [ceil(c 2^20/ncell), ceil((c+1) 2^20/ncell)):
     * width >= floor(2^20/ncell) >= reach, so neighbours are at most one cell away. */
    int64_t nc3 = (int64_t)ncell * ncell * ncell;
    int64_t *start = (int64_t *)calloc((size_t)nc3 + 1, sizeof(int64_t));
    int64_t *items = (int64_t *)malloc((size_t)n * sizeof(int64_t));
    int64_t *cid = (int64_t *)malloc((size_t)n * sizeof(int64_t));
    for (int64_t i = 0; i < n; ++i) {
        int64_t cx = ((int64_t)m[3 * i + 0] * ncell) >> G3O_GRID_BITS;
        int64_t cy = ((int64_t)m[3 * i + 1] * ncell) >> G3O_GRID_BITS;
        int64_t cz = ((int64_t)m[3 * i + 2] * ncell) >> G3O_GRID_BITS;
        cid[i] = (cx * ncell + cy) * ncell + cz;
        start[cid[i] + 1] += 1;
    }
    for (int64_t c = 0; c < nc3; ++c) start[c + 1] += start[c];
    int64_t *fill = (int64_t *)malloc((size_t)nc3 * sizeof(int64_t));
    memcpy(fill, start, (size_t)nc3 * sizeof(int64_t));
    for (int64_t i = 0; i < n; ++i) items[fill[cid[i]]++] = i;
    frame_generic(m, n, start, items, ncell, T_r, n_r, T_t, n_t, H, stats);
    free(start); free(items); free(cid); free(fill);
}

/* Convenience: quantise fp64 positions and accumulate F frames.
 * mode 0 = reference all-pairs routine, 1 = cell-grid pre-filter.            */
void g3o_accumulate(const double *pos, int64_t n_frames, int64_t n, double box, double r_max,
                    int32_t n_r, int32_t n_t, int32_t mode, uint64_t *H, uint64_t *stats)
{
    uint64_t *T_r = (uint64_t *)malloc((size_t)(n_r + 1) * sizeof(uint64_t));
    uint64_t *T_t = (uint64_t *)malloc((size_t)(n_t + 1) * sizeof(uint64_t));
    int32_t *m = (int32_t *)malloc((size_t)(3 * n) * sizeof(int32_t));
    g3o_thresholds(box, r_max, n_r, n_t, T_r, T_t);
    for (int64_t f = 0; f < n_frames; ++f) {
        g3o_quantise(pos + f * 3 * n, n, box, m);
        if (mode == 0) g3o_frame_allpairs(m, n, T_r, n_r, T_t, n_t, H, stats);
        else g3o_frame_cells(m, n, T_r, n_r, T_t, n_t, H, stats);
    }
    free(T_r); free(T_t); free(m);
}

/* ------------------------------------------------------------------------- */
/* S5  bin volumes.  V_abc = integral over the bin of the ideal-gas triplet
 * density in (r, s, t) = (r_ij, r_ik, r_jk):
 *     8 pi^2 r s t  on  |r - s| <= t <= r + s,  0 elsewhere
 * (shell 4 pi r^2 dr for j, ring 2 pi s^2 sin(theta) dtheta ds for k, and
 * t dt = r s sin(theta) dtheta).  Integrating t first,
 *     V = 8 pi^2  int_r  r  int_s  s h(r,s) ds dr,
 *     h = (1/2) [ min(t1, r+s)^2 - max(t0, |r-s|)^2 ]_+ .
 * h is piecewise polynomial; the s range is split where its form changes
 * (r+s = t0, r+s = t1, |r-s| = t0, |r-s| = t1) and the r range where one of
 * those breakpoints crosses s0 or s1 or another breakpoint, so that 5-point
 * Gauss-Legendre is exact (to rounding) on every piece.                      */
static const double GL_X[5] = {
    -0.90617984593866399280, -0.53846931010568309104, 0.0,
     0.53846931010568309104,  0.90617984593866399280 };
static const double GL_W[5] = {
    0.23692688505618908751, 0.47862867049936646804, 0.56888888888888888889,
    0.47862867049936646804, 0.23692688505618908751 };

#define PI_SQ 9.8696044010893586188

static int cmp_double(const void *a, const void *b)
{
    double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

static double h_of(double r, double s, double t0, double t1)
{
    double up = r + s < t1 ? r + s : t1;
    double lo = fabs(r - s) > t0 ? fabs(r - s) : t0;
    return up > lo ? 0.5 * (up * up - lo * lo) : 0.0;
}

static double inner_s(double r, double s0, double s1, double t0, double t1)
{
    double cut[8] = { s0, s1, t1 - r, t0 - r, r - t0, r + t0, r - t1, r + t1 };
    for (int q = 2; q < 8; ++q) { if (cut[q] < s0) cut[q] = s0; if (cut[q] > s1) cut[q] = s1; }
    qsort(cut, 8, sizeof(double), cmp_double);
    double sum = 0.0;
    for (int q = 0; q + 1 < 8; ++q) {
        double a = cut[q], b = cut[q + 1];
        if (!(b > a)) continue;
        double mid = 0.5 * (a + b), half = 0.5 * (b - a), piece = 0.0;
        for (int g = 0; g < 5; ++g) {
            double s = mid + half * GL_X[g];
            piece += GL_W[g] * s * h_of(r, s, t0, t1);
        }
        sum += half * piece;
    }
    return sum;
}

static double bin_volume(double r0, double r1, double s0, double s1, double t0, double t1)
{
    const double PI = 3.14159265358979323846;
    double cut[18];
    int nc = 0;
    cut[nc++] = r0; cut[nc++] = r1;
    double ss[2] = { s0, s1 }, tt[2] = { t0, t1 };
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) {
            cut[nc++] = tt[b] - ss[a];
            cut[nc++] = ss[a] - tt[b];
            cut[nc++] = ss[a] + tt[b];
        }
    cut[nc++] = 0.5 * (t0 + t1); cut[nc++] = 0.5 * (t1 - t0); cut[nc++] = t0; cut[nc++] = t1;
    for (int q = 2; q < nc; ++q) { if (cut[q] < r0) cut[q] = r0; if (cut[q] > r1) cut[q] = r1; }
    qsort(cut, (size_t)nc, sizeof(double), cmp_double);
    double sum = 0.0;
    for (int q = 0; q + 1 < nc; ++q) {
        double a = cut[q], b = cut[q + 1];
        if (!(b > a)) continue;
        double mid = 0.5 * (a + b), half = 0.5 * (b - a), piece = 0.0;
        for (int g = 0; g < 5; ++g) {
            double r = mid + half * GL_X[g];
            piece += GL_W[g] * r * inner_s(r, s0, s1, t0, t1);
        }
        sum += half * piece;
    }
    return 8.0 * PI * PI * sum;
}

/* V [n_r][n_r][n_t], c fastest, in (length unit of r_max)^6. */
void g3o_volumes(double r_max, int32_t n_r, int32_t n_t, double *V)
{
    double w = r_max / (double)n_r, wt = (2.0 * r_max) / (double)n_t;
#pragma omp parallel for collapse(2) schedule(dynamic, 8)
    for (int32_t a = 0; a < n_r; ++a)
        for (int32_t b = 0; b < n_r; ++b)
            for (int32_t c = 0; c < n_t; ++c) {
                double r0 = a * w, r1 = (a + 1) * w, s0 = b * w, s1 = (b + 1) * w;
                double t0 = c * wt, t1 = (c + 1) * wt;
                double v = bin_volume(r0, r1, s0, s1, t0, t1);
                /* A bin that meets the support |r-s| <= t <= r+s only in a corner or an edge has
                 * V = 0 exactly, but rounded break points can leave ~1e-50.  Anything below 1e-12
                 * of the unclipped box integral pi^2 D(r^2) D(s^2) D(t^2) is such a bin: V = 0
                 * (reading Q17 in DESIGN.md), so that "g3 = 0 where V_abc = 0" applies to it.     */
                double boxint = PI_SQ * (r1 * r1 - r0 * r0) * (s1 * s1 - s0 * s0) * (t1 * t1 - t0 * t0);
                V[((int64_t)a * n_r + b) * n_t + c] = v < 1e-12 * boxint ? 0.0 : v;
            }
}

/* g3 = H / (F N rho^2 V_abc), rho = N / L^3 (Eq. 3's rho^3 convention, PAPER.md:405;
 * readings Q8, Q9); 0 where V_abc = 0.                                       */
void g3o_normalise(const uint64_t *H, const double *V, int64_t nbins,
                   int64_t n_frames, int64_t n, double box, double *g3)
{
    double rho = (double)n / (box * box * box);
    double ideal = (double)n_frames * (double)n * rho * rho;   /* expected ordered pairs per unit V */
    for (int64_t b = 0; b < nbins; ++b)
        g3[b] = V[b] > 0.0 ? (double)H[b] / (ideal * V[b]) : 0.0;
}

/* ------------------------------------------------------------------------- */
/* g2: the pair distribution function from the same pair loop.
 * Algorithm 6 computes it beside the neighbour vectors ("Calculate the minimum image
 * distance ... Update the g2 histogram") and Algorithm 7's CUDA_g2 kernel
 * does the same per thread i.  Reading G1: the paper's g2
 * cut-off is L/2; here the pair histogram covers the neighbour range [0, r_max) with the n_r
 * shells of r_ij, i.e. H2[a] = number of ORDERED pairs (i, j), j != i, whose minimum-image
 * squared distance falls in [T_r[a], T_r[a+1]).  Plain all-pairs double loop, no cell list.
 * H2 [n_r] is ADDED to.  Pins: tests/test_oracle_g2.py.                                    */
void g3o_g2_frame(const int32_t *m, int64_t n, const uint64_t *T_r, int32_t n_r, uint64_t *H2)
{
    /* OpenMP splits the centres i over threads, one private histogram each, summed at the end
     * (integer sums: the result does not depend on the split).                              */
#pragma omp parallel
    {
        uint64_t *h = (uint64_t *)calloc((size_t)n_r, sizeof(uint64_t));
#pragma omp for schedule(static)
        for (int64_t i = 0; i < n; ++i)
            for (int64_t j = 0; j < n; ++j) {
                if (j == i) continue;
                int64_t dx = wrap((int64_t)m[3 * j + 0] - m[3 * i + 0]);
                int64_t dy = wrap((int64_t)m[3 * j + 1] - m[3 * i + 1]);
                int64_t dz = wrap((int64_t)m[3 * j + 2] - m[3 * i + 2]);
                uint64_t d2 = (uint64_t)(dx * dx + dy * dy + dz * dz);
                if (d2 < T_r[n_r]) h[bin_of(T_r, n_r, d2)] += 1;
            }
#pragma omp critical
        for (int32_t a = 0; a < n_r; ++a) H2[a] += h[a];
        free(h);
    }
}

/* g2[a] = H2[a] / (F N rho V_a), V_a = (4 pi / 3)(r_{a+1}^3 - r_a^3), rho = N / L^3: the
 * ideal-gas value is (N-1)/N (same rho convention as Eq. 3, reading Q9).                   */
void g3o_g2_normalise(const uint64_t *H2, int32_t n_r, double r_max, int64_t n_frames, int64_t n,
                      double box, double *g2)
{
    double rho = (double)n / (box * box * box);
    double w = r_max / (double)n_r;
    for (int32_t a = 0; a < n_r; ++a) {
        double r0 = a * w, r1 = (a + 1) * w;
        double V = (4.0 * 3.14159265358979323846 / 3.0) * (r1 * r1 * r1 - r0 * r0 * r0);
        g2[a] = n_frames > 0 ? (double)H2[a] / ((double)n_frames * (double)n * rho * V) : 0.0;
    }
}

/* ------------------------------------------------------------------------- */
/* q_tet: the tetrahedral order parameter, Eq. 1:
 *     q = 1 - (3/8) sum_{j<k} (cos psi_jk + 1/3)^2
 * over the six pairs of the FOUR NEAREST neighbours j, k of atom i, psi_jk the angle between
 * the bond vectors r_ij and r_ik; Algorithm 2: all minimum-image distances
 * from i, sort, four nearest, Eq. 1, "Update histogram with qtet".
 * Readings (T1-T4; the paper states none of these):
 *  T1 nearest = smallest squared minimum-image distance on the integer grid; ties are broken by
 *     the vector itself, (d2, dx, dy, dz) in lexicographic order, so the choice does not depend
 *     on particle numbering;
 *  T2 arithmetic in fp64, one rounding per operation, in exactly this order: n_j = sqrt(d2_j);
 *     c = dot / (n_j * n_k) with the integer dot product converted exactly; t = c + 1/3;
 *     acc += t * t over (1,2),(1,3),(1,4),(2,3),(2,4),(3,4) of the sorted four; q = 1 - 0.375 acc;
 *  T3 histogram: n_q bins of width 4/n_q on [-3, 1]; bin = floor((q + 3) * (n_q / 4)), q = 1
 *     goes to the last bin;
 *  T4 an atom with a coincident neighbour among the four (d2 = 0: no bond direction) is skipped
 *     and counted in stats[1]; stats[0] counts the atoms binned.
 * Plain all-pairs loop (no cell list); H [n_q] and stats [2] are ADDED to.                  */
typedef struct { uint64_t d2; int64_t x, y, z; } qt_nb;

static int qt_less(const qt_nb *a, const qt_nb *b)
{
    if (a->d2 != b->d2) return a->d2 < b->d2;
    if (a->x != b->x) return a->x < b->x;
    if (a->y != b->y) return a->y < b->y;
    return a->z < b->z;
}

/* q of one atom from its four nearest neighbours, sorted (reading T2); returns 0 if skipped (T4) */
static int qt_value(const qt_nb *nb, double *q)
{
    double nrm[4];
    for (int j = 0; j < 4; ++j) {
        if (nb[j].d2 == 0) return 0;
        nrm[j] = sqrt((double)nb[j].d2);
    }
    double acc = 0.0;
    for (int j = 0; j < 3; ++j)
        for (int k = j + 1; k < 4; ++k) {
            int64_t dot = nb[j].x * nb[k].x + nb[j].y * nb[k].y + nb[j].z * nb[k].z;
            double den = nrm[j] * nrm[k];
            double c = (double)dot / den;
            double t = c + 1.0 / 3.0;
            double t2 = t * t;
            acc = acc + t2;
        }
    double s = 0.375 * acc;
    *q = 1.0 - s;
    return 1;
}

/* q_out (may be NULL): q of every atom of this frame, NaN where skipped.                   */
void g3o_qtet_frame(const int32_t *m, int64_t n, int32_t n_q, uint64_t *H, uint64_t *stats,
                    double *q_out)
{
    double scale = (double)n_q / 4.0;
    uint64_t binned = 0, skipped = 0;
#pragma omp parallel reduction(+ : binned, skipped)
    {
        uint64_t *h = (uint64_t *)calloc((size_t)n_q, sizeof(uint64_t));
#pragma omp for schedule(static)
        for (int64_t i = 0; i < n; ++i) {
            qt_nb best[4];
            int have = 0;
            for (int64_t j = 0; j < n; ++j) {
                if (j == i) continue;
                qt_nb c;
                c.x = wrap((int64_t)m[3 * j + 0] - m[3 * i + 0]);
                c.y = wrap((int64_t)m[3 * j + 1] - m[3 * i + 1]);
                c.z = wrap((int64_t)m[3 * j + 2] - m[3 * i + 2]);
                c.d2 = (uint64_t)(c.x * c.x + c.y * c.y + c.z * c.z);
                /* insertion into the sorted list of the four smallest (T1) */
                int pos = have;
                while (pos > 0 && qt_less(&c, &best[pos - 1])) --pos;
                if (pos >= 4) continue;
                int last = have < 4 ? have : 3;
                for (int t = last; t > pos; --t) best[t] = best[t - 1];
                best[pos] = c;
                if (have < 4) ++have;
            }
            double q;
            if (have < 4 || !qt_value(best, &q)) {
                skipped += 1;
                if (q_out) q_out[i] = NAN;
                continue;
            }
            if (q_out) q_out[i] = q;
            double pos = (q + 3.0) * scale;
            int64_t b = (int64_t)floor(pos);
            if (b < 0) b = 0;
            if (b > n_q - 1) b = n_q - 1;
            h[b] += 1;
            binned += 1;
        }
#pragma omp critical
        for (int32_t b = 0; b < n_q; ++b) H[b] += h[b];
        free(h);
    }
    stats[0] += binned;
    stats[1] += skipped;
}

/* ------------------------------------------------------------------------- */
/* MSD: the mean square displacement over all time origins, Eq. 5
 * and Algorithm 10: "Starting from unwrapped" positions, loop
 * over the particles, over the time interval dt = 0 .. and over the origins t = 1 .. Nframe-dt,
 * "Compute MSD of particle between t and t+dt", "Accumulate MSD array".
 * Readings (M1-M3; the paper states none of these):
 *  M1 positions are snapped to the box/2^20 grid WITHOUT wrapping, m = llrint(x * 2^20 / box),
 *     so every squared displacement is an integer and the sums are exact; |m| < 2^30 is required
 *     (returns the number of coordinates outside, and no result, otherwise);
 *  M2 S[dt] = sum_i sum_{t=0}^{F-dt-1} |m_i(t+dt) - m_i(t)|^2 as a 128-bit integer, returned as
 *     (lo, hi) 64-bit words; lags dt = 0 .. max_lag, max_lag <= F - 1;
 *  M3 msd[dt] = (hi 2^64 + lo) g^2 / (N (F - dt)) in fp64, g = box / 2^20, evaluated as
 *     s = (double)hi * 2^64 + (double)lo; num = s * (g * g); den = (double)N * (double)(F - dt);
 *     msd = num / den.
 * pos [F][n][3] fp64; sums [max_lag+1][2]; msd [max_lag+1].                                  */
int64_t g3o_msd(const double *pos, int64_t n_frames, int64_t n, double box, int64_t max_lag,
                uint64_t *sums, double *msd)
{
    double inv_g = 1048576.0 / box;
    int64_t total = n_frames * n * 3, bad = 0;
    int64_t *m = (int64_t *)malloc(sizeof(int64_t) * (size_t)total);
    for (int64_t q = 0; q < total; ++q) {
        m[q] = (int64_t)llrint(pos[q] * inv_g);
        if (m[q] >= ((int64_t)1 << 30) || m[q] <= -((int64_t)1 << 30)) bad += 1;
    }
    if (bad) { free(m); return bad; }
    unsigned __int128 *S = (unsigned __int128 *)calloc((size_t)(max_lag + 1), sizeof(unsigned __int128));
#pragma omp parallel
    {
        unsigned __int128 *loc = (unsigned __int128 *)calloc((size_t)(max_lag + 1), sizeof(unsigned __int128));
#pragma omp for schedule(static)
        for (int64_t i = 0; i < n; ++i)                       /* Loop 1 over the particles      */
            for (int64_t dt = 0; dt <= max_lag; ++dt)         /* Loop 2 over the time interval  */
                for (int64_t t = 0; t < n_frames - dt; ++t) { /* Loop 3 over the origins        */
                    const int64_t *a = m + ((t * n) + i) * 3, *b = m + (((t + dt) * n) + i) * 3;
                    int64_t dx = b[0] - a[0], dy = b[1] - a[1], dz = b[2] - a[2];
                    loc[dt] += (unsigned __int128)((uint64_t)(dx * dx) + (uint64_t)(dy * dy) + (uint64_t)(dz * dz));
                }
#pragma omp critical
        for (int64_t dt = 0; dt <= max_lag; ++dt) S[dt] += loc[dt];
        free(loc);
    }
    double g = box / 1048576.0;
    double gg = g * g;
    for (int64_t dt = 0; dt <= max_lag; ++dt) {
        uint64_t lo = (uint64_t)S[dt], hi = (uint64_t)(S[dt] >> 64);
        sums[2 * dt + 0] = lo;
        sums[2 * dt + 1] = hi;
        double s = (double)hi * 18446744073709551616.0 + (double)lo;
        double num = s * gg;
        double den = (double)n * (double)(n_frames - dt);
        msd[dt] = num / den;
    }
    free(S);
    free(m);
    return 0;
}

/* Thread count of the OpenMP loops (bench.py's single-thread figure: the analogue of the paper's
 * serial code).  No effect on any result: the sums are integers. */
void g3o_set_num_threads(int32_t n)
{
#ifdef _OPENMP
    if (n >= 1) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int32_t g3o_num_threads(void)
{
#ifdef _OPENMP
    return (int32_t)omp_get_max_threads();
#else
    return 1;
#endif
}
