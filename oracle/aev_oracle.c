/*
 * aev_oracle.c -- fp64 CPU ORACLE for the ANI-style AEV hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load this.  It shares no code, header,
 * table or helper with the CUDA library (paper_2310_03121_b200/csrc) and neither
 * includes the other.
 *
 * What it computes is the plain definition of the path named by
 * BASELINE.json:north_star (PAPER.md:112 names the operations -- "atom-centered
 * symmetry functions used in the ANI family of potentials, building neighbor
 * lists"; PAPER.md:75 fixes the contract -- positions in, energy out, forces by
 * backpropagation).  The paper gives no formulas; the formulas are north_star's,
 * written out exactly as SURVEY.md section 8(c) steps 1-6 restate them:
 *
 *   step 1  pairs      d_ij = x_j - x_i - L*rint((x_j - x_i)/L), r_ij < R_c   (strict, G3)
 *   step 2  cutoff     f_c(r;R) = 0.5*cos(pi*r/R) + 0.5
 *   step 3  radial     G_R = 0.25*exp(-eta_R*(r-R_s)^2)*f_c(r;R_cr)
 *   step 4  angular    G_A = 2^(1-zeta)*(1+cos(theta-theta_s))^zeta
 *                            *exp(-eta_A*((r_ij+r_ik)/2-R_s)^2)*f_c(r_ij)*f_c(r_ik)
 *                      over UNORDERED neighbour pairs {j,k} (G1), theta = acos(c*cos_raw) (G2)
 *   step 5  backward   forces = -sum g * dAEV/dx (analytic chain rule)
 *   step 6  MLP        z = hW + b, CELU_alpha hidden, linear last layer, E = sum E_i
 *
 * All arithmetic is double.  Inputs are the float32 arrays the CUDA path also
 * receives, promoted to double (G9).  No blocking, fusion or reordering: explicit
 * double/triple loops in the order of the definition.  OpenMP (if compiled in)
 * only distributes the outer loop over central atoms.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): closed forms for 2- and 3-atom
 * systems and one water (tests/golden/), brute force vs cell list vs scipy cKDTree
 * pair sets, translation / rotation / permutation / periodic-image invariance, zero
 * net force and torque, central finite differences, torch-CPU fp64 autograd of an
 * independently written definition, MLP special cases.  Parity status: pinned
 * (the CHOICE among readings G1/G2/G6/G7/G13/G14 is a convention).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_PI 3.14159265358979323846264338327950288

typedef struct {
    int32_t num_species;
    double rcr, rca;
    double eta_r;
    int32_t n_shf_r;
    const double *shf_r;
    double eta_a, zeta;
    int32_t n_shf_a;
    const double *shf_a;
    int32_t n_shf_z;
    const double *shf_z;
    double cos_scale;
} oracle_params;

/* ------------------------------------------------------------------ threads */
int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ------------------------------------------------------------------ step 1: pairs */
/* Triclinic cell (PAPER.md:223 names periodic ML cells): when a lattice is
 * set, `box` arguments are ignored and the displacement is the SHORTEST of x_j - x_i - (na a + nb b + nc c)
 * over the image shifts na, nb, nc in {-2..2} around the fractional-coordinate rounding -- the definition
 * of the minimum image written as a search (125 candidates), not the sequential rint the CUDA path uses.
 * Valid for lattices whose perpendicular widths exceed 2 R_c.  Set / cleared from one thread before a call. */
static int g_tri = 0;
static double g_lat[9], g_inv[9];   /* rows a, b, c; inverse such that frac = v * g_inv (row vector) */

int oracle_set_lattice(const double *lat)
{
    if (!lat) { g_tri = 0; return 0; }
    const double *a = lat, *b = lat + 3, *c = lat + 6;
    double det = a[0] * (b[1] * c[2] - b[2] * c[1]) - a[1] * (b[0] * c[2] - b[2] * c[0])
               + a[2] * (b[0] * c[1] - b[1] * c[0]);
    if (!(fabs(det) > 0.0)) return -1;
    memcpy(g_lat, lat, sizeof(g_lat));
    /* inverse of the matrix with rows a, b, c (cofactors / det) */
    g_inv[0] = (b[1] * c[2] - b[2] * c[1]) / det; g_inv[1] = (a[2] * c[1] - a[1] * c[2]) / det; g_inv[2] = (a[1] * b[2] - a[2] * b[1]) / det;
    g_inv[3] = (b[2] * c[0] - b[0] * c[2]) / det; g_inv[4] = (a[0] * c[2] - a[2] * c[0]) / det; g_inv[5] = (a[2] * b[0] - a[0] * b[2]) / det;
    g_inv[6] = (b[0] * c[1] - b[1] * c[0]) / det; g_inv[7] = (a[1] * c[0] - a[0] * c[1]) / det; g_inv[8] = (a[0] * b[1] - a[1] * b[0]) / det;
    g_tri = 1;
    return 0;
}

static inline void displacement(const float *pos, const float *box, int64_t i, int64_t j, double d[3])
{
    if (g_tri) {
        double v[3], f[3];
        for (int a = 0; a < 3; ++a) v[a] = (double)pos[3 * j + a] - (double)pos[3 * i + a];
        /* fractional coordinates of v, rounded: brings v next to the origin cell */
        for (int k = 0; k < 3; ++k) f[k] = rint(v[0] * g_inv[k] + v[1] * g_inv[3 + k] + v[2] * g_inv[6 + k]);
        for (int a = 0; a < 3; ++a) v[a] -= f[0] * g_lat[a] + f[1] * g_lat[3 + a] + f[2] * g_lat[6 + a];
        double best = -1.0;
        for (int na = -2; na <= 2; ++na)
            for (int nb = -2; nb <= 2; ++nb)
                for (int nc = -2; nc <= 2; ++nc) {
                    double w[3];
                    for (int a = 0; a < 3; ++a) w[a] = v[a] - (na * g_lat[a] + nb * g_lat[3 + a] + nc * g_lat[6 + a]);
                    double r2 = w[0] * w[0] + w[1] * w[1] + w[2] * w[2];
                    if (best < 0.0 || r2 < best) { best = r2; d[0] = w[0]; d[1] = w[1]; d[2] = w[2]; }
                }
        return;
    }
    for (int a = 0; a < 3; ++a) {
        double v = (double)pos[3 * j + a] - (double)pos[3 * i + a];
        if (box) {
            double L = (double)box[a];
            v -= L * rint(v / L);
        }
        d[a] = v;
    }
}

/* Brute force: all i<j, lexicographic order.  Returns the number of pairs found
 * (which may exceed cap; only the first cap are written).  species may be NULL;
 * atoms with species < 0 are padding and belong to no pair (G12). */
int64_t oracle_pairs_brute(const float *pos, const int32_t *species, const float *box,
                           int32_t n, double rc, int32_t *pairs_out, int64_t cap)
{
    int64_t cnt = 0;
    for (int64_t i = 0; i < n; ++i) {
        if (species && species[i] < 0) continue;
        for (int64_t j = i + 1; j < n; ++j) {
            if (species && species[j] < 0) continue;
            double d[3];
            displacement(pos, box, i, j, d);
            double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            if (sqrt(r2) < rc) {
                if (cnt < cap) { pairs_out[2 * cnt] = (int32_t)i; pairs_out[2 * cnt + 1] = (int32_t)j; }
                ++cnt;
            }
        }
    }
    return cnt;
}

/* Cell list (periodic only, every edge >= 3 cells of size >= rc): same pair set as
 * the brute force by construction of the 27-cell stencil; order is by cell, then
 * sorted lexicographically before return. */
typedef struct { int32_t *cell_of; int32_t *start; int32_t *items; int nc[3]; } cell_grid;

static int build_grid(const float *pos, const int32_t *species, const float *box, int32_t n,
                      double rc, cell_grid *g)
{
    int64_t ncell = 1;
    for (int a = 0; a < 3; ++a) {
        g->nc[a] = (int)floor((double)box[a] / rc);
        if (g->nc[a] < 3) return -1;
        ncell *= g->nc[a];
    }
    g->cell_of = (int32_t *)malloc(sizeof(int32_t) * (size_t)n);
    g->start = (int32_t *)calloc((size_t)ncell + 1, sizeof(int32_t));
    g->items = (int32_t *)malloc(sizeof(int32_t) * (size_t)n);
    for (int32_t i = 0; i < n; ++i) {
        if (species && species[i] < 0) { g->cell_of[i] = -1; continue; }
        int c[3];
        for (int a = 0; a < 3; ++a) {
            double L = (double)box[a];
            double x = (double)pos[3 * i + a];
            x -= L * floor(x / L);
            int k = (int)floor(x / L * g->nc[a]);
            if (k >= g->nc[a]) k = g->nc[a] - 1;
            if (k < 0) k = 0;
            c[a] = k;
        }
        int32_t cell = (c[2] * g->nc[1] + c[1]) * g->nc[0] + c[0];
        g->cell_of[i] = cell;
        g->start[cell + 1]++;
    }
    for (int64_t c = 0; c < ncell; ++c) g->start[c + 1] += g->start[c];
    int32_t *fill = (int32_t *)calloc((size_t)ncell, sizeof(int32_t));
    for (int32_t i = 0; i < n; ++i) {
        int32_t cell = g->cell_of[i];
        if (cell < 0) continue;
        g->items[g->start[cell] + fill[cell]++] = i;
    }
    free(fill);
    return 0;
}

static void free_grid(cell_grid *g) { free(g->cell_of); free(g->start); free(g->items); }

static int cmp_pair(const void *a, const void *b)
{
    const int32_t *x = (const int32_t *)a, *y = (const int32_t *)b;
    if (x[0] != y[0]) return x[0] < y[0] ? -1 : 1;
    if (x[1] != y[1]) return x[1] < y[1] ? -1 : 1;
    return 0;
}

int64_t oracle_pairs_cell(const float *pos, const int32_t *species, const float *box,
                          int32_t n, double rc, int32_t *pairs_out, int64_t cap)
{
    cell_grid g;
    if (!box || build_grid(pos, species, box, n, rc, &g) != 0) return -1;
    int64_t cnt = 0;
    for (int32_t i = 0; i < n; ++i) {
        int32_t ci = g.cell_of[i];
        if (ci < 0) continue;
        int cx = ci % g.nc[0], cy = (ci / g.nc[0]) % g.nc[1], cz = ci / (g.nc[0] * g.nc[1]);
        for (int dz = -1; dz <= 1; ++dz)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    int x = (cx + dx + g.nc[0]) % g.nc[0];
                    int y = (cy + dy + g.nc[1]) % g.nc[1];
                    int z = (cz + dz + g.nc[2]) % g.nc[2];
                    int32_t c = (z * g.nc[1] + y) * g.nc[0] + x;
                    for (int32_t q = g.start[c]; q < g.start[c + 1]; ++q) {
                        int32_t j = g.items[q];
                        if (j <= i) continue;
                        double d[3];
                        displacement(pos, box, i, j, d);
                        double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
                        if (sqrt(r2) < rc) {
                            if (cnt < cap) { pairs_out[2 * cnt] = i; pairs_out[2 * cnt + 1] = j; }
                            ++cnt;
                        }
                    }
                }
    }
    free_grid(&g);
    qsort(pairs_out, (size_t)(cnt < cap ? cnt : cap), 2 * sizeof(int32_t), cmp_pair);
    return cnt;
}

/* Per-atom neighbour table for the featurizer: for atom i, entries q in
 * [start[i], start[i+1]) give neighbour index nbr[q], displacement d[3q..], r[q],
 * all with r < rcr, in increasing neighbour index. */
typedef struct { int64_t *start; int32_t *nbr; double *d; double *r; } nbr_table;

static void free_table(nbr_table *t) { free(t->start); free(t->nbr); free(t->d); free(t->r); }

static int build_table(const float *pos, const int32_t *species, const float *box, int32_t n,
                       double rcr, int use_cells, nbr_table *t)
{
    int64_t cap = (int64_t)n * 64 + 64;
    int32_t *pairs = NULL;
    int64_t cnt;
    for (;;) {
        pairs = (int32_t *)malloc(sizeof(int32_t) * 2 * (size_t)cap);
        cnt = use_cells ? oracle_pairs_cell(pos, species, box, n, rcr, pairs, cap)
                        : oracle_pairs_brute(pos, species, box, n, rcr, pairs, cap);
        if (cnt < 0) { free(pairs); return -1; }
        if (cnt <= cap) break;
        free(pairs);
        cap = cnt;
    }
    t->start = (int64_t *)calloc((size_t)n + 1, sizeof(int64_t));
    for (int64_t p = 0; p < cnt; ++p) { t->start[pairs[2 * p] + 1]++; t->start[pairs[2 * p + 1] + 1]++; }
    for (int32_t i = 0; i < n; ++i) t->start[i + 1] += t->start[i];
    t->nbr = (int32_t *)malloc(sizeof(int32_t) * (size_t)(2 * cnt + 1));
    t->d = (double *)malloc(sizeof(double) * 3 * (size_t)(2 * cnt + 1));
    t->r = (double *)malloc(sizeof(double) * (size_t)(2 * cnt + 1));
    int64_t *fill = (int64_t *)calloc((size_t)n, sizeof(int64_t));
    /* pairs are sorted (i asc, j asc): inserting j into i's list and i into j's list in
     * this order leaves every list in increasing neighbour index. */
    for (int pass = 0; pass < 2; ++pass)
        for (int64_t p = 0; p < cnt; ++p) {
            int32_t i = pairs[2 * p], j = pairs[2 * p + 1];
            /* pass 0 fills the "smaller neighbours" (i into j's list), pass 1 the larger ones */
            int32_t a = pass == 0 ? j : i, b = pass == 0 ? i : j;
            int64_t q = t->start[a] + fill[a]++;
            t->nbr[q] = b;
            displacement(pos, box, a, b, &t->d[3 * q]);
            t->r[q] = sqrt(t->d[3 * q] * t->d[3 * q] + t->d[3 * q + 1] * t->d[3 * q + 1] +
                           t->d[3 * q + 2] * t->d[3 * q + 2]);
        }
    free(fill);
    free(pairs);
    return 0;
}

/* ------------------------------------------------------------------ step 2: cutoff */
static inline double fc(double r, double R) { return r < R ? 0.5 * cos(ORACLE_PI * r / R) + 0.5 : 0.0; }
static inline double dfc(double r, double R) { return r < R ? -0.5 * ORACLE_PI / R * sin(ORACLE_PI * r / R) : 0.0; }

int32_t oracle_aev_length(const oracle_params *p)
{
    int S = p->num_species;
    return S * p->n_shf_r + S * (S + 1) / 2 * p->n_shf_a * p->n_shf_z;
}

/* block index of the unordered species pair, row-major upper triangle (G6) */
static inline int pair_block(int s1, int s2, int S)
{
    if (s1 > s2) { int t = s1; s1 = s2; s2 = t; }
    return s1 * (2 * S - s1 - 1) / 2 + s2;
}

/* ------------------------------------------------------------------ steps 3+4: forward
 * pos  f32 [batch][n][3], species i32 [batch][n] (<0 = padding), box f32[3] or NULL,
 * aev  f64 [batch][n][L] (overwritten).  Returns 0, or -1 if the cell list cannot be
 * built (box too small). */
int oracle_aev_forward(const oracle_params *p, const float *pos, const int32_t *species,
                       const float *box, int32_t n, int32_t batch, int use_cells, double *aev)
{
    const int S = p->num_species, nR = p->n_shf_r, nA = p->n_shf_a, nZ = p->n_shf_z;
    const int L = oracle_aev_length(p);
    memset(aev, 0, sizeof(double) * (size_t)batch * (size_t)n * (size_t)L);
    for (int32_t b = 0; b < batch; ++b) {
        const float *X = pos + (size_t)b * n * 3;
        const int32_t *Z = species + (size_t)b * n;
        double *A = aev + (size_t)b * n * L;
        nbr_table t;
        if (build_table(X, Z, box, n, p->rcr, use_cells, &t) != 0) return -1;
#pragma omp parallel for schedule(dynamic, 16)
        for (int32_t i = 0; i < n; ++i) {
            if (Z[i] < 0) continue;
            double *row = A + (size_t)i * L;
            /* step 3: radial */
            for (int64_t q = t.start[i]; q < t.start[i + 1]; ++q) {
                double r = t.r[q];
                int sj = Z[t.nbr[q]];
                double f = fc(r, p->rcr);
                for (int m = 0; m < nR; ++m) {
                    double dr = r - p->shf_r[m];
                    row[sj * nR + m] += 0.25 * exp(-p->eta_r * dr * dr) * f;
                }
            }
            /* step 4: angular, unordered pairs {j,k} with r < rca */
            for (int64_t q1 = t.start[i]; q1 < t.start[i + 1]; ++q1) {
                if (!(t.r[q1] < p->rca)) continue;
                for (int64_t q2 = q1 + 1; q2 < t.start[i + 1]; ++q2) {
                    if (!(t.r[q2] < p->rca)) continue;
                    const double *dj = &t.d[3 * q1], *dk = &t.d[3 * q2];
                    double rj = t.r[q1], rk = t.r[q2];
                    double cosr = (dj[0] * dk[0] + dj[1] * dk[1] + dj[2] * dk[2]) / (rj * rk);
                    double arg = p->cos_scale * cosr;
                    if (arg > 1.0) arg = 1.0;
                    if (arg < -1.0) arg = -1.0;
                    double theta = acos(arg);
                    double rho = 0.5 * (rj + rk);
                    double ff = fc(rj, p->rca) * fc(rk, p->rca);
                    double *blk = row + S * nR + pair_block(Z[t.nbr[q1]], Z[t.nbr[q2]], S) * nA * nZ;
                    for (int a = 0; a < nA; ++a) {
                        double dr = rho - p->shf_a[a];
                        double rad = exp(-p->eta_a * dr * dr);
                        for (int z = 0; z < nZ; ++z) {
                            double ang = pow(1.0 + cos(theta - p->shf_z[z]), p->zeta);
                            blk[a * nZ + z] += pow(2.0, 1.0 - p->zeta) * ang * rad * ff;
                        }
                    }
                }
            }
        }
        free_table(&t);
    }
    return 0;
}

/* ------------------------------------------------------------------ step 5: backward
 * g f32 [batch][n][L] upstream dE/dAEV; forces f64 [batch][n][3] = -dE/dx (G11). */
int oracle_aev_backward(const oracle_params *p, const float *pos, const int32_t *species,
                        const float *box, int32_t n, int32_t batch, int use_cells,
                        const float *g, double *forces)
{
    const int S = p->num_species, nR = p->n_shf_r, nA = p->n_shf_a, nZ = p->n_shf_z;
    const int L = oracle_aev_length(p);
    const double c = p->cos_scale;
    memset(forces, 0, sizeof(double) * (size_t)batch * (size_t)n * 3);
    int nthreads = oracle_max_threads();
    for (int32_t b = 0; b < batch; ++b) {
        const float *X = pos + (size_t)b * n * 3;
        const int32_t *Z = species + (size_t)b * n;
        const float *G = g + (size_t)b * n * L;
        double *F = forces + (size_t)b * n * 3;
        nbr_table t;
        if (build_table(X, Z, box, n, p->rcr, use_cells, &t) != 0) return -1;
        /* gradient accumulators, one private copy per thread, summed in thread order */
        double *grad = (double *)calloc((size_t)nthreads * (size_t)n * 3, sizeof(double));
#pragma omp parallel for schedule(dynamic, 16)
        for (int32_t i = 0; i < n; ++i) {
            if (Z[i] < 0) continue;
#ifdef _OPENMP
            double *gr = grad + (size_t)omp_get_thread_num() * (size_t)n * 3;
#else
            double *gr = grad;
#endif
            const float *grow = G + (size_t)i * L;
            /* radial: dE/dr_ij = sum_m g[i][s_j nR + m] * phi'_m(r) */
            for (int64_t q = t.start[i]; q < t.start[i + 1]; ++q) {
                double r = t.r[q];
                int j = t.nbr[q], sj = Z[j];
                double f = fc(r, p->rcr), df = dfc(r, p->rcr);
                double w = 0.0;
                for (int m = 0; m < nR; ++m) {
                    double dr = r - p->shf_r[m];
                    double e = exp(-p->eta_r * dr * dr);
                    w += (double)grow[sj * nR + m] * 0.25 * e * (-2.0 * p->eta_r * dr * f + df);
                }
                for (int a = 0; a < 3; ++a) {
                    double u = t.d[3 * q + a] / r;
                    gr[3 * j + a] += w * u;
                    gr[3 * i + a] -= w * u;
                }
            }
            /* angular */
            for (int64_t q1 = t.start[i]; q1 < t.start[i + 1]; ++q1) {
                if (!(t.r[q1] < p->rca)) continue;
                for (int64_t q2 = q1 + 1; q2 < t.start[i + 1]; ++q2) {
                    if (!(t.r[q2] < p->rca)) continue;
                    const double *dj = &t.d[3 * q1], *dk = &t.d[3 * q2];
                    double rj = t.r[q1], rk = t.r[q2];
                    int j = t.nbr[q1], k = t.nbr[q2];
                    double uj[3], uk[3];
                    for (int a = 0; a < 3; ++a) { uj[a] = dj[a] / rj; uk[a] = dk[a] / rk; }
                    double cosr = uj[0] * uk[0] + uj[1] * uk[1] + uj[2] * uk[2];
                    double arg = c * cosr;
                    if (arg > 1.0) arg = 1.0;
                    if (arg < -1.0) arg = -1.0;
                    double theta = acos(arg);
                    double sin2 = 1.0 - arg * arg;
                    /* d(theta)/d(cos_raw) = -c/sin(theta); at the cone point the
                     * perpendicular part is defined as 0 (G2) */
                    double dtheta_dcos = sin2 < 1e-12 ? 0.0 : -c / sqrt(sin2);
                    double rho = 0.5 * (rj + rk);
                    double fj = fc(rj, p->rca), fk = fc(rk, p->rca);
                    double dfj = dfc(rj, p->rca), dfk = dfc(rk, p->rca);
                    const float *gb = grow + S * nR + pair_block(Z[j], Z[k], S) * nA * nZ;
                    double pref = pow(2.0, 1.0 - p->zeta);
                    double dE_dtheta = 0.0, dE_drho = 0.0, dE_dfj = 0.0, dE_dfk = 0.0;
                    for (int a = 0; a < nA; ++a) {
                        double dr = rho - p->shf_a[a];
                        double rad = exp(-p->eta_a * dr * dr);
                        double drad = -2.0 * p->eta_a * dr * rad;
                        for (int z = 0; z < nZ; ++z) {
                            double base = 1.0 + cos(theta - p->shf_z[z]);
                            double ang = pow(base, p->zeta);
                            double dang = p->zeta * pow(base, p->zeta - 1.0) * (-sin(theta - p->shf_z[z]));
                            double gg = (double)gb[a * nZ + z] * pref;
                            dE_dtheta += gg * dang * rad * fj * fk;
                            dE_drho += gg * ang * drad * fj * fk;
                            dE_dfj += gg * ang * rad * fk;
                            dE_dfk += gg * ang * rad * fj;
                        }
                    }
                    double dE_dcos = dE_dtheta * dtheta_dcos;
                    double dE_drj = 0.5 * dE_drho + dE_dfj * dfj;
                    double dE_drk = 0.5 * dE_drho + dE_dfk * dfk;
                    for (int a = 0; a < 3; ++a) {
                        double gj = dE_drj * uj[a] + dE_dcos * (uk[a] - cosr * uj[a]) / rj;
                        double gk = dE_drk * uk[a] + dE_dcos * (uj[a] - cosr * uk[a]) / rk;
                        gr[3 * j + a] += gj;
                        gr[3 * k + a] += gk;
                        gr[3 * i + a] -= gj + gk;
                    }
                }
            }
        }
        for (int th = 0; th < nthreads; ++th)
            for (int64_t q = 0; q < (int64_t)n * 3; ++q) F[q] -= grad[(size_t)th * (size_t)n * 3 + q];
        free(grad);
        free_table(&t);
    }
    return 0;
}

/* ------------------------------------------------------------------ step 6: per-species MLP
 * One network applied to n_rows input rows x f64 [n_rows][dims[0]].
 * W[l] f64 [dims[l]][dims[l+1]] row-major ("[in][out]"), b[l] f64 [dims[l+1]].
 * Hidden layers CELU_alpha, last layer linear, dims[n_layers] must be 1.
 * energy f64 [n_rows]; grad_x f64 [n_rows][dims[0]] = dE_row/dx (may be NULL). */
static inline double celu(double x, double alpha) { return x > 0.0 ? x : alpha * (exp(x / alpha) - 1.0); }
static inline double dcelu(double x, double alpha) { return x > 0.0 ? 1.0 : exp(x / alpha); }

int oracle_mlp(int32_t n_rows, const double *x, int32_t n_layers, const int32_t *dims,
               const double *const *W, const double *const *b, double alpha,
               double *energy, double *grad_x)
{
    if (dims[n_layers] != 1) return -1;
    int maxd = 0;
    for (int l = 0; l <= n_layers; ++l) if (dims[l] > maxd) maxd = dims[l];
#pragma omp parallel
    {
        /* pre-activations z[l] kept for the backward chain */
        double *z = (double *)malloc(sizeof(double) * (size_t)n_layers * (size_t)maxd);
        double *h = (double *)malloc(sizeof(double) * (size_t)maxd);
        double *gcur = (double *)malloc(sizeof(double) * (size_t)maxd);
        double *gnext = (double *)malloc(sizeof(double) * (size_t)maxd);
#pragma omp for schedule(static)
        for (int32_t row = 0; row < n_rows; ++row) {
            const double *in = x + (size_t)row * dims[0];
            for (int l = 0; l < n_layers; ++l) {
                const double *src = l == 0 ? in : h;
                double *zl = z + (size_t)l * maxd;
                for (int o = 0; o < dims[l + 1]; ++o) {
                    double acc = b[l][o];
                    for (int k = 0; k < dims[l]; ++k) acc += src[k] * W[l][(size_t)k * dims[l + 1] + o];
                    zl[o] = acc;
                }
                if (l < n_layers - 1)
                    for (int o = 0; o < dims[l + 1]; ++o) h[o] = celu(zl[o], alpha);
            }
            energy[row] = z[(size_t)(n_layers - 1) * maxd];
            if (!grad_x) continue;
            /* transposed chain, seed dE/dz_last = 1 */
            gcur[0] = 1.0;
            for (int l = n_layers - 1; l >= 0; --l) {
                /* gcur = dE/dz[l] (size dims[l+1]);  dE/dh[l-1] = W[l] gcur */
                for (int k = 0; k < dims[l]; ++k) {
                    double acc = 0.0;
                    for (int o = 0; o < dims[l + 1]; ++o) acc += W[l][(size_t)k * dims[l + 1] + o] * gcur[o];
                    gnext[k] = acc;
                }
                if (l > 0) {
                    const double *zp = z + (size_t)(l - 1) * maxd;
                    for (int k = 0; k < dims[l]; ++k) gcur[k] = gnext[k] * dcelu(zp[k], alpha);
                } else {
                    for (int k = 0; k < dims[0]; ++k) grad_x[(size_t)row * dims[0] + k] = gnext[k];
                }
            }
        }
        free(z); free(h); free(gcur); free(gnext);
    }
    return 0;
}
