/* sdm_oracle.c -- plain CPU oracle for one SDM coalescence timestep.  See sdm_oracle.h.
 *
 * TEST INFRASTRUCTURE ONLY: never linked into, imported by or called from the product path.
 * Written from the paper (PAPER.md = arXiv 2101.06318) step by step, in the paper's order and
 * notation; no blocking, fusion or reordering.  Build: gcc -O2 -ffp-contract=off -fPIC -shared.
 */
#include "sdm_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------------------------
 * Philox4x32-10 (R6; the paper only says "random numbers").
 * One round:  (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2,
 *             c' = { hi1^c1^k0, lo1, hi0^c3^k1, lo0 };  the key is bumped by the Weyl
 * constants between rounds (before rounds 2..10).
 * ------------------------------------------------------------------------------------------ */
#define PHILOX_M0 0xD2511F53u
#define PHILOX_M1 0xCD9E8D57u
#define PHILOX_W0 0x9E3779B9u
#define PHILOX_W1 0xBB67AE85u

void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += PHILOX_W0; k1 += PHILOX_W1; }
        uint64_t p0 = (uint64_t)PHILOX_M0 * c0;
        uint64_t p1 = (uint64_t)PHILOX_M1 * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* DESIGN.md R6: counter = {sid lo, sid hi, step lo, step hi}, key = {seed lo, seed hi};
 * sort key = words 0-1, pair uniform = 53 top bits of words 2-3, times 2^-53 (phi ~ U[0,1),
 * PAPER.md:102). */
void orc_rng(int64_t n, const int64_t *sid, uint64_t seed, uint64_t step,
             uint64_t *key64, double *ucand)
{
    for (int64_t i = 0; i < n; ++i) {
        uint64_t s = (uint64_t)(sid ? sid[i] : i);
        uint32_t ctr[4] = { (uint32_t)s, (uint32_t)(s >> 32), (uint32_t)step, (uint32_t)(step >> 32) };
        uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
        uint32_t w[4];
        orc_philox4x32_10(ctr, key, w);
        key64[i] = (uint64_t)w[0] | ((uint64_t)w[1] << 32);
        uint64_t bits = (uint64_t)w[2] | ((uint64_t)w[3] << 32);
        ucand[i] = (double)(bits >> 11) * 0x1.0p-53;
    }
}

/* PAPER.md:151 "cell_start = Storage(N_CELL + 1, int)". */
int orc_cell_start(int64_t n, const int32_t *cell_id, int32_t n_cell, int32_t *cell_start)
{
    for (int32_t c = 0; c <= n_cell; ++c) cell_start[c] = 0;
    for (int64_t i = 0; i < n; ++i) {
        if (cell_id[i] < 0 || cell_id[i] >= n_cell) return -1;
        cell_start[cell_id[i] + 1] += 1;                 /* count of cell c at slot c+1 */
    }
    for (int32_t c = 0; c < n_cell; ++c) cell_start[c + 1] += cell_start[c];
    return 0;
}

/* Step 1: the GPU backend of the paper permutes by sorting on a
 * random key with the cell id as the major key.  Ties on the key are broken by storage index
 * (R7). */
typedef struct { int32_t cell; uint64_t key; int64_t sid; int32_t pos; } orc_rec_t;

static int orc_rec_cmp(const void *pa, const void *pb)
{
    const orc_rec_t *a = (const orc_rec_t *)pa, *b = (const orc_rec_t *)pb;
    if (a->cell != b->cell) return a->cell < b->cell ? -1 : 1;
    if (a->key != b->key) return a->key < b->key ? -1 : 1;
    if (a->sid != b->sid) return a->sid < b->sid ? -1 : 1;
    return 0;
}

void orc_permutation(int64_t n, const int32_t *cell_id, const uint64_t *key64,
                     const int64_t *sid, int32_t *idx)
{
    orc_rec_t *rec = (orc_rec_t *)malloc((size_t)(n > 0 ? n : 1) * sizeof(orc_rec_t));
    for (int64_t i = 0; i < n; ++i) {
        rec[i].cell = cell_id[i];
        rec[i].key = key64[i];
        rec[i].sid = sid ? sid[i] : i;
        rec[i].pos = (int32_t)i;
    }
    qsort(rec, (size_t)n, sizeof(orc_rec_t), orc_rec_cmp);
    for (int64_t i = 0; i < n; ++i) idx[i] = rec[i].pos;
    free(rec);
}

/* DESIGN.md R10: cube root as a fixed sequence of IEEE double operations (libm's cbrt is not
 * correctly rounded, so it cannot be part of a bit-exact contract).
 *   y0 = bits -> double( MAGIC - bits(x)/3 )            ~ x^(-1/3), |rel err| < 3.5e-2
 *   4 x Newton for x^(-1/3):  y <- y * (4/3 - (1/3) * (x*(y*y*y)))
 *   r  = (x*y)*y                                           ~ x^(1/3)
 *   r <- r - ((r*r)*r - x) * ((y*y) * (1/3))               one Newton step for r^3 = x
 * Every product and sum is rounded separately (no FMA).  Result within 1 ulp of the true
 * cube root for positive normal x (checked in tests/test_oracle_kernels.py). */
double orc_cbrt_spec(double x)
{
    uint64_t bits;
    memcpy(&bits, &x, sizeof bits);
    uint64_t ybits = 0x553EEEEEEEEEF000ull - bits / 3ull;
    double y;
    memcpy(&y, &ybits, sizeof y);
    const double c43 = 0x1.5555555555555p+0;   /* 4/3 rounded */
    const double c13 = 0x1.5555555555555p-2;   /* 1/3 rounded */
    for (int it = 0; it < 4; ++it) {
        double t = y * y;
        t = t * y;
        t = x * t;
        t = c13 * t;
        t = c43 - t;
        y = y * t;
    }
    double r = x * y;
    r = r * y;
    double d = r * r;
    d = d * r;
    d = d - x;
    double h = y * y;
    h = h * c13;
    d = d * h;
    r = r - d;
    return r;
}

/* Terminal velocity of BASELINE.json config 3 (Rogers-Yau three-regime fit); R9:
 * the middle branch owns r = 40 um, the top branch owns r = 600 um. */
static double orc_terminal_velocity(double r)
{
    if (r < 40e-6) { double t = 1.19e8 * r; return t * r; }
    if (r < 600e-6) return 8e3 * r;
    return 220.0 * sqrt(r);
}

/* NEXT-2 ("potentially user-supplied kernel code", kernels "after Berry 1967" with
 * collection efficiencies): a user-supplied collection-efficiency table E(r_1, r_2) on a rectangular radius
 * grid r_0 < r_1 < ... < r_{n-1}, bilinear in (r_1, r_2), clamped outside the grid (R16).
 * One table per process: the oracle is single-threaded test infrastructure. */
static int32_t orc_eff_n = 0;
static double *orc_eff_grid = NULL, *orc_eff_tab = NULL;

int orc_set_efficiency_table(int32_t n_r, const double *r_grid, const double *E)
{
    if (n_r < 2 || !r_grid || !E) return -1;
    for (int32_t i = 0; i < n_r; ++i) {
        if (!(r_grid[i] > 0.0) || !isfinite(r_grid[i])) return -1;
        if (i > 0 && !(r_grid[i] > r_grid[i - 1])) return -1;
    }
    for (int64_t i = 0; i < (int64_t)n_r * n_r; ++i)
        if (!(E[i] >= 0.0) || !isfinite(E[i])) return -1;
    free(orc_eff_grid); free(orc_eff_tab);
    orc_eff_grid = (double *)malloc((size_t)n_r * sizeof(double));
    orc_eff_tab = (double *)malloc((size_t)n_r * n_r * sizeof(double));
    memcpy(orc_eff_grid, r_grid, (size_t)n_r * sizeof(double));
    memcpy(orc_eff_tab, E, (size_t)n_r * n_r * sizeof(double));
    orc_eff_n = n_r;
    return 0;
}

/* grid interval of r and the weight inside it: i in [0, n-2], t in [0, 1] */
static void orc_eff_locate(double r, int32_t *i_out, double *t_out)
{
    const int32_t n = orc_eff_n;
    if (r < orc_eff_grid[0]) { *i_out = 0; *t_out = 0.0; return; }
    if (r >= orc_eff_grid[n - 1]) { *i_out = n - 2; *t_out = 1.0; return; }
    int32_t i = 0;
    while (orc_eff_grid[i + 1] <= r) ++i;             /* grid[i] <= r < grid[i+1] */
    double num = r - orc_eff_grid[i];
    double den = orc_eff_grid[i + 1] - orc_eff_grid[i];
    *i_out = i;
    *t_out = num / den;
}

double orc_efficiency(double rj, double rk)
{
    int32_t i, k;
    double t, u;
    orc_eff_locate(rj, &i, &t);
    orc_eff_locate(rk, &k, &u);
    const int32_t n = orc_eff_n;
    double e00 = orc_eff_tab[(int64_t)i * n + k], e10 = orc_eff_tab[(int64_t)(i + 1) * n + k];
    double e01 = orc_eff_tab[(int64_t)i * n + k + 1], e11 = orc_eff_tab[(int64_t)(i + 1) * n + k + 1];
    double d0 = e10 - e00;
    double e0 = e00 + t * d0;                         /* along r_j at r-grid column k   */
    double d1 = e11 - e01;
    double e1 = e01 + t * d1;                         /* along r_j at column k+1         */
    double d = e1 - e0;
    return e0 + u * d;                                /* along r_k                       */
}

static orc_user_kernel_fn orc_user_fn = NULL;
static double orc_user_params[16];

void orc_set_user_kernel(orc_user_kernel_fn fn, const double *params, int32_t n_params)
{
    orc_user_fn = fn;
    for (int32_t i = 0; i < 16; ++i) orc_user_params[i] = (params && i < n_params) ? params[i] : 0.0;
}

double orc_kernel(int32_t type, double kparam, double vj, double vk)
{
    if (type == ORC_KERNEL_USER) return orc_user_fn(vj, vk, orc_user_params);
    if (type == ORC_KERNEL_GOLOVIN) {
        /* a(v1, v2) = b (v1 + v2) */
        double s = vj + vk;
        return kparam * s;
    }
    /* K = E * pi * (r_j + r_k)^2 * |w_j - w_k|, evaluated left to right; r = cbrt(3 v / (4 pi)) */
    const double c = 0x1.e8ec8a4aeacc4p-3;     /* 3/(4 pi) */
    const double pi = 0x1.921fb54442d18p+1;
    double rj = orc_cbrt_spec(vj * c);
    double rk = orc_cbrt_spec(vk * c);
    double wj = orc_terminal_velocity(rj);
    double wk = orc_terminal_velocity(rk);
    double s = rj + rk;
    double s2 = s * s;
    double E = kparam;
    if (type == ORC_KERNEL_GRAVITATIONAL_TABULATED) E = kparam * orc_efficiency(rj, rk);
    double K = E * pi;
    K = K * s2;
    K = K * fabs(wj - wk);
    return K;
}

/* Eq. 3:  p = a(v_j,v_k) * max(xi_j,xi_k) * [(n^2-n)/2]/floor(n/2) * dt/dV,
 * in the order of the routines kernel -> times_max -> normalize. */
double orc_pair_probability(double K, int64_t xi_max, int64_t n_s, double dt, double dV)
{
    double p = K * (double)xi_max;                               /* times_max */
    int64_t all_pairs = (n_s * (n_s - 1)) / 2;                   /* (n^2 - n)/2 */
    int64_t cand_pairs = n_s / 2;                                /* floor(n/2) */
    double norm = (dt / dV) * ((double)all_pairs / (double)cand_pairs);
    return p * norm;                                             /* normalize */
}

/* gamma = ceil(p - phi), phi ~ U[0,1) == floor(p) + [phi < p - floor(p)]
 * (R4); gamma_tilde = min(gamma, floor(xi_j/xi_k)) (Eq. 4).
 * The comparison with q is made in double first so that a huge p never overflows the
 * conversion to int64 (R8). */
int64_t orc_gamma_tilde(double p, double u, int64_t xi_j, int64_t xi_k)
{
    /* DESIGN.md R20: Eq. 3 is a probability-like number >= 0 for every kernel of the paper.  A p that is not > 0
     * (negative or NaN: only user-supplied kernel code can produce one) means "no event" -- without this the
     * cast of NaN below would be undefined, and a negative gamma would make multiplicities grow.  For p = 0 the
     * lines below give 0 as well, so nothing changes for p >= 0. */
    if (!(p > 0.0)) return 0;
    double fl = floor(p);
    double gamma = fl + ((u < p - fl) ? 1.0 : 0.0);
    int64_t q = xi_j / xi_k;
    if (fl >= (double)q) return q;
    int64_t g = (int64_t)gamma;
    return g < q ? g : q;
}

/* Fig. 5 for one pair (a = first-in-pair, b = second) and n_attr extensive
 * attributes stored as rows of a 2-D row-major array with leading dimension ld (PAPER.md:138, 145:
 * "attributes = Storage((N_ATTR, N_SD), float)"; the loop "for attr in range(len(attributes))" at
 * PAPER.md:271-287).  Row 0 is the volume (volume_view). */
void orc_collide_pair_attr(int64_t *xi, double *attr, int32_t n_attr, int64_t ld, int64_t a, int64_t b,
                           int64_t gamma)
{
    int64_t j = a, k = b;
    if (xi[j] < xi[k]) { j = b; k = a; }
    if (xi[k] == 0) return;                           /* DESIGN.md R11: zero-xi partner */
    int64_t q = xi[j] / xi[k];
    int64_t g = gamma < q ? gamma : q;                /* PAPER.md:260 (Eq. 4) */
    if (g == 0) return;
    int64_t new_n = xi[j] - g * xi[k];
    if (new_n > 0) {                                  /* Eq. 5 */
        xi[j] = new_n;
        for (int32_t r = 0; r < n_attr; ++r) {
            double *A = attr + (int64_t)r * ld;
            double t = (double)g * A[j];
            A[k] = A[k] + t;
        }
    } else {                                          /* Eq. 6 */
        xi[j] = xi[k] / 2;
        xi[k] = xi[k] - xi[j];
        for (int32_t r = 0; r < n_attr; ++r) {
            double *A = attr + (int64_t)r * ld;
            double t = A[j] * (double)g;
            A[j] = t + A[k];
            A[k] = A[j];
        }
    }
}

/* One pair, one attribute, operands by pointer (the form the pair-level pins use). */
void orc_collide_pair(int64_t *xi_a, double *v_a, int64_t *xi_b, double *v_b, int64_t gamma)
{
    int64_t xi[2] = { *xi_a, *xi_b };
    double A[2] = { *v_a, *v_b };
    orc_collide_pair_attr(xi, A, 1, 2, 0, 1, gamma);
    *xi_a = xi[0]; *xi_b = xi[1]; *v_a = A[0]; *v_b = A[1];
}

int orc_step_attr(int64_t n, int64_t *xi, double *attr, int32_t n_attr, int64_t ld,
                  const int32_t *cell_id, int32_t n_cell,
                  const int64_t *sid, double dt, double dV, int32_t kernel, double kparam,
                  uint64_t seed, uint64_t step, int32_t *idx_out, int32_t *cell_start_out,
                  int64_t *n_events_out)
{
    if (n < 0 || n_cell < 1 || n_attr < 1 || ld < n) return -1;
    double *v = attr;                                 /* volume_view = attributes[0, :] */
    uint64_t *key64 = (uint64_t *)malloc((size_t)(n + 1) * sizeof(uint64_t));
    double *ucand = (double *)malloc((size_t)(n + 1) * sizeof(double));
    int32_t *idx = (int32_t *)malloc((size_t)(n + 1) * sizeof(int32_t));
    int32_t *cell_start = (int32_t *)malloc((size_t)(n_cell + 1) * sizeof(int32_t));
    int64_t n_events = 0;
    int rc = 0;

    /* step 1: random numbers, cell-wise shuffling */
    orc_rng(n, sid, seed, step, key64, ucand);
    if (orc_cell_start(n, cell_id, n_cell, cell_start) != 0) { rc = -1; goto done; }
    orc_permutation(n, cell_id, key64, sid, idx);

    /* steps 2-3 for every candidate pair (2m, 2m+1) of every cell */
    for (int32_t c = 0; c < n_cell; ++c) {
        int64_t s = cell_start[c];
        int64_t n_s = cell_start[c + 1] - s;
        for (int64_t m = 0; m < n_s / 2; ++m) {
            int32_t a = idx[s + 2 * m];               /* first-in-pair */
            int32_t b = idx[s + 2 * m + 1];
            int32_t j = a, k = b;
            if (xi[j] < xi[k]) { j = b; k = a; }
            if (xi[k] == 0) continue;                 /* DESIGN.md R11 */
            double K = orc_kernel(kernel, kparam, v[j], v[k]);
            double p = orc_pair_probability(K, xi[j], n_s, dt, dV);
            double u = ucand[a];                      /* DESIGN.md R6: uniform of the first member */
            int64_t g = orc_gamma_tilde(p, u, xi[j], xi[k]);
            if (g == 0) continue;
            n_events += 1;
            /* gamma_tilde <= floor(xi_j/xi_k), so passing it as gamma leaves it unchanged */
            orc_collide_pair_attr(xi, attr, n_attr, ld, a, b, g);
        }
    }
    if (idx_out) memcpy(idx_out, idx, (size_t)n * sizeof(int32_t));
    if (cell_start_out) memcpy(cell_start_out, cell_start, (size_t)(n_cell + 1) * sizeof(int32_t));
    if (n_events_out) *n_events_out = n_events;
done:
    free(key64); free(ucand); free(idx); free(cell_start);
    return rc;
}

int orc_step(int64_t n, int64_t *xi, double *v, const int32_t *cell_id, int32_t n_cell,
             const int64_t *sid, double dt, double dV, int32_t kernel, double kparam,
             uint64_t seed, uint64_t step, int32_t *idx_out, int32_t *cell_start_out,
             int64_t *n_events_out)
{
    return orc_step_attr(n, xi, v, 1, n, cell_id, n_cell, sid, dt, dV, kernel, kparam, seed, step,
                         idx_out, cell_start_out, n_events_out);
}

/* Step 0: filter, order preserved (R12); every attribute row moves
 * with its droplet. */
int64_t orc_remove_zero_attr(int64_t n, int64_t *xi, double *attr, int32_t n_attr, int64_t ld,
                             int32_t *cell_id)
{
    int64_t m = 0;
    for (int64_t i = 0; i < n; ++i) {
        if (xi[i] != 0) {
            xi[m] = xi[i]; cell_id[m] = cell_id[i];
            for (int32_t r = 0; r < n_attr; ++r) attr[(int64_t)r * ld + m] = attr[(int64_t)r * ld + i];
            m += 1;
        }
    }
    return m;
}

int64_t orc_remove_zero(int64_t n, int64_t *xi, double *v, int32_t *cell_id)
{
    return orc_remove_zero_attr(n, xi, v, 1, n, cell_id);
}

/* Neumaier compensated accumulation: sum += x with a running error term. */
static void orc_acc(double *sum, double *comp, double x)
{
    double t = *sum + x;
    if (fabs(*sum) >= fabs(x)) *comp += (*sum - t) + x;
    else                       *comp += (x - t) + *sum;
    *sum = t;
}

void orc_moments(int64_t n, const int64_t *xi, const double *v, const int32_t *cell_id,
                 int32_t n_cell, int32_t per_cell, int64_t *m0, double *m1, double *m2)
{
    int32_t nout = per_cell ? n_cell : 1;
    double *c1 = (double *)calloc((size_t)nout, sizeof(double));
    double *c2 = (double *)calloc((size_t)nout, sizeof(double));
    for (int32_t c = 0; c < nout; ++c) { m0[c] = 0; m1[c] = 0.0; m2[c] = 0.0; }
    for (int64_t i = 0; i < n; ++i) {
        int32_t c = per_cell ? cell_id[i] : 0;
        double xv = (double)xi[i] * v[i];             /* xi v   */
        double xvv = xv * v[i];                       /* xi v^2 */
        m0[c] += xi[i];
        orc_acc(&m1[c], &c1[c], xv);
        orc_acc(&m2[c], &c2[c], xvv);
    }
    for (int32_t c = 0; c < nout; ++c) { m1[c] += c1[c]; m2[c] += c2[c]; }
    free(c1); free(c2);
}

/* NEXT-3 (Fig. 6): "the mass of droplets per unit of ln r ... aggregating super-particle
 * multiplicities onto a grid of ca. 100 bins, and smoothing the result twice with a running average with a
 * centered window spanning five bins".  Readings (R17): bin b holds the droplets with
 * v_edges[b] <= v < v_edges[b+1]; its value is (sum xi*v) * rho / V / dlnr[b]  [kg m^-3 per unit ln r], the
 * bin widths dlnr[b] = ln(r_{b+1}/r_b) being an INPUT (so that no logarithm has to agree between
 * implementations); each smoothing pass replaces a bin by the mean of the bins b-2..b+2 that exist (the
 * window is truncated at the ends), summed left to right. */
void orc_spectrum(int64_t n, const int64_t *xi, const double *v, int32_t n_bins, const double *v_edges,
                  const double *dlnr, double rho, double V, int32_t n_smooth, double *out)
{
    double *comp = (double *)calloc((size_t)n_bins, sizeof(double));
    double *tmp = (double *)calloc((size_t)n_bins, sizeof(double));
    for (int32_t b = 0; b < n_bins; ++b) out[b] = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        if (!(v[i] >= v_edges[0]) || !(v[i] < v_edges[n_bins])) continue;
        int32_t b = 0;
        while (v_edges[b + 1] <= v[i]) ++b;           /* v_edges[b] <= v < v_edges[b+1] */
        double m = (double)xi[i] * v[i];
        orc_acc(&out[b], &comp[b], m);
    }
    for (int32_t b = 0; b < n_bins; ++b) {
        double s = out[b] + comp[b];
        s = s * rho;
        s = s / V;
        out[b] = s / dlnr[b];
    }
    for (int32_t pass = 0; pass < n_smooth; ++pass) {
        for (int32_t b = 0; b < n_bins; ++b) {
            int32_t lo = b - 2 < 0 ? 0 : b - 2, hi = b + 2 > n_bins - 1 ? n_bins - 1 : b + 2;
            double s = 0.0;
            for (int32_t k = lo; k <= hi; ++k) s = s + out[k];
            tmp[b] = s / (double)(hi - lo + 1);
        }
        memcpy(out, tmp, (size_t)n_bins * sizeof(double));
    }
    free(comp); free(tmp);
}
