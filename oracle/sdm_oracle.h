/* sdm_oracle.h -- plain CPU oracle for one Super-Droplet Method coalescence timestep.
 *
 * TEST INFRASTRUCTURE ONLY.  This is the slow, obviously-correct restatement of the method
 * from the paper (Bartman & Arabas, arXiv 2101.06318; cited as PAPER.md:<line>), used by
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
 * It shares no code with the CUDA path (paper_2101_06318_b200/csrc) and the product never
 * calls it.  Single-threaded, fp64, compiled with -O2 -ffp-contract=off (no FMA contraction).
 *
 * All pointers are HOST pointers.  Conventions where the paper is silent are the readings
 * R1..R17 of DESIGN.md ("Readings of the paper").
 *
 * Pins (tests/test_oracle_*.py): Philox known answers, the paper's worked example
 * (PAPER.md:106), the xi_k = 1 special case, hand-worked 4-droplet examples
 * (tests/golden/), invariants, Golovin closed-form moments, the one-step mean-field identity
 * by brute force, exhaustive enumeration on 2..4-droplet cells, filter/sum semantics.
 * Parity unpinned: none of the functions below is without a pin; the key-tie rule (R7) is
 * pinned only through orc_permutation() with hand-made keys, never through Philox output.
 */
#ifndef SDM_ORACLE_H
#define SDM_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_KERNEL_GOLOVIN = 0, ORC_KERNEL_GRAVITATIONAL = 1, ORC_KERNEL_GRAVITATIONAL_TABULATED = 2, ORC_KERNEL_USER = 3 };

/* Philox4x32-10 (Salmon et al. 2011), one block.  DESIGN.md R6. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* Step "urand": per storage index sid[i] one Philox block ->
 * key64[i] (sort key) and ucand[i] in [0,1).  sid == NULL means sid[i] = i. */
void orc_rng(int64_t n, const int64_t *sid, uint64_t seed, uint64_t step,
             uint64_t *key64, double *ucand);

/* cell_start = exclusive scan of per-cell counts, length n_cell+1.
 * Returns 0, or -1 if a cell id is out of range. */
int orc_cell_start(int64_t n, const int32_t *cell_id, int32_t n_cell, int32_t *cell_start);

/* idx = positions 0..n-1 sorted ascending by (cell_id, key64, sid). */
void orc_permutation(int64_t n, const int32_t *cell_id, const uint64_t *key64,
                     const int64_t *sid, int32_t *idx);

/* The specified cube root (R10): fixed sequence of IEEE-754 double operations. */
double orc_cbrt_spec(double x);

/* Coalescence kernel a(v_j, v_k) [m^3/s]: Golovin b*(v_j+v_k) or the
 * gravitational kernel of BASELINE.json config 3 (PAPER.md:326 gives no formula). */
double orc_kernel(int32_t type, double kparam, double vj, double vk);

/* NEXT-2, "potentially user-supplied kernel code" (second kernel family of Fig. 8):
 * ORC_KERNEL_USER evaluates a(v_j, v_k) = fn(v_j, v_k, params) with a caller-supplied C function (v_j: the volume of the
 * pair member with the larger multiplicity, as for the built-in kernels); kparam is ignored.  The function must be
 * compiled without FMA contraction if its result is to be compared bit for bit.  One function per process. */
typedef double (*orc_user_kernel_fn)(double vj, double vk, const double *params);
void orc_set_user_kernel(orc_user_kernel_fn fn, const double *params, int32_t n_params);

/* NEXT-2: user-supplied collection efficiency E(r_1, r_2) for ORC_KERNEL_GRAVITATIONAL_TABULATED
 * (a = kparam * E(r_j, r_k) * pi * (r_j + r_k)^2 * |w_j - w_k|): n_r x n_r table,
 * row-major, on the strictly increasing radius grid r_grid; bilinear, clamped outside (R16).
 * Returns 0, -1 on an invalid table.  The table is copied. */
int orc_set_efficiency_table(int32_t n_r, const double *r_grid, const double *E);
double orc_efficiency(double rj, double rk);

/* Eq. 3, evaluated in the routine order of Fig. 3. */
double orc_pair_probability(double K, int64_t xi_max, int64_t n_s, double dt, double dV);

/* gamma = ceil(p - phi) in its floor form (R4) capped by
 * floor(xi_j/xi_k) (Eq. 4).  Requires xi_j >= xi_k > 0. */
int64_t orc_gamma_tilde(double p, double u, int64_t xi_j, int64_t xi_k);

/* Fig. 5 body / Eqs. 5-6 for one pair and one
 * extensive attribute, given the UNCAPPED gamma.  (a, b) is (first-in-pair, second). */
void orc_collide_pair(int64_t *xi_a, double *v_a, int64_t *xi_b, double *v_b, int64_t gamma);

/* The same for n_attr extensive attributes, rows of a row-major (n_attr, ld) array, row 0 = volume
 * (PAPER.md:138, 145-147, 271-287); a, b index the droplets (a = first-in-pair). */
void orc_collide_pair_attr(int64_t *xi, double *attr, int32_t n_attr, int64_t ld, int64_t a, int64_t b,
                           int64_t gamma);

/* One coalescence step (Fig. 3 steps 1-3) in place on (xi, v).
 * idx_out[n], cell_start_out[n_cell+1] may be NULL.  sid may be NULL (identity).
 * n_events_out (may be NULL): number of pairs with gamma_tilde > 0.
 * Returns 0, -1 on invalid input. */
int orc_step(int64_t n, int64_t *xi, double *v, const int32_t *cell_id, int32_t n_cell,
             const int64_t *sid, double dt, double dV, int32_t kernel, double kparam,
             uint64_t seed, uint64_t step, int32_t *idx_out, int32_t *cell_start_out,
             int64_t *n_events_out);

/* orc_step with n_attr >= 1 extensive attributes (row 0 = volume, which alone enters Eq. 3). */
int orc_step_attr(int64_t n, int64_t *xi, double *attr, int32_t n_attr, int64_t ld,
                  const int32_t *cell_id, int32_t n_cell,
                  const int64_t *sid, double dt, double dV, int32_t kernel, double kparam,
                  uint64_t seed, uint64_t step, int32_t *idx_out, int32_t *cell_start_out,
                  int64_t *n_events_out);

/* Step 0: drop xi == 0, keep storage order.  Returns survivors. */
int64_t orc_remove_zero_attr(int64_t n, int64_t *xi, double *attr, int32_t n_attr, int64_t ld,
                             int32_t *cell_id);
int64_t orc_remove_zero(int64_t n, int64_t *xi, double *v, int32_t *cell_id);

/* Moments M_k = sum xi v^k, k = 0,1,2 (R13).  per_cell == 0:
 * three scalars; else arrays of n_cell.  fp64 sums are compensated (Neumaier). */
void orc_moments(int64_t n, const int64_t *xi, const double *v, const int32_t *cell_id,
                 int32_t n_cell, int32_t per_cell, int64_t *m0, double *m1, double *m2);

/* NEXT-3: binned mass density per unit ln r, out[n_bins]; bins by volume edges
 * v_edges[n_bins+1] (strictly increasing), widths dlnr[n_bins], n_smooth passes of a centered 5-bin running
 * mean truncated at the ends (R17). */
void orc_spectrum(int64_t n, const int64_t *xi, const double *v, int32_t n_bins, const double *v_edges,
                  const double *dlnr, double rho, double V, int32_t n_smooth, double *out);

#ifdef __cplusplus
}
#endif
#endif
