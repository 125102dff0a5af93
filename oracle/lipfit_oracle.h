/*
 * lipfit_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU restatement of what the LipFit hot path
 * computes, written from the paper's formulas (PAPER.md = the text of
 * arxiv/paper_2606_04670).  It shares no code, header, table or helper with
 * the CUDA path under paper_2606_04670_b200/, and only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call it.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): hand-computed worked
 * example P0 (tests/golden/p0_worked_example.txt), interpolation, sandwich,
 * enclosure of the generator, Lipschitz and monotone properties, 1-D closed
 * forms, scipy cdist / cKDTree special cases, metamorphic relations, N=2
 * smoothing closed form, finite-difference gradient, brute force on tiny
 * inputs; for region monotonicity (oracle_bounds_region, R26) the limits a = b and
 * a = -inf, b = +inf, admissible 1-D functions (enclosure and attainment) and an
 * independent NumPy integration of the "may grow" indicator along the way.  The one thing left "parity unpinned" by design is the LBFGS
 * TRAJECTORY of smoothing (the minimiser itself is unique and is pinned).
 *
 * All inputs are fp32 arrays on the host (the same arrays the GPU gets); every
 * intermediate and every floating-point output is double.
 *
 * Notation: delta_i = xq_i - x^k_i (query minus datum);
 *   mask s_i in {-1,0,+1}; weights w_i >= 0; norm p in {1 (L1), 2 (L2), 3 (Linf)}
 *   u_i = w_i*|delta_i|            if s_i == 0, else w_i*max( s_i*delta_i, 0)
 *   l_i = w_i*|delta_i|            if s_i == 0, else w_i*max(-s_i*delta_i, 0)
 *   D^u = ||u||_p = d_s(x^k, x),  D^l = ||l||_p = d_s(x, x^k)
 * (Eq.(4) PAPER.md:142 with the sign convention of PAPER.md:140; reading R1.)
 */
#ifndef LIPFIT_ORACLE_H
#define LIPFIT_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Eq.(2),(3) PAPER.md:103-116 with the distance of Eq.(4) PAPER.md:142.
 * upper/lower/g: double[Q], each may be NULL.  Returns 0, or <0 on bad args. */
int oracle_bounds(const float* X, const float* y, int64_t N, int32_t d,
                  const float* Xq, int64_t Q, double M,
                  const int32_t* mono_mask, int32_t norm, const float* weights,
                  double* upper, double* lower, double* g);

/* k nearest data per query by distance (PAPER.md:179 d_(1), d_(2), ...):
 * side 0 = symmetric weighted norm (mask ignored), +1 = D^u, -1 = D^l.
 * Ties are broken by the lower index.  idx: int32[Q*k], dist: double[Q*k]. */
int oracle_knn(const float* X, int64_t N, int32_t d, const float* Xq, int64_t Q,
               const int32_t* mono_mask, int32_t side, int32_t norm,
               const float* weights, int32_t k, int32_t* idx, double* dist);

/* Eq.(7), literally the two sums over ordered pairs i != k, with
 * d_ik of constraint (5) = d_s(x^k,x^i) and of (6) = d_s(x^i,x^k) (reading R12);
 * eps: double[N]; F: double*; grad: double[N] (analytic dF/deps), may be NULL. */
int oracle_smooth_objective(const float* X, const float* y, int64_t N, int32_t d,
                            double M, const int32_t* mono_mask, int32_t norm,
                            const float* weights, double p, const double* eps,
                            double* F, double* grad);

/* max over ordered pairs i != k of violation (z_i - z_k - M d_s(x^k,x^i))_+ ,
 * z = y + eps (eps may be NULL = 0): 0 iff the data are consistent with
 * constraints (5),(6) PAPER.md:191-193. */
int oracle_max_violation(const float* X, const float* y, int64_t N, int32_t d,
                         double M, const int32_t* mono_mask, int32_t norm,
                         const float* weights, const double* eps, double* out);

/* Eq.(7) restricted to listed rows: grad_rows[r] = dF/deps_{rows[r]}, f_rows[r] = row share of F
 * (may be NULL).  For spot checks at sizes where the full double loop is unaffordable. */
int oracle_smooth_rows(const float* X, const float* y, int64_t N, int32_t d, double M,
                       const int32_t* mono_mask, int32_t norm, const float* weights, double p,
                       const double* eps, const int64_t* rows, int64_t nrows, double* grad_rows,
                       double* f_rows);

/* Smallest Lipschitz constant consistent with the data:
 * max over ordered pairs with y_i > y_k of (y_i - y_k) / d_s(x^k, x^i); +inf if such a pair has
 * zero distance; 0 if there is none. */
int oracle_lipschitz_constant(const float* X, const float* y, int64_t N, int32_t d,
                              const int32_t* mono_mask, int32_t norm, const float* weights,
                              double* out);

/* ---- Local Lipschitz interpolation, PAPER.md:169-183 (radial symmetric distance) ---------------- */
/* knots[j-1] = nearest-rank j/J quantile of the S sampled inter-point distances D(x^{pair_i}, x^{pair_k}). */
int oracle_distance_quantiles(const float* X, int64_t N, int32_t d, int32_t norm, const float* weights,
                              const int32_t* pair_i, const int32_t* pair_k, int64_t S, int32_t J,
                              double* knots);
/* table[k*J+j] = value of the step function M_k on (t_{j-1}, t_j] (last knot = +inf). */
int oracle_local_lipschitz(const float* X, const float* y, int64_t N, int32_t d, int32_t norm,
                           const float* weights, const double* knots, int32_t J, double* table);
/* Rows rows[0..R) of the same table only: table_rows[r*J+j] = M_{rows[r]} on (t_{j-1}, t_j]. */
int oracle_local_lipschitz_rows(const float* X, const float* y, int64_t N, int32_t d, int32_t norm,
                                const float* weights, const double* knots, int32_t J, const int64_t* rows,
                                int64_t R, double* table_rows);
/* Eq.(2),(3) with M -> M_k(D(x, x^k)). */
int oracle_values_local(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                        int32_t norm, const float* weights, const double* knots, int32_t J,
                        const double* table, double* upper, double* lower, double* g);

/* k > 1 approximation: upper = sum_j wk[j] * (j-th smallest of y^k + M D^u),
 * lower = sum_j wk[j] * (j-th largest of y^k - M D^l), j = 1..k; wk: float[k]. */
int oracle_bounds_topk(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                       double M, const int32_t* mono_mask, int32_t norm, const float* weights, int32_t k,
                       const float* wk, double* upper, double* lower, double* g);

/* Eq.(2),(3) under monotonicity on parts of the domain (cases I-IV; reading R26):
 * mon[i] in {0,1,2,3,4} (0 = unrestricted, 1..4 = case I..IV), a[i] <= b[i] (a = -inf / b = +inf allowed)
 * for every coordinate with mon[i] != 0.  Per coordinate, walking from x^k_i to x_i,
 *   u_i = w_i (length of the way in AB + length in A / B where f may grow in the direction of travel),
 *   l_i = w_i (length of the way in AB + length in A / B where f may fall in the direction of travel),
 * upper = min_k (y^k + M ||u||_p), lower = max_k (y^k - M ||l||_p), g their midpoint. */
int oracle_bounds_region(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                         double M, const int32_t* mon, const float* a, const float* b, int32_t norm,
                         const float* weights, double* upper, double* lower, double* g);

int oracle_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
