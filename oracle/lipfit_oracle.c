/*
 * lipfit_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see lipfit_oracle.h).
 *
 * Plain double-precision CPU code following PAPER.md equation by equation.
 * No blocking, fusion or reordering beyond what the formulas state; the only
 * parallelism is an OpenMP `parallel for` over independent queries / rows.
 * Build: gcc -O2 -fopenmp -shared -fPIC (oracle/build.py).
 */
#include "lipfit_oracle.h"

#include <math.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static int check_common(const void* X, int64_t N, int32_t d, const int32_t* mask,
                        int32_t norm, const float* w) {
    if (!X) return -1;
    if (d < 1) return -2;
    if (N < 1) return -3;
    if (norm < 1 || norm > 3) return -4;
    for (int i = 0; i < d; ++i) {
        if (mask && (mask[i] < -1 || mask[i] > 1)) return -4;
        if (w && !(w[i] >= 0.0f && isfinite(w[i]))) return -4;
    }
    return 0;
}

/* The two one-sided distances between a point x ("query" role) and a datum
 * xk.  Eq.(4): dist = ||(x - x^k)_+|| on the monotone-increasing
 * coordinates; PAPER.md:140 fixes which side serves which bound (R1):
 *   *Du = d_s(x^k, x) uses (x - x^k)_+   -> goes into H^upper,
 *   *Dl = d_s(x, x^k) uses (x^k - x)_+   -> goes into H^lower.
 * s_i = -1 is the mirrored coordinate (R2); s_i = 0 contributes |delta| to
 * both (R4).  The norm is ||w (.) v||_p, p in {1,2,inf} (R3). */
static void one_sided_distances(const float* x, const float* xk, int32_t d,
                                const int32_t* mask, int32_t norm, const float* w,
                                double* Du, double* Dl) {
    double au = 0.0, al = 0.0;
    for (int i = 0; i < d; ++i) {
        double delta = (double)x[i] - (double)xk[i];
        int s = mask ? mask[i] : 0;
        double cu, cl;
        if (s == 0) {
            cu = fabs(delta);
            cl = fabs(delta);
        } else {
            cu = fmax((double)s * delta, 0.0);
            cl = fmax(-(double)s * delta, 0.0);
        }
        double wi = w ? (double)w[i] : 1.0;
        cu *= wi;
        cl *= wi;
        if (norm == 1) {
            au += cu;
            al += cl;
        } else if (norm == 2) {
            au += cu * cu;
            al += cl * cl;
        } else {
            au = fmax(au, cu);
            al = fmax(al, cl);
        }
    }
    if (norm == 2) {
        au = sqrt(au);
        al = sqrt(al);
    }
    *Du = au;
    *Dl = al;
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Eq.(2): H^upper(x) = min_k (y^k + M dist), H^lower(x) = max_k (y^k - M dist);
 * Eq.(3): g = (H^lower + H^upper)/2.  PAPER.md:103-116. */
int oracle_bounds(const float* X, const float* y, int64_t N, int32_t d,
                  const float* Xq, int64_t Q, double M,
                  const int32_t* mono_mask, int32_t norm, const float* weights,
                  double* upper, double* lower, double* g) {
    int rc = check_common(X, N, d, mono_mask, norm, weights);
    if (rc) return rc;
    if (!y || (Q > 0 && !Xq)) return -1;
    if (Q < 0) return -3;
    if (!(M >= 0.0) || !isfinite(M)) return -4;
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < Q; ++q) {
        double U = INFINITY, L = -INFINITY;
        for (int64_t k = 0; k < N; ++k) {
            double Du, Dl;
            one_sided_distances(Xq + q * d, X + k * d, d, mono_mask, norm, weights, &Du, &Dl);
            double hi = (double)y[k] + M * Du;
            double lo = (double)y[k] - M * Dl;
            if (hi < U) U = hi;
            if (lo > L) L = lo;
        }
        if (upper) upper[q] = U;
        if (lower) lower[q] = L;
        if (g) g[q] = 0.5 * (U + L);
    }
    return 0;
}

/* k nearest by distance; keep the k smallest (dist, index) seen so far in
 * ascending order by straight insertion.  PAPER.md:179 (d_(1) <= d_(2) ...). */
int oracle_knn(const float* X, int64_t N, int32_t d, const float* Xq, int64_t Q,
               const int32_t* mono_mask, int32_t side, int32_t norm,
               const float* weights, int32_t k, int32_t* idx, double* dist) {
    int rc = check_common(X, N, d, mono_mask, norm, weights);
    if (rc) return rc;
    if ((Q > 0 && !Xq) || !idx || !dist) return -1;
    if (Q < 0 || k < 1 || k > N) return -3;
    if (side < -1 || side > 1) return -4;
    const int32_t* m = (side == 0) ? NULL : mono_mask; /* side 0: symmetric, mask ignored (R6) */
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < Q; ++q) {
        int32_t* bi = idx + q * k;
        double* bd = dist + q * k;
        int32_t have = 0;
        for (int64_t j = 0; j < N; ++j) {
            double Du, Dl;
            one_sided_distances(Xq + q * d, X + j * d, d, m, norm, weights, &Du, &Dl);
            double dj = (side < 0) ? Dl : Du;
            /* position: after every kept (dist,idx) that is <= (dj,j); j grows, so
             * equal distances keep the earlier (lower) index first (R7). */
            int32_t pos = have;
            while (pos > 0 && bd[pos - 1] > dj) --pos;
            if (pos >= k) continue;
            int32_t last = (have < k) ? have : k - 1;
            for (int32_t t = last; t > pos; --t) {
                bd[t] = bd[t - 1];
                bi[t] = bi[t - 1];
            }
            bd[pos] = dj;
            bi[pos] = (int32_t)j;
            if (have < k) ++have;
        }
    }
    return 0;
}

/* Eq.(7) PAPER.md:197:
 *   F = (1/p)||eps||^2
 *     + sum_{i!=k} ((y_i - y_k - M d_ik - (eps_k - eps_i))_+)^2      [from (5)]
 *     + sum_{i!=k} ((y_k - y_i - M d'_ik + eps_k - eps_i)_+)^2       [from (6)]
 * with d_ik = d_s(x^k,x^i) (upper-bound distance of datum k seen from x^i) and
 * d'_ik = d_s(x^i,x^k) (lower-bound distance), reading R12.  Gradient by the
 * chain rule, term by term:  d/deps_i of the (5)-term (i,k) is +2A_ik, of the
 * (5)-term (k,i) is -2A_ki, of the (6)-term (i,k) is -2B_ik, of (k,i) +2B_ki. */
int oracle_smooth_objective(const float* X, const float* y, int64_t N, int32_t d,
                            double M, const int32_t* mono_mask, int32_t norm,
                            const float* weights, double p, const double* eps,
                            double* F, double* grad) {
    int rc = check_common(X, N, d, mono_mask, norm, weights);
    if (rc) return rc;
    if (!y || !eps || !F) return -1;
    if (!(M >= 0.0) || !isfinite(M) || !(p > 0.0)) return -4;
    double total = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : total)
    for (int64_t i = 0; i < N; ++i) {
        double zi = (double)y[i] + eps[i];
        double gi = 2.0 * eps[i] / p;
        double fi = eps[i] * eps[i] / p;
        for (int64_t k = 0; k < N; ++k) {
            if (k == i) continue;
            double zk = (double)y[k] + eps[k];
            double d_ik, dp_ik; /* point x^i against datum x^k */
            one_sided_distances(X + i * d, X + k * d, d, mono_mask, norm, weights, &d_ik, &dp_ik);
            double d_ki, dp_ki; /* point x^k against datum x^i */
            one_sided_distances(X + k * d, X + i * d, d, mono_mask, norm, weights, &d_ki, &dp_ki);
            double A_ik = fmax(zi - zk - M * d_ik, 0.0);  /* (5) at (i,k) */
            double B_ik = fmax(zk - zi - M * dp_ik, 0.0); /* (6) at (i,k) */
            double A_ki = fmax(zk - zi - M * d_ki, 0.0);  /* (5) at (k,i) */
            double B_ki = fmax(zi - zk - M * dp_ki, 0.0); /* (6) at (k,i) */
            fi += A_ik * A_ik + B_ik * B_ik; /* the two (i,k) terms of the sums */
            gi += 2.0 * A_ik - 2.0 * A_ki - 2.0 * B_ik + 2.0 * B_ki;
        }
        total += fi;
        if (grad) grad[i] = gi;
    }
    *F = total;
    return 0;
}

int oracle_max_violation(const float* X, const float* y, int64_t N, int32_t d,
                         double M, const int32_t* mono_mask, int32_t norm,
                         const float* weights, const double* eps, double* out) {
    int rc = check_common(X, N, d, mono_mask, norm, weights);
    if (rc) return rc;
    if (!y || !out) return -1;
    double worst = 0.0;
#pragma omp parallel for schedule(static) reduction(max : worst)
    for (int64_t i = 0; i < N; ++i) {
        double zi = (double)y[i] + (eps ? eps[i] : 0.0);
        for (int64_t k = 0; k < N; ++k) {
            if (k == i) continue;
            double zk = (double)y[k] + (eps ? eps[k] : 0.0);
            double Du, Dl;
            one_sided_distances(X + i * d, X + k * d, d, mono_mask, norm, weights, &Du, &Dl);
            double v = zi - zk - M * Du;
            if (v > worst) worst = v;
        }
    }
    *out = worst;
    return 0;
}

/* The same Eq.(7), restricted to a list of rows i (full-size spot checks): for each
 * listed i, grad_rows = dF/deps_i and f_rows = eps_i^2/p + sum_{k!=i} (A_ik^2 + B_ik^2), i.e. row
 * i's share of F (F = sum over ALL i of that share).  Statement by statement the inner loop of
 * oracle_smooth_objective. */
int oracle_smooth_rows(const float* X, const float* y, int64_t N, int32_t d, double M,
                       const int32_t* mono_mask, int32_t norm, const float* weights, double p,
                       const double* eps, const int64_t* rows, int64_t nrows, double* grad_rows,
                       double* f_rows) {
    int rc = check_common(X, N, d, mono_mask, norm, weights);
    if (rc) return rc;
    if (!y || !eps || !rows || !grad_rows) return -1;
    if (!(M >= 0.0) || !isfinite(M) || !(p > 0.0)) return -4;
    for (int64_t r = 0; r < nrows; ++r)
        if (rows[r] < 0 || rows[r] >= N) return -3;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < nrows; ++r) {
        int64_t i = rows[r];
        double zi = (double)y[i] + eps[i];
        double gi = 2.0 * eps[i] / p;
        double fi = eps[i] * eps[i] / p;
        for (int64_t k = 0; k < N; ++k) {
            if (k == i) continue;
            double zk = (double)y[k] + eps[k];
            double d_ik, dp_ik, d_ki, dp_ki;
            one_sided_distances(X + i * d, X + k * d, d, mono_mask, norm, weights, &d_ik, &dp_ik);
            one_sided_distances(X + k * d, X + i * d, d, mono_mask, norm, weights, &d_ki, &dp_ki);
            double A_ik = fmax(zi - zk - M * d_ik, 0.0);
            double B_ik = fmax(zk - zi - M * dp_ik, 0.0);
            double A_ki = fmax(zk - zi - M * d_ki, 0.0);
            double B_ki = fmax(zi - zk - M * dp_ki, 0.0);
            fi += A_ik * A_ik + B_ik * B_ik;
            gi += 2.0 * A_ik - 2.0 * A_ki - 2.0 * B_ik + 2.0 * B_ki;
        }
        grad_rows[r] = gi;
        if (f_rows) f_rows[r] = fi;
    }
    return 0;
}

/* Smallest Lipschitz constant consistent with the data ("all pairwise distances
 * and then the ratios |y_i - y_k| / dist(x^i, x^k)"): the least M for which constraint (5)
 * z_i <= z_k + M d_s(x^k, x^i) holds for every ordered pair,
 *     L = max_{i != k, y_i > y_k} (y_i - y_k) / d_s(x^k, x^i).
 * Without monotonicity d_s is symmetric and this is max |y_i - y_k| / ||x^i - x^k||.  A pair with
 * y_i > y_k at zero distance makes the data inconsistent for every M: +infinity.  N = 1 or all
 * y_i <= y_k wherever it matters: 0. */
int oracle_lipschitz_constant(const float* X, const float* y, int64_t N, int32_t d,
                              const int32_t* mono_mask, int32_t norm, const float* weights,
                              double* out) {
    int rc = check_common(X, N, d, mono_mask, norm, weights);
    if (rc) return rc;
    if (!y || !out) return -1;
    double best = 0.0;
#pragma omp parallel for schedule(static) reduction(max : best)
    for (int64_t i = 0; i < N; ++i) {
        for (int64_t k = 0; k < N; ++k) {
            if (k == i) continue;
            double dy = (double)y[i] - (double)y[k];
            if (!(dy > 0.0)) continue;
            double Du, Dl;
            one_sided_distances(X + i * d, X + k * d, d, mono_mask, norm, weights, &Du, &Dl);
            double ratio = (Du > 0.0) ? dy / Du : INFINITY;
            if (ratio > best) best = ratio;
        }
    }
    *out = best;
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * Local Lipschitz interpolation, PAPER.md:169-183 (section 4.3), readings R20-R23 of DESIGN.md.
 * Radial (symmetric, weighted) distance D(a,b) = ||w (a - b)||_p: "an approximation to M(x) based on
 * radial distances from data x^k".
 * ------------------------------------------------------------------------------------------- */
static double radial_distance(const float* a, const float* b, int32_t d, int32_t norm, const float* w) {
    double Du, Dl;
    one_sided_distances(a, b, d, NULL, norm, w, &Du, &Dl);
    return Du;
}

static int cmp_double(const void* a, const void* b) {
    double x = *(const double*)a, y = *(const double*)b;
    return (x > y) - (x < y);
}

/* Spline knots: "quantiles of the distribution of distances from a random point x_k, approximated from
 * a sample of interpoint distances".  The sample is the list of index pairs
 * (pair_i[s], pair_k[s]); knot j (1-based) is the nearest-rank j/J quantile of the S sampled distances,
 * i.e. the sorted sample at index ceil(j S / J) - 1 (R20). */
int oracle_distance_quantiles(const float* X, int64_t N, int32_t d, int32_t norm, const float* weights,
                              const int32_t* pair_i, const int32_t* pair_k, int64_t S, int32_t J,
                              double* knots) {
    int rc = check_common(X, N, d, NULL, norm, weights);
    if (rc) return rc;
    if (!pair_i || !pair_k || !knots) return -1;
    if (S < 1 || J < 1 || J > S) return -3;
    double* ds = (double*)malloc(sizeof(double) * (size_t)S);
    if (!ds) return -6;
    for (int64_t s = 0; s < S; ++s) {
        if (pair_i[s] < 0 || pair_i[s] >= N || pair_k[s] < 0 || pair_k[s] >= N) {
            free(ds);
            return -3;
        }
        ds[s] = radial_distance(X + (int64_t)pair_i[s] * d, X + (int64_t)pair_k[s] * d, d, norm, weights);
    }
    qsort(ds, (size_t)S, sizeof(double), cmp_double);
    for (int32_t j = 1; j <= J; ++j) {
        int64_t idx = ((int64_t)j * S + J - 1) / J - 1; /* ceil(j S / J) - 1 */
        knots[j - 1] = ds[idx];
    }
    free(ds);
    return 0;
}

/* Per-datum non-decreasing step function M_k: table[k*J + j] is the value of M_k on
 * (t_{j-1}, t_j]:
 *     max( |y_k - y_(1)| / d_(1),  max_{i != k, D(x^k,x^i) <= t_j} |y_k - y_i| / D(x^k,x^i) ),
 * where d_(1) is the distance from x^k to its closest neighbour ("the first segment ... has the value
 * |y_k - y_(1)|/d_(1) ... the smallest value consistent with the data"; several closest neighbours at
 * the same distance: the largest of their ratios) and the LAST knot is treated as +infinity, so the
 * last column is the maximum over all data (R21).  A different value at zero distance gives +infinity;
 * an equal value at zero distance (a duplicate) is ignored. */
/* One row of the table: the step function M_k of datum k, see oracle_local_lipschitz. */
static void local_lipschitz_row(const float* X, const float* y, int64_t N, int32_t d, int32_t norm,
                                const float* weights, const double* knots, int32_t J, int64_t k, double* M) {
    for (int32_t j = 0; j < J; ++j) M[j] = 0.0;
    double dmin = INFINITY, rnn = 0.0;
    for (int64_t i = 0; i < N; ++i) {
        if (i == k) continue;
        double D = radial_distance(X + k * d, X + i * d, d, norm, weights);
        double dy = fabs((double)y[k] - (double)y[i]);
        if (D == 0.0 && dy == 0.0) continue; /* duplicate datum */
        double ratio = (D > 0.0) ? dy / D : INFINITY;
        if (D < dmin) {
            dmin = D;
            rnn = ratio;
        } else if (D == dmin && ratio > rnn) {
            rnn = ratio;
        }
        for (int32_t j = 0; j < J; ++j)
            if ((j == J - 1 || D <= knots[j]) && ratio > M[j]) M[j] = ratio;
    }
    for (int32_t j = 0; j < J; ++j)
        if (rnn > M[j]) M[j] = rnn;
}

int oracle_local_lipschitz(const float* X, const float* y, int64_t N, int32_t d, int32_t norm,
                           const float* weights, const double* knots, int32_t J, double* table) {
    int rc = check_common(X, N, d, NULL, norm, weights);
    if (rc) return rc;
    if (!y || !knots || !table) return -1;
    if (J < 1) return -3;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < N; ++k)
        local_lipschitz_row(X, y, N, d, norm, weights, knots, J, k, table + k * J);
    return 0;
}

/* The same rows for a list of data only (full-size parity samples): table_rows[r*J + j] = M_{rows[r]}. */
int oracle_local_lipschitz_rows(const float* X, const float* y, int64_t N, int32_t d, int32_t norm,
                                const float* weights, const double* knots, int32_t J, const int64_t* rows,
                                int64_t R, double* table_rows) {
    int rc = check_common(X, N, d, NULL, norm, weights);
    if (rc) return rc;
    if (!y || !knots || !table_rows || (R > 0 && !rows)) return -1;
    if (J < 1 || R < 0) return -3;
    for (int64_t r = 0; r < R; ++r)
        if (rows[r] < 0 || rows[r] >= N) return -3;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < R; ++r)
        local_lipschitz_row(X, y, N, d, norm, weights, knots, J, rows[r], table_rows + r * J);
    return 0;
}

/* Eq.(2),(3) "with global constant M replaced with M_k(||x - x^k||)":
 *   upper = min_k (y_k + M_k(D) D),  lower = max_k (y_k - M_k(D) D),  D = D(x, x^k),
 * M_k(D) = table[k*J + b], b the first knot index with D <= t_b (the last one if none). */
int oracle_values_local(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                        int32_t norm, const float* weights, const double* knots, int32_t J,
                        const double* table, double* upper, double* lower, double* g) {
    int rc = check_common(X, N, d, NULL, norm, weights);
    if (rc) return rc;
    if (!y || !knots || !table || (Q > 0 && !Xq)) return -1;
    if (J < 1 || Q < 0) return -3;
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < Q; ++q) {
        double U = INFINITY, L = -INFINITY;
        for (int64_t k = 0; k < N; ++k) {
            double D = radial_distance(Xq + q * d, X + k * d, d, norm, weights);
            int32_t b = J - 1;
            for (int32_t j = 0; j < J - 1; ++j)
                if (D <= knots[j]) {
                    b = j;
                    break;
                }
            double Mk = table[k * J + b];
            double MD = (D == 0.0) ? 0.0 : Mk * D; /* M_k may be +inf at a duplicate: inf * 0 := 0 */
            double hi = (double)y[k] + MD, lo = (double)y[k] - MD;
            if (hi < U) U = hi;
            if (lo > L) L = lo;
        }
        if (upper) upper[q] = U;
        if (lower) lower[q] = L;
        if (g) g[q] = 0.5 * (U + L);
    }
    return 0;
}

/* Approximation with k > 1 ("Extra features" 2; PAPER.md:226 `values(query, LC, model, k)`):
 * "a weighting vector w in R^k_+ ... the weights of the 'nearest' neighbour, second nearest and so on, so
 * that both upper and lower bound are calculated using k neighbours", evaluated with torch.topk
 * (PAPER.md:206).  Reading R24: with u_(1) <= u_(2) <= ... the sorted values y^k + M D^u and
 * l_(1) >= l_(2) >= ... the sorted values y^k - M D^l,
 *     upper = sum_j w_j u_(j),   lower = sum_j w_j l_(j),   g = (upper + lower) / 2,   j = 1..k.
 * k = 1, w = (1) is Eq.(2),(3). */
static int cmp_double_desc(const void* a, const void* b) { return -cmp_double(a, b); }

int oracle_bounds_topk(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                       double M, const int32_t* mono_mask, int32_t norm, const float* weights, int32_t k,
                       const float* wk, double* upper, double* lower, double* g) {
    int rc = check_common(X, N, d, mono_mask, norm, weights);
    if (rc) return rc;
    if (!y || !wk || (Q > 0 && !Xq)) return -1;
    if (Q < 0 || k < 1 || k > N) return -3;
    if (!(M >= 0.0) || !isfinite(M)) return -4;
    int bad = 0;
#pragma omp parallel
    {
        double* hi = (double*)malloc(sizeof(double) * (size_t)N);
        double* lo = (double*)malloc(sizeof(double) * (size_t)N);
        if (!hi || !lo) {
#pragma omp atomic write
            bad = 1;
        } else {
#pragma omp for schedule(static)
            for (int64_t q = 0; q < Q; ++q) {
                for (int64_t j = 0; j < N; ++j) {
                    double Du, Dl;
                    one_sided_distances(Xq + q * d, X + j * d, d, mono_mask, norm, weights, &Du, &Dl);
                    hi[j] = (double)y[j] + M * Du;
                    lo[j] = (double)y[j] - M * Dl;
                }
                qsort(hi, (size_t)N, sizeof(double), cmp_double);
                qsort(lo, (size_t)N, sizeof(double), cmp_double_desc);
                double U = 0.0, L = 0.0;
                for (int32_t j = 0; j < k; ++j) {
                    U += (double)wk[j] * hi[j];
                    L += (double)wk[j] * lo[j];
                }
                if (upper) upper[q] = U;
                if (lower) lower[q] = L;
                if (g) g[q] = 0.5 * (U + L);
            }
        }
        free(hi);
        free(lo);
    }
    return bad ? -6 : 0;
}


/* ---- Monotonicity on parts of the domain, PAPER.md:147-167 (section 4.2), reading R26 of DESIGN.md ----
 * Per coordinate i the line is cut into A: t <= a_i, AB: a_i <= t <= b_i, B: t >= b_i, and
 *   mon_i = 0: unrestricted,        1: case I   (increasing on A and B),  2: case II (decreasing on A and B),
 *           3: case III (decreasing on A, increasing on B),               4: case IV (increasing on A, decreasing on B);
 * AB is unrestricted in every case.  The paper withholds the formula ("can be expressed through components
 * of the distance vector"); R26 derives it.  Walking coordinate i from the datum's x^k_i to
 * the query's x_i, f can only GROW on the part of the way where it is not known to fall in the direction
 * of travel, and can only FALL on the part where it is not known to grow:
 *   u_i = w_i * (length of the way inside AB
 *                + length inside A if f may grow there in the direction of travel
 *                + length inside B if f may grow there in the direction of travel),
 *   l_i = the same with "fall" for "grow",
 *   f(x) <= y^k + M ||u||_p,   f(x) >= y^k - M ||l||_p,   then Eq.(2),(3) unchanged.
 * "f may grow in the direction of travel" = travelling up through an increasing region, or down through a
 * decreasing one.  a_i = -inf / b_i = +inf are allowed (empty A / empty B). */
static void region_distances(const float* x, const float* xk, int32_t d, const int32_t* mon,
                             const float* a, const float* b, int32_t norm, const float* w,
                             double* Du, double* Dl) {
    double au = 0.0, al = 0.0;
    for (int i = 0; i < d; ++i) {
        double from = (double)xk[i], to = (double)x[i];
        double lo = fmin(from, to), hi = fmax(from, to);
        int m = mon ? mon[i] : 0;
        double cu, cl;
        if (m == 0) {
            cu = hi - lo;
            cl = hi - lo;
        } else {
            double ai = (double)a[i], bi = (double)b[i];
            double lenA = fmax(0.0, fmin(hi, ai) - lo);            /* part of [lo, hi] inside A  */
            double lenB = fmax(0.0, hi - fmax(lo, bi));            /* part inside B              */
            double lenM = fmax(0.0, fmin(hi, bi) - fmax(lo, ai));  /* part inside AB             */
            int incA = (m == 1 || m == 4), incB = (m == 1 || m == 3); /* f increasing on A / on B */
            int up = (to >= from);                                 /* direction of travel        */
            int growA = up ? incA : !incA, growB = up ? incB : !incB;
            cu = lenM + (growA ? lenA : 0.0) + (growB ? lenB : 0.0);
            cl = lenM + (growA ? 0.0 : lenA) + (growB ? 0.0 : lenB);
        }
        double wi = w ? (double)w[i] : 1.0;
        cu *= wi;
        cl *= wi;
        if (norm == 1) {
            au += cu;
            al += cl;
        } else if (norm == 2) {
            au += cu * cu;
            al += cl * cl;
        } else {
            au = fmax(au, cu);
            al = fmax(al, cl);
        }
    }
    if (norm == 2) {
        au = sqrt(au);
        al = sqrt(al);
    }
    *Du = au;
    *Dl = al;
}

int oracle_bounds_region(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                         double M, const int32_t* mon, const float* a, const float* b, int32_t norm,
                         const float* weights, double* upper, double* lower, double* g) {
    int rc = check_common(X, N, d, NULL, norm, weights);
    if (rc) return rc;
    if (!y || (Q > 0 && !Xq)) return -1;
    if (Q < 0) return -3;
    if (!(M >= 0.0) || !isfinite(M)) return -4;
    for (int i = 0; i < d; ++i) {
        int m = mon ? mon[i] : 0;
        if (m < 0 || m > 4) return -4;
        if (m != 0 && (!a || !b || !(a[i] <= b[i]))) return -4; /* also rejects NaN */
    }
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < Q; ++q) {
        double U = INFINITY, L = -INFINITY;
        for (int64_t k = 0; k < N; ++k) {
            double Du, Dl;
            region_distances(Xq + q * d, X + k * d, d, mon, a, b, norm, weights, &Du, &Dl);
            double hi = (double)y[k] + M * Du;
            double lo = (double)y[k] - M * Dl;
            if (hi < U) U = hi;
            if (lo > L) L = lo;
        }
        if (upper) upper[q] = U;
        if (lower) lower[q] = L;
        if (g) g[q] = 0.5 * (U + L);
    }
    return 0;
}
