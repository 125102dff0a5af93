// lbfgs.cpp -- host LBFGS (two-loop recursion) + strong-Wolfe line search (bracket / zoom with
// safeguarded cubic interpolation).  See lbfgs.h for the readings this encodes.
#include "lbfgs.h"

#include <algorithm>
#include <cmath>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace lipfit {
namespace {

// Vector kernels of the recursion.  Long vectors (config 5: n = 2e5, 40 history vectors) are cut into a FIXED
// number of chunks that OpenMP threads share; every chunk is summed sequentially and the partial sums are added
// in chunk order, so the results do not depend on the number of threads (same bits on any host).
constexpr int kChunks = 64;
constexpr size_t kParallelFrom = 1 << 15;

inline int host_threads(size_t n) {
#ifdef _OPENMP
    if (n < kParallelFrom) return 1;
    const int t = omp_get_max_threads();
    return t < 1 ? 1 : (t > 16 ? 16 : t);
#else
    (void)n;
    return 1;
#endif
}

template <class F>  // F(begin, end) -> partial sum of the chunk
double chunked_sum(size_t n, const F& f) {
    if (n < kParallelFrom) return f(static_cast<size_t>(0), n);
    double part[kChunks];
    const size_t step = (n + kChunks - 1) / kChunks;
    const int nt = host_threads(n);
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (int c = 0; c < kChunks; ++c) {
        const size_t b = std::min(n, static_cast<size_t>(c) * step), e = std::min(n, b + step);
        part[c] = f(b, e);
    }
    double s = 0.0;
    for (int c = 0; c < kChunks; ++c) s += part[c];
    return s;
}

double dot(const std::vector<double>& a, const std::vector<double>& b) {
    const double* pa = a.data();
    const double* pb = b.data();
    return chunked_sum(a.size(), [=](size_t i0, size_t i1) {
        double s = 0.0;
        for (size_t i = i0; i < i1; ++i) s += pa[i] * pb[i];
        return s;
    });
}
// d += a * v, then returns dot(w, d) (w may be null: returns 0): one pass instead of two
double axpy_dot(std::vector<double>& d, double a, const std::vector<double>& v, const std::vector<double>* w) {
    double* pd = d.data();
    const double* pv = v.data();
    const double* pw = w ? w->data() : nullptr;
    return chunked_sum(d.size(), [=](size_t i0, size_t i1) {
        double s = 0.0;
        for (size_t i = i0; i < i1; ++i) {
            pd[i] += a * pv[i];
            if (pw) s += pw[i] * pd[i];
        }
        return s;
    });
}
// d *= a, then returns dot(w, d)
double scale_dot(std::vector<double>& d, double a, const std::vector<double>* w) {
    double* pd = d.data();
    const double* pw = w ? w->data() : nullptr;
    return chunked_sum(d.size(), [=](size_t i0, size_t i1) {
        double s = 0.0;
        for (size_t i = i0; i < i1; ++i) {
            pd[i] *= a;
            if (pw) s += pw[i] * pd[i];
        }
        return s;
    });
}
double norm_inf(const std::vector<double>& a) {
    double m = 0.0;
    for (double v : a) m = std::max(m, std::fabs(v));
    return m;
}
double norm1(const std::vector<double>& a) {
    double s = 0.0;
    for (double v : a) s += std::fabs(v);
    return s;
}

// minimiser of the cubic through (a, fa, ga), (b, fb, gb); falls back to bisection
double cubic_min(double a, double fa, double ga, double b, double fb, double gb) {
    double d1 = ga + gb - 3.0 * (fa - fb) / (a - b);
    double disc = d1 * d1 - ga * gb;
    if (!(disc >= 0.0) || !std::isfinite(disc)) return 0.5 * (a + b);
    double d2 = std::sqrt(disc) * ((b > a) ? 1.0 : -1.0);
    double den = gb - ga + 2.0 * d2;
    if (den == 0.0 || !std::isfinite(den)) return 0.5 * (a + b);
    double t = b - (b - a) * (gb + d2 - d1) / den;
    return std::isfinite(t) ? t : 0.5 * (a + b);
}

struct Trial {
    double a = 0.0, f = 0.0, dg = 0.0;
    int eval_index = -1;
};

}  // namespace

int lbfgs_minimize(int n, double* x_io, const LbfgsEval& eval, int max_iter, double tol_grad,
                   int history, LbfgsResult* out, const LbfgsAccept& on_accept, double ftol_rel) {
    const double c1 = 1e-4, c2 = 0.9;
    const int max_ls = 40;
    std::vector<double> x(x_io, x_io + n), g(n), d(n), xt(n), gt(n), xb(n), gb(n);
    std::vector<std::vector<double>> S, Y;
    std::vector<double> rho;
    LbfgsResult res;
    double f = 0.0;
    int rc = eval(x.data(), &f, g.data());
    res.evals = 1;
    if (rc) {
        res.status = rc;
        if (out) *out = res;
        return rc;
    }
    if (on_accept) on_accept(0);
    res.f0 = f;
    res.status = 1;

    auto try_step = [&](double a, Trial* t) -> int {
        for (int i = 0; i < n; ++i) xt[i] = x[i] + a * d[i];
        double ft = 0.0;
        int r = eval(xt.data(), &ft, gt.data());
        t->eval_index = res.evals;
        ++res.evals;
        if (r) return r;
        t->a = a;
        t->f = ft;
        t->dg = dot(gt, d);
        return 0;
    };

    for (int it = 0; it < max_iter; ++it) {
        res.gnorm_inf = norm_inf(g);
        if (res.gnorm_inf <= tol_grad) {
            res.status = 0;
            break;
        }
        // ---- direction: two-loop recursion ----
        d = g;
        const int m = static_cast<int>(S.size());
        std::vector<double> alpha(m);
        if (m > 0) {
            // first loop: alpha_j = rho_j s_j.d, d -= alpha_j y_j; the update of d and the next dot product
            // share one pass over the vectors
            double sd = dot(S[m - 1], d);
            for (int j = m - 1; j >= 0; --j) {
                alpha[j] = rho[j] * sd;
                sd = axpy_dot(d, -alpha[j], Y[j], j > 0 ? &S[j - 1] : nullptr);
            }
            const double gamma = dot(S[m - 1], Y[m - 1]) / dot(Y[m - 1], Y[m - 1]);
            double yd = scale_dot(d, gamma, &Y[0]);
            for (int j = 0; j < m; ++j) {
                const double beta = rho[j] * yd;
                yd = axpy_dot(d, alpha[j] - beta, S[j], j + 1 < m ? &Y[j + 1] : nullptr);
            }
        }
        (void)scale_dot(d, -1.0, nullptr);
        double dg0 = dot(g, d);
        if (!(dg0 < 0.0)) {  // not a descent direction: restart from steepest descent
            S.clear();
            Y.clear();
            rho.clear();
            for (int i = 0; i < n; ++i) d[i] = -g[i];
            dg0 = -dot(g, g);
        }
        if (ftol_rel > 0.0 && !S.empty() && -dg0 <= ftol_rel * std::fabs(f)) {
            res.status = 2;  // predicted decrease below the resolution of the objective
            break;
        }
        // ---- strong-Wolfe line search (Nocedal & Wright Alg. 3.5 / 3.6) ----
        double a = (S.empty()) ? std::min(1.0, 1.0 / std::max(norm1(g), 1e-300)) : 1.0;
        Trial lo{0.0, f, dg0, -1}, hi{}, cur{};
        bool have_hi = false, accepted = false, have_best = false;
        Trial best{};
        Trial prev = lo;
        int ls = 0;
        auto remember = [&](const Trial& t) {  // keep the lowest sufficient-decrease point seen
            if (t.f <= f + c1 * t.a * dg0 && (!have_best || t.f < best.f)) {
                best = t;
                xb = xt;
                gb = gt;
                have_best = true;
            }
        };
        // bracketing phase
        for (; ls < max_ls && !accepted && !have_hi; ++ls) {
            rc = try_step(a, &cur);
            if (rc) break;
            if (!std::isfinite(cur.f)) {  // overshoot into nonsense: shrink
                a *= 0.25;
                continue;
            }
            remember(cur);
            if (cur.f > f + c1 * cur.a * dg0 || (ls > 0 && cur.f >= prev.f)) {
                lo = prev;
                hi = cur;
                have_hi = true;
            } else if (std::fabs(cur.dg) <= -c2 * dg0) {
                accepted = true;
            } else if (cur.dg >= 0.0) {
                lo = cur;
                hi = prev;
                have_hi = true;
            } else {
                prev = cur;
                a *= 2.0;
            }
        }
        // zoom phase
        for (; !rc && ls < max_ls && !accepted && have_hi; ++ls) {
            double w = hi.a - lo.a;
            double t = cubic_min(lo.a, lo.f, lo.dg, hi.a, hi.f, hi.dg);
            double lo_b = std::min(lo.a, hi.a) + 0.1 * std::fabs(w);
            double hi_b = std::max(lo.a, hi.a) - 0.1 * std::fabs(w);
            if (!(t >= lo_b && t <= hi_b)) t = 0.5 * (lo.a + hi.a);
            if (std::fabs(w) <= 1e-16 * std::max(1.0, std::fabs(lo.a))) break;
            rc = try_step(t, &cur);
            if (rc) break;
            remember(cur);
            if (cur.f > f + c1 * cur.a * dg0 || cur.f >= lo.f) {
                hi = cur;
            } else {
                if (std::fabs(cur.dg) <= -c2 * dg0) {
                    accepted = true;
                    break;
                }
                if (cur.dg * (hi.a - lo.a) >= 0.0) hi = lo;
                lo = cur;
            }
        }
        if (rc) {
            res.status = rc;
            break;
        }
        if (accepted) {
            best = cur;
            xb = xt;
            gb = gt;
            have_best = true;
        }
        if (!have_best || !(best.f < f)) {
            // no point with a decrease: at the resolution of the (fp32-evaluated) objective we are done
            res.status = 2;
            break;
        }
        // ---- update ----
        std::vector<double> s(n), yv(n);
        for (int i = 0; i < n; ++i) {
            s[i] = xb[i] - x[i];
            yv[i] = gb[i] - g[i];
        }
        double sy = dot(s, yv);
        x = xb;
        g = gb;
        f = best.f;
        ++res.iters;
        if (on_accept) on_accept(best.eval_index);
        if (sy > 1e-300 * std::max(1.0, dot(yv, yv))) {
            if (static_cast<int>(S.size()) == history) {
                S.erase(S.begin());
                Y.erase(Y.begin());
                rho.erase(rho.begin());
            }
            S.push_back(std::move(s));
            Y.push_back(std::move(yv));
            rho.push_back(1.0 / sy);
        }
    }
    res.gnorm_inf = norm_inf(g);
    if (res.status == 1 && res.gnorm_inf <= tol_grad) res.status = 0;
    res.f = f;
    std::copy(x.begin(), x.end(), x_io);
    if (out) *out = res;
    return res.status < 0 ? res.status : 0;
}

}  // namespace lipfit
