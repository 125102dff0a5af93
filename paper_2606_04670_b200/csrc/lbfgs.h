// lbfgs.h -- step a5: host-side limited-memory BFGS with a strong-Wolfe line
// search.  PAPER.md:200 ("an unconstrained minimisation method like LBFGS") and PAPER.md:212
// (torch.optim.LBFGS) fix only the method's name; the hyper-parameters are reading R14:
// history 20, c1 = 1e-4, c2 = 0.9, gamma = s'y / y'y initial scaling, first trial step
// min(1, 1/||g||_1), stop at ||g||_inf <= tol_grad, at max_iter, or when no further progress is
// possible.  Eq.(7) is strongly convex, so the minimiser does not depend on these choices.
#pragma once
#include <functional>

namespace lipfit {

struct LbfgsResult {
    int iters = 0;
    int evals = 0;
    int status = 0;  // 0 converged, 1 max_iter, 2 no further progress, <0 evaluation error code
    double f0 = 0.0, f = 0.0, gnorm_inf = 0.0;
};

// eval(x, &f, g) returns 0 on success, else an error code that aborts the minimisation.
using LbfgsEval = std::function<int(const double* x, double* f, double* g)>;
// called with the index of the evaluation that produced the accepted iterate
using LbfgsAccept = std::function<void(int eval_index)>;

// ftol_rel > 0: also stop (status 2) when the decrease the quasi-Newton model predicts for the unit step,
// -g'd, is <= ftol_rel * |f|: the iterate sits at the resolution of an objective that is evaluated with
// rounding noise (lipfit_smooth: fp32 pair arithmetic), where a line search can only burn evaluations.
int lbfgs_minimize(int n, double* x, const LbfgsEval& eval, int max_iter, double tol_grad,
                   int history, LbfgsResult* out, const LbfgsAccept& on_accept = nullptr,
                   double ftol_rel = 0.0);

}  // namespace lipfit
