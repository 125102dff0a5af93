// api_smooth.cu -- extern "C" entry points of the smoothing path (Eq.(5)-(7) PAPER.md:189-200):
// lipfit_smooth_objective, lipfit_smooth (host LBFGS loop around the device pass), lipfit_lbfgs.
#include <cmath>
#include <vector>

#include <cstring>

#include "kernels.h"
#include "lbfgs.h"

using namespace lipfit;

namespace {

int check_common(const float* X, const float* y, int64_t N, int32_t d, float M, int32_t norm,
                 float p) {
    if (d < 1 || d > LIPFIT_MAX_DIM) return LIPFIT_E_DIM;
    if (N < 1 || N > 0x7fffffffLL) return LIPFIT_E_SIZE;
    if (norm < 1 || norm > 3 || !(M >= 0.f) || !std::isfinite(M) || !(p > 0.f) || !std::isfinite(p))
        return LIPFIT_E_PARAM;
    if (!X || !y) return LIPFIT_E_NULL;
    return LIPFIT_OK;
}

struct Pinned {
    void* p = nullptr;
    int alloc(size_t bytes) {
        cudaError_t e = cudaMallocHost(&p, bytes ? bytes : 16);
        if (e != cudaSuccess) {
            (void)cudaGetLastError();
            p = nullptr;
            return LIPFIT_E_NOMEM;
        }
        return LIPFIT_OK;
    }
    ~Pinned() {
        if (p) cudaFreeHost(p);
    }
    template <class T>
    T* as() const { return reinterpret_cast<T*>(p); }
};

}  // namespace

#define LIPFIT_API __attribute__((visibility("default")))
extern "C" {

int lipfit_smooth_objective(const float* X, const float* y, int64_t N, int32_t d, float M,
                            const int32_t* mono_mask, int32_t norm, const float* weights, float p,
                            const float* eps, double* F, float* grad, void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_smooth_objective");
    int rc = check_common(X, y, N, d, M, norm, p);
    if (rc) return rc;
    Xform xf;
    rc = make_xform(d, mono_mask, weights, false, false, &xf);
    if (rc) return rc;
    if (!F && !grad) return LIPFIT_E_NULL;
    Ctx c;
    rc = make_ctx(cuda_stream, &c);
    if (rc) return rc;
    RecLayout lay = smooth_layout(xf, norm);
    Workspace rec, fdev;
    rc = rec.alloc(sizeof(float) * static_cast<size_t>(N) * lay.rf, c.stream);
    if (rc) return rc;
    rc = fdev.alloc(sizeof(double) * 2, c.stream);
    if (rc) return rc;
    rc = launch_prepack(c, X, nullptr, nullptr, N, scale_xform(xf, M), lay, rec.as<float>(), X /* centre */);
    if (rc) return rc;
    rc = launch_smooth_objective(c, rec.as<float>(), y, eps, N, xf, norm, p,
                                 F ? fdev.as<double>() : nullptr, grad, nullptr);
    if (rc) return rc;
    if (F) {
        LIPFIT_CUDA(cudaMemcpyAsync(F, fdev.p, sizeof(double), cudaMemcpyDeviceToHost, c.stream));
        LIPFIT_CUDA(cudaStreamSynchronize(c.stream));
    }
    return LIPFIT_OK;
}

int lipfit_smooth_objective_pruned(const float* X, const float* y, int64_t N, int32_t d, float M,
                                   const int32_t* mono_mask, int32_t norm, const float* weights, float p,
                                   const float* eps, double* F, float* grad, int64_t* pairs_evaluated,
                                   void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_smooth_objective_pruned");
    int rc = check_common(X, y, N, d, M, norm, p);
    if (rc) return rc;
    Xform xf;
    rc = make_xform(d, mono_mask, weights, false, false, &xf);
    if (rc) return rc;
    if (!F) return LIPFIT_E_NULL;
    Ctx c;
    rc = make_ctx(cuda_stream, &c);
    if (rc) return rc;
    Workspace fdev;
    rc = fdev.alloc(sizeof(double) + 2 * sizeof(unsigned long long), c.stream);
    if (rc) return rc;
    LIPFIT_CUDA(cudaMemsetAsync(fdev.p, 0, sizeof(double) + 2 * sizeof(unsigned long long), c.stream));  // stats
    unsigned long long* stats = reinterpret_cast<unsigned long long*>(fdev.as<double>() + 1);
    rc = launch_smooth_objective_pruned(c, X, y, eps, N, xf, norm, M, p, fdev.as<double>(), grad,
                                        pairs_evaluated ? stats : nullptr);
    if (rc) return rc;
    unsigned long long h[3] = {0, 0, 0};
    LIPFIT_CUDA(cudaMemcpyAsync(h, fdev.p, sizeof(h), cudaMemcpyDeviceToHost, c.stream));
    LIPFIT_CUDA(cudaStreamSynchronize(c.stream));
    std::memcpy(F, &h[0], sizeof(double));
    if (pairs_evaluated) *pairs_evaluated = static_cast<int64_t>(h[1]) * 1024;
    return LIPFIT_OK;
}

int lipfit_smooth(const float* X, float* y_inout, int64_t N, int32_t d, float M,
                  const int32_t* mono_mask, int32_t norm, const float* weights, float p,
                  int32_t max_iter, double tol_grad, float* eps_out, lipfit_smooth_info* info,
                  void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_smooth");
    int rc = check_common(X, y_inout, N, d, M, norm, p);
    if (rc) return rc;
    if (max_iter < 0 || !(tol_grad >= 0.0)) return LIPFIT_E_PARAM;
    Xform xf;
    rc = make_xform(d, mono_mask, weights, false, false, &xf);
    if (rc) return rc;
    Ctx c;
    rc = make_ctx(cuda_stream, &c);
    if (rc) return rc;
    const size_t n = static_cast<size_t>(N);
    RecLayout lay = smooth_layout(xf, norm);
    Workspace rec, eps_d, grad_d, fv_d;
    if ((rc = rec.alloc(sizeof(float) * n * lay.rf, c.stream))) return rc;
    if ((rc = eps_d.alloc(sizeof(float) * n, c.stream))) return rc;
    if ((rc = grad_d.alloc(sizeof(float) * n, c.stream))) return rc;
    if ((rc = fv_d.alloc(sizeof(double) * 2, c.stream))) return rc;
    Pinned eps_h, grad_h, fv_h;
    if ((rc = eps_h.alloc(sizeof(float) * n))) return rc;
    if ((rc = grad_h.alloc(sizeof(float) * n))) return rc;
    if ((rc = fv_h.alloc(sizeof(double) * 2))) return rc;
    const bool use_pruned = smooth_prefers_pruned(xf, N);
    Workspace order;  // pruned pass: the Morton order of the data, computed once (X does not change)
    if (use_pruned) {
        if ((rc = smooth_pruned_order(c, X, N, xf, order))) return rc;
    } else {
        rc = launch_prepack(c, X, nullptr, nullptr, N, scale_xform(xf, M), lay, rec.as<float>(), X /* centre */);
        if (rc) return rc;
    }

    std::vector<double> viol;  // max violation seen by each evaluation
    auto eval = [&](const double* x, double* f, double* g) -> int {
        float* eh = eps_h.as<float>();
        for (size_t i = 0; i < n; ++i) eh[i] = static_cast<float>(x[i]);
        LIPFIT_CUDA(cudaMemcpyAsync(eps_d.p, eh, sizeof(float) * n, cudaMemcpyHostToDevice, c.stream));
        int r = use_pruned
                    ? launch_smooth_objective_pruned(c, X, y_inout, eps_d.as<float>(), N, xf, norm, M, p,
                                                     fv_d.as<double>(), grad_d.as<float>(), nullptr,
                                                     fv_d.as<double>() + 1, order.as<int32_t>())
                    : launch_smooth_objective(c, rec.as<float>(), y_inout, eps_d.as<float>(), N, xf, norm, p,
                                              fv_d.as<double>(), grad_d.as<float>(), fv_d.as<double>() + 1);
        if (r) return r;
        LIPFIT_CUDA(cudaMemcpyAsync(grad_h.p, grad_d.p, sizeof(float) * n, cudaMemcpyDeviceToHost,
                                    c.stream));
        LIPFIT_CUDA(cudaMemcpyAsync(fv_h.p, fv_d.p, sizeof(double) * 2, cudaMemcpyDeviceToHost,
                                    c.stream));
        LIPFIT_CUDA(cudaStreamSynchronize(c.stream));
        // F and grad are those of the fp32-rounded point eps = (float)x.
        const float* gh = grad_h.as<float>();
        for (size_t i = 0; i < n; ++i) g[i] = static_cast<double>(gh[i]);
        *f = fv_h.as<double>()[0];
        viol.push_back(fv_h.as<double>()[1]);
        return LIPFIT_OK;
    };

    std::vector<double> x(n, 0.0);
    LbfgsResult res;
    int accepted_eval = 0;
    // DESIGN.md R14: the device pass resolves F to ~1e-9 relative (fp32 pair arithmetic, fp64 sums); once the
    // model predicts less than that, further line searches only burn evaluations (config 5: 207 -> 47)
    const double ftol = 1e-9;
    rc = lbfgs_minimize(static_cast<int>(N), x.data(), eval, max_iter, tol_grad, 20, &res,
                        [&](int e) { accepted_eval = e; }, ftol);
    if (rc) return rc < 0 ? rc : LIPFIT_E_CUDA;

    // y <- y + eps, eps_out <- eps
    float* eh = eps_h.as<float>();
    for (size_t i = 0; i < n; ++i) eh[i] = static_cast<float>(x[i]);
    LIPFIT_CUDA(cudaMemcpyAsync(eps_d.p, eh, sizeof(float) * n, cudaMemcpyHostToDevice, c.stream));
    rc = launch_axpy(c, y_inout, eps_d.as<float>(), N);
    if (rc) return rc;
    if (eps_out)
        LIPFIT_CUDA(cudaMemcpyAsync(eps_out, eps_d.p, sizeof(float) * n, cudaMemcpyDeviceToDevice,
                                    c.stream));
    LIPFIT_CUDA(cudaStreamSynchronize(c.stream));
    if (info) {
        info->iters = res.iters;
        info->evals = res.evals;
        info->status = res.status;
        info->reserved = 0;
        info->F0 = res.f0;
        info->F = res.f;
        info->gnorm_inf = res.gnorm_inf;
        info->max_violation0 = viol.empty() ? 0.0 : viol[0];
        info->max_violation =
            (accepted_eval >= 0 && accepted_eval < static_cast<int>(viol.size())) ? viol[accepted_eval]
                                                                                  : 0.0;
    }
    return LIPFIT_OK;
}

int lipfit_smooth_host(const float* X, float* y_inout, int64_t N, int32_t d, float M,
                       const int32_t* mono_mask, int32_t norm, const float* weights, float p,
                       int32_t max_iter, double tol_grad, float* eps_out, lipfit_smooth_info* info,
                       void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_smooth_host");
    int rc = check_common(X, y_inout, N, d, M, norm, p);
    if (rc) return rc;
    if (max_iter < 0 || !(tol_grad >= 0.0)) return LIPFIT_E_PARAM;
    Xform xf;
    if ((rc = make_xform(d, mono_mask, weights, false, false, &xf))) return rc;
    cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);
    const size_t n = static_cast<size_t>(N);
    Workspace dX, dy, de;
    if ((rc = dX.alloc(sizeof(float) * n * d, s))) return rc;
    if ((rc = dy.alloc(sizeof(float) * n, s))) return rc;
    if ((rc = de.alloc(sizeof(float) * n, s))) return rc;
    LIPFIT_CUDA(cudaMemcpyAsync(dX.p, X, sizeof(float) * n * d, cudaMemcpyHostToDevice, s));
    LIPFIT_CUDA(cudaMemcpyAsync(dy.p, y_inout, sizeof(float) * n, cudaMemcpyHostToDevice, s));
    rc = lipfit_smooth(dX.as<float>(), dy.as<float>(), N, d, M, mono_mask, norm, weights, p, max_iter,
                       tol_grad, de.as<float>(), info, cuda_stream);
    if (rc) return rc;
    LIPFIT_CUDA(cudaMemcpyAsync(y_inout, dy.p, sizeof(float) * n, cudaMemcpyDeviceToHost, s));
    if (eps_out) LIPFIT_CUDA(cudaMemcpyAsync(eps_out, de.p, sizeof(float) * n, cudaMemcpyDeviceToHost, s));
    LIPFIT_CUDA(cudaStreamSynchronize(s));
    return LIPFIT_OK;
}

int lipfit_lipschitz_constant(const float* X, const float* y, int64_t N, int32_t d,
                              const int32_t* mono_mask, int32_t norm, const float* weights, float* L,
                              void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_lipschitz_constant");
    int rc = check_common(X, y, N, d, 0.f, norm, 1.f);
    if (rc) return rc;
    if (!L) return LIPFIT_E_NULL;
    Xform xf;
    rc = make_xform(d, mono_mask, weights, false, false, &xf);
    if (rc) return rc;
    Ctx c;
    rc = make_ctx(cuda_stream, &c);
    if (rc) return rc;
    RecLayout lay = lipconst_layout(xf, norm);
    Workspace rec;
    rc = rec.alloc(sizeof(float) * static_cast<size_t>(N) * lay.rf, c.stream);
    if (rc) return rc;
    rc = launch_prepack(c, X, nullptr, nullptr, N, xf, lay, rec.as<float>());
    if (rc) return rc;
    return launch_lipschitz_constant(c, X, rec.as<float>(), y, N, xf, norm, L);
}

int lipfit_lipschitz_constant_host(const float* X, const float* y, int64_t N, int32_t d,
                                   const int32_t* mono_mask, int32_t norm, const float* weights,
                                   float* L, void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_lipschitz_constant_host");
    int rc = check_common(X, y, N, d, 0.f, norm, 1.f);
    if (rc) return rc;
    if (!L) return LIPFIT_E_NULL;
    Xform xf;
    if ((rc = make_xform(d, mono_mask, weights, false, false, &xf))) return rc;
    cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);
    const size_t n = static_cast<size_t>(N);
    Workspace dX, dy, dL;
    if ((rc = dX.alloc(sizeof(float) * n * d, s))) return rc;
    if ((rc = dy.alloc(sizeof(float) * n, s))) return rc;
    if ((rc = dL.alloc(sizeof(float), s))) return rc;
    LIPFIT_CUDA(cudaMemcpyAsync(dX.p, X, sizeof(float) * n * d, cudaMemcpyHostToDevice, s));
    LIPFIT_CUDA(cudaMemcpyAsync(dy.p, y, sizeof(float) * n, cudaMemcpyHostToDevice, s));
    rc = lipfit_lipschitz_constant(dX.as<float>(), dy.as<float>(), N, d, mono_mask, norm, weights,
                                   dL.as<float>(), cuda_stream);
    if (rc) return rc;
    LIPFIT_CUDA(cudaMemcpyAsync(L, dL.p, sizeof(float), cudaMemcpyDeviceToHost, s));
    LIPFIT_CUDA(cudaStreamSynchronize(s));
    return LIPFIT_OK;
}

int lipfit_lbfgs(int64_t n, double* x, lipfit_eval_fn fn, void* user, int32_t max_iter,
                 double tol_grad, int32_t history, lipfit_smooth_info* info) {
    NvtxRange nvtx_range("lipfit_lbfgs");
    if (!x || !fn) return LIPFIT_E_NULL;
    if (n < 1 || n > 0x7fffffffLL || max_iter < 0 || history < 1 || !(tol_grad >= 0.0))
        return LIPFIT_E_SIZE;
    LbfgsResult res;
    int rc = lbfgs_minimize(
        static_cast<int>(n), x,
        [&](const double* xx, double* f, double* g) {
            int r = fn(user, xx, f, g);
            return r > 0 ? -r : r;
        },
        max_iter, tol_grad, history, &res);
    if (info) {
        info->iters = res.iters;
        info->evals = res.evals;
        info->status = res.status;
        info->reserved = 0;
        info->F0 = res.f0;
        info->F = res.f;
        info->gnorm_inf = res.gnorm_inf;
        info->max_violation0 = info->max_violation = 0.0;
    }
    return rc;
}

}  // extern "C"
