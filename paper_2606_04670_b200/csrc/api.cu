// api.cu -- the extern "C" boundary declared in include/lipfit.h: argument validation, workspace,
// and the order of device steps.  No arithmetic of the method lives here.
#include <cmath>
#include <cstring>
#include <vector>

#include "kernels.h"
#include "lbfgs.h"

using namespace lipfit;

namespace {

int check_sizes(int64_t N, int32_t d, int64_t Q) {
    if (d < 1 || d > LIPFIT_MAX_DIM) return LIPFIT_E_DIM;
    if (N < 1 || Q < 0 || N > 0x7fffffffLL || Q > 0x7fffffffLL) return LIPFIT_E_SIZE;
    return LIPFIT_OK;
}
int check_norm(int32_t norm) { return (norm >= 1 && norm <= 3) ? LIPFIT_OK : LIPFIT_E_PARAM; }
int check_M(float M) { return (M >= 0.f && std::isfinite(M)) ? LIPFIT_OK : LIPFIT_E_PARAM; }

// device copy of a host array (stream-ordered)
template <class T>
int to_device(Workspace& w, const T* host, size_t n, cudaStream_t s) {
    int rc = w.alloc(n * sizeof(T), s);
    if (rc) return rc;
    if (n) LIPFIT_CUDA(cudaMemcpyAsync(w.p, host, n * sizeof(T), cudaMemcpyHostToDevice, s));
    return LIPFIT_OK;
}

}  // namespace

#define LIPFIT_API __attribute__((visibility("default")))
extern "C" {

const char* lipfit_status_string(int code) {
    switch (code) {
        case LIPFIT_OK: return "ok";
        case LIPFIT_E_NULL: return "null pointer";
        case LIPFIT_E_DIM: return "bad dimension (need 1 <= d <= 32)";
        case LIPFIT_E_SIZE: return "bad size";
        case LIPFIT_E_PARAM: return "bad parameter";
        case LIPFIT_E_CUDA: return "CUDA error (no device or launch failure)";
        case LIPFIT_E_NOMEM: return "out of device memory";
        case LIPFIT_E_LIMIT: return "sizes beyond the fixed scratch of a no-allocation entry point";
        default: return "unknown status";
    }
}

const char* lipfit_version(void) { return "0.1.0"; }

int64_t lipfit_launch_count(void) { return g_launches.load(); }

void lipfit_set_timing(int32_t on) { timing_set(on); }

int lipfit_get_timing(int32_t which, double* total_ms, int64_t* launches) {
    long long n = 0;
    int rc = timing_get(which, total_ms, &n);
    if (launches) *launches = n;
    return rc;
}

int lipfit_bounds_variant(int32_t d, const int32_t* mono_mask, int32_t norm, char* out, int32_t cap) {
    if (!out || cap < 1) return LIPFIT_E_NULL;
    if (check_norm(norm)) return LIPFIT_E_PARAM;
    Xform xf;
    int rc = make_xform(d, mono_mask, nullptr, false, false, &xf);
    if (rc) return rc;
    std::strncpy(out, bounds_variant_name(bounds_xform(xf, norm), norm), static_cast<size_t>(cap) - 1);
    out[cap - 1] = '\0';
    return LIPFIT_OK;
}

int lipfit_release_workspace(void) { return workspace_release(); }

int lipfit_pipe_throughput(int32_t which, double* lane_results_per_clk_sm, double* warp_instr_per_clk_sm,
                           void* cuda_stream) {
    Ctx c;
    int rc = make_ctx(cuda_stream, &c);
    if (rc) return rc;
    return pipe_throughput(c, which, lane_results_per_clk_sm, warp_instr_per_clk_sm);
}
const char* lipfit_pipe_name(int32_t which) {
    static const char* const names[] = {"FFMA", "FADD", "FADD2 (add.f32x2)", "FFMA2 (fma.f32x2)", "FMNMX", "FMNMX3 (3-input min)",
                                        "MUFU.SQRT", "FFMA + FMNMX interleaved", "FADD2 + FMNMX3 interleaved",
                                        "FADD with |.| source modifier", "FADD2 + FMNMX interleaved",
                                        "FFMA + FMNMX3 interleaved", "2 FADD2 + 1 FMNMX3", "1 FADD2 + 2 FMNMX3",
                                        "FADD2 + FADD interleaved", "2 FFMA + 1 FMNMX3"};
    return (which >= 0 && which < 16) ? names[which] : "";
}

int lipfit_knn_variant(int32_t d, int32_t side, int32_t norm, int32_t flags, char* out, int32_t cap) {
    if (!out || cap < 1) return LIPFIT_E_NULL;
    if (check_norm(norm) || side < -1 || side > 1 || (flags & ~LIPFIT_KNN_NO_TENSOR_CORES)) return LIPFIT_E_PARAM;
    if (d < 1 || d > LIPFIT_MAX_DIM) return LIPFIT_E_DIM;
    Xform xf;
    std::vector<int32_t> mask(static_cast<size_t>(d), side == 0 ? 0 : 1);  // any constrained coordinate => one-sided
    int rc = make_xform(d, mask.data(), nullptr, side == 0, false, &xf);
    if (rc) return rc;
    std::strncpy(out, knn_variant_name(xf, norm, !(flags & LIPFIT_KNN_NO_TENSOR_CORES)), static_cast<size_t>(cap) - 1);
    out[cap - 1] = '\0';
    return LIPFIT_OK;
}

// lipfit_bounds_ex: Eq.(2),(3) with an explicit evaluation policy (include/lipfit.h).
int lipfit_bounds_ex(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q, float M,
                     const int32_t* mono_mask, int32_t norm, const float* weights, float* upper, float* lower,
                     float* g, int32_t policy, int64_t* pairs_evaluated, void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_bounds");
    int rc = check_sizes(N, d, Q);
    if (rc) return rc;
    if (check_norm(norm) || check_M(M)) return LIPFIT_E_PARAM;
    if (policy != LIPFIT_BOUNDS_AUTO && policy != LIPFIT_BOUNDS_BRUTE && policy != LIPFIT_BOUNDS_PRUNED)
        return LIPFIT_E_PARAM;
    Xform xf;
    rc = make_xform(d, mono_mask, weights, false, false, &xf);
    if (rc) return rc;
    if (!X || !y) return LIPFIT_E_NULL;
    if (Q == 0) {
        if (pairs_evaluated) pairs_evaluated[0] = pairs_evaluated[1] = pairs_evaluated[2] = 0;
        return LIPFIT_OK;
    }
    if (!Xq || (!upper && !lower && !g)) return LIPFIT_E_NULL;
    Ctx c;
    rc = make_ctx(cuda_stream, &c);
    if (rc) return rc;
    const bool pruned = policy == LIPFIT_BOUNDS_PRUNED || (policy == LIPFIT_BOUNDS_AUTO && bounds_prefers_pruned(xf, N, Q));
    if (policy == LIPFIT_BOUNDS_AUTO && bounds_small_applies(xf, N, Q)) {  // latency-bound call: one launch (small.cu)
        rc = launch_bounds_small(c, X, y, N, Xq, Q, xf, norm, M, upper, lower, g);
        if (rc) return rc;
        if (pairs_evaluated) {
            LIPFIT_CUDA(cudaStreamSynchronize(c.stream));
            pairs_evaluated[0] = N * Q;
            pairs_evaluated[1] = pairs_evaluated[2] = 0;
        }
        return LIPFIT_OK;
    }
    if (pruned) {
        Workspace stats;
        if (pairs_evaluated) {
            rc = stats.alloc(4 * sizeof(unsigned long long), c.stream);
            if (rc) return rc;
            LIPFIT_CUDA(cudaMemsetAsync(stats.p, 0, 4 * sizeof(unsigned long long), c.stream));
        }
        bool declined = false;  // AUTO: the finished query groups evaluated too many of their pairs for pruning to pay
        rc = launch_bounds_pruned(c, X, y, N, Xq, Q, xf, norm, M, upper, lower, g,
                                  pairs_evaluated ? stats.as<unsigned long long>() : nullptr,
                                  policy == LIPFIT_BOUNDS_AUTO ? kPrunedGuardLimit : 0.f, &declined);
        if (rc) return rc;
        if (!declined) {
            if (pairs_evaluated) {
                unsigned long long h[4] = {0, 0, 0, 0};
                LIPFIT_CUDA(cudaMemcpyAsync(h, stats.p, sizeof(h), cudaMemcpyDeviceToHost, c.stream));
                LIPFIT_CUDA(cudaStreamSynchronize(c.stream));
                pairs_evaluated[0] = static_cast<int64_t>(h[0]) * 1024;
                pairs_evaluated[1] = static_cast<int64_t>(h[1]);
                pairs_evaluated[2] = static_cast<int64_t>(h[2]);
            }
            return LIPFIT_OK;
        }
    }
    {
        const Xform xfb = bounds_xform(xf, norm);  // off-table shapes with d <= 8: even-rounded coordinate counts
        RecLayout lay = bounds_layout(c, xfb, norm, Q);
        if (lay.rf == 0) return LIPFIT_E_PARAM;
        const Xform xfp = lay.mscale ? scale_xform(xfb, M) : xfb;  // some kernel families fold M into the coordinates
        const float* centre = lay.mscale ? X : nullptr;          // ... and those are translated to the first datum
        Workspace rec;
        rc = rec.alloc(sizeof(float) * static_cast<size_t>(N) * lay.rf, c.stream);
        if (rc) return rc;
        rc = launch_prepack(c, X, y, nullptr, N, xfp, lay, rec.as<float>(), centre);
        if (rc) return rc;
        rc = launch_bounds(c, rec.as<float>(), N, Xq, Q, xfp, norm, M, upper, lower, g, centre);
        if (rc) return rc;
        if (pairs_evaluated) {
            LIPFIT_CUDA(cudaStreamSynchronize(c.stream));
            pairs_evaluated[0] = N * Q;
            pairs_evaluated[1] = pairs_evaluated[2] = 0;
        }
        return LIPFIT_OK;
    }
}

int lipfit_bounds(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                  float M, const int32_t* mono_mask, int32_t norm, const float* weights, float* upper,
                  float* lower, float* g, void* cuda_stream) {
    return lipfit_bounds_ex(X, y, N, d, Xq, Q, M, mono_mask, norm, weights, upper, lower, g, LIPFIT_BOUNDS_AUTO,
                            nullptr, cuda_stream);
}

int lipfit_bounds_pruned(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                         float M, const int32_t* mono_mask, int32_t norm, const float* weights, float* upper,
                         float* lower, float* g, int64_t* pairs_evaluated, void* cuda_stream) {
    return lipfit_bounds_ex(X, y, N, d, Xq, Q, M, mono_mask, norm, weights, upper, lower, g, LIPFIT_BOUNDS_PRUNED,
                            pairs_evaluated, cuda_stream);
}

int lipfit_bounds_noalloc(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                          float M, const int32_t* mono_mask, int32_t norm, const float* weights, float* upper,
                          float* lower, float* g, void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_bounds_noalloc");
    int rc = check_sizes(N, d, Q);
    if (rc) return rc;
    if (check_norm(norm) || check_M(M)) return LIPFIT_E_PARAM;
    Xform xf;
    rc = make_xform(d, mono_mask, weights, false, false, &xf);
    if (rc) return rc;
    if (!X || !y) return LIPFIT_E_NULL;
    if (Q == 0) return LIPFIT_OK;
    if (!Xq || (!upper && !lower && !g)) return LIPFIT_E_NULL;
    Ctx c;
    rc = make_ctx(cuda_stream, &c);
    if (rc) return rc;
    return launch_bounds_noalloc(c, X, y, N, Xq, Q, xf, norm, M, upper, lower, g);
}

int lipfit_bounds_region(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                         float M, const int32_t* mon, const float* a, const float* b, int32_t norm,
                         const float* weights, float* upper, float* lower, float* g, void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_bounds_region");
    int rc = check_sizes(N, d, Q);
    if (rc) return rc;
    if (check_norm(norm) || check_M(M)) return LIPFIT_E_PARAM;
    for (int i = 0; i < d; ++i) {
        const int m = mon ? mon[i] : 0;
        if (m < 0 || m > 4) return LIPFIT_E_PARAM;
        if (m != 0) {
            if (!a || !b) return LIPFIT_E_NULL;
            if (!(a[i] <= b[i]) || a[i] == INFINITY || b[i] == -INFINITY) return LIPFIT_E_PARAM;  // also NaN
        }
        if (weights && !(weights[i] >= 0.f && std::isfinite(weights[i]))) return LIPFIT_E_PARAM;
    }
    if (!X || !y) return LIPFIT_E_NULL;
    if (Q == 0) return LIPFIT_OK;
    if (!Xq || (!upper && !lower && !g)) return LIPFIT_E_NULL;
    Ctx c;
    rc = make_ctx(cuda_stream, &c);
    if (rc) return rc;
    return launch_bounds_region(c, X, y, N, d, Xq, Q, M, mon, a, b, norm, weights, upper, lower, g);
}

int lipfit_bounds_topk(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                       float M, const int32_t* mono_mask, int32_t norm, const float* weights, int32_t k,
                       const float* wk, float* upper, float* lower, float* g, void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_bounds_topk");
    int rc = check_sizes(N, d, Q);
    if (rc) return rc;
    if (k < 1 || k > LIPFIT_MAX_TOPK || k > N) return LIPFIT_E_SIZE;
    if (check_norm(norm) || check_M(M)) return LIPFIT_E_PARAM;
    if (!wk) return LIPFIT_E_NULL;
    for (int j = 0; j < k; ++j)
        if (!(wk[j] >= 0.f) || !std::isfinite(wk[j])) return LIPFIT_E_PARAM;
    Xform xf;
    rc = make_xform(d, mono_mask, weights, false, false, &xf);
    if (rc) return rc;
    if (!X || !y) return LIPFIT_E_NULL;
    if (Q == 0) return LIPFIT_OK;
    if (!Xq || (!upper && !lower && !g)) return LIPFIT_E_NULL;
    Ctx c;
    rc = make_ctx(cuda_stream, &c);
    if (rc) return rc;
    RecLayout lay = bounds_topk_layout(c, xf, norm, Q);
    if (lay.rf == 0) return LIPFIT_E_PARAM;
    const Xform xfp = lay.mscale ? scale_xform(xf, M) : xf;  // as lipfit_bounds_ex
    const float* centre = lay.mscale ? X : nullptr;
    Workspace rec;
    rc = rec.alloc(sizeof(float) * static_cast<size_t>(N) * lay.rf, c.stream);
    if (rc) return rc;
    rc = launch_prepack(c, X, y, nullptr, N, xfp, lay, rec.as<float>(), centre);
    if (rc) return rc;
    return launch_bounds_topk(c, rec.as<float>(), N, Xq, Q, xfp, norm, M, k, wk, upper, lower, g, centre, lay.dup);
}

int lipfit_bounds_host_ex(const float* X, const float* y, int64_t N, int32_t d, const float* Xq,
                          int64_t Q, float M, const int32_t* mono_mask, int32_t norm,
                          const float* weights, float* upper, float* lower, float* g, int32_t policy,
                          int64_t* pairs_evaluated, void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_bounds_host");
    int rc = check_sizes(N, d, Q);
    if (rc) return rc;
    if (check_norm(norm) || check_M(M)) return LIPFIT_E_PARAM;
    if (policy != LIPFIT_BOUNDS_AUTO && policy != LIPFIT_BOUNDS_BRUTE && policy != LIPFIT_BOUNDS_PRUNED)
        return LIPFIT_E_PARAM;
    Xform xf;
    if ((rc = make_xform(d, mono_mask, weights, false, false, &xf))) return rc;
    if (!X || !y || (Q > 0 && !Xq)) return LIPFIT_E_NULL;
    if (Q == 0) {
        if (pairs_evaluated) pairs_evaluated[0] = pairs_evaluated[1] = pairs_evaluated[2] = 0;
        return LIPFIT_OK;
    }
    cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);
    Workspace dX, dy, dXq, dout;
    if ((rc = to_device(dX, X, static_cast<size_t>(N) * d, s))) return rc;
    if ((rc = to_device(dy, y, static_cast<size_t>(N), s))) return rc;
    if ((rc = to_device(dXq, Xq, static_cast<size_t>(Q) * d, s))) return rc;
    if ((rc = dout.alloc(sizeof(float) * 3 * static_cast<size_t>(Q), s))) return rc;
    float* du = upper ? dout.as<float>() : nullptr;
    float* dl = lower ? dout.as<float>() + Q : nullptr;
    float* dg = g ? dout.as<float>() + 2 * Q : nullptr;
    rc = lipfit_bounds_ex(dX.as<float>(), dy.as<float>(), N, d, dXq.as<float>(), Q, M, mono_mask, norm,
                          weights, du, dl, dg, policy, pairs_evaluated, cuda_stream);
    if (rc) return rc;
    const size_t ob = sizeof(float) * static_cast<size_t>(Q);
    if (upper && Q) LIPFIT_CUDA(cudaMemcpyAsync(upper, du, ob, cudaMemcpyDeviceToHost, s));
    if (lower && Q) LIPFIT_CUDA(cudaMemcpyAsync(lower, dl, ob, cudaMemcpyDeviceToHost, s));
    if (g && Q) LIPFIT_CUDA(cudaMemcpyAsync(g, dg, ob, cudaMemcpyDeviceToHost, s));
    LIPFIT_CUDA(cudaStreamSynchronize(s));
    return LIPFIT_OK;
}

int lipfit_bounds_host(const float* X, const float* y, int64_t N, int32_t d, const float* Xq,
                       int64_t Q, float M, const int32_t* mono_mask, int32_t norm,
                       const float* weights, float* upper, float* lower, float* g,
                       void* cuda_stream) {
    return lipfit_bounds_host_ex(X, y, N, d, Xq, Q, M, mono_mask, norm, weights, upper, lower, g,
                                 LIPFIT_BOUNDS_AUTO, nullptr, cuda_stream);
}

int lipfit_knn(const float* X, int64_t N, int32_t d, const float* Xq, int64_t Q,
               const int32_t* mono_mask, int32_t side, int32_t norm, const float* weights, int32_t k,
               int32_t* idx, float* dist, void* cuda_stream) {
    return lipfit_knn_ex(X, N, d, Xq, Q, mono_mask, side, norm, weights, k, idx, dist, 0, nullptr, cuda_stream);
}

int lipfit_knn_ex(const float* X, int64_t N, int32_t d, const float* Xq, int64_t Q,
                  const int32_t* mono_mask, int32_t side, int32_t norm, const float* weights, int32_t k,
                  int32_t* idx, float* dist, int32_t flags, lipfit_knn_info* info, void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_knn_ex");
    int rc = check_sizes(N, d, Q);
    if (rc) return rc;
    if (k < 1 || k > N || k > LIPFIT_MAX_K) return LIPFIT_E_SIZE;
    if (check_norm(norm) || side < -1 || side > 1 || (flags & ~LIPFIT_KNN_NO_TENSOR_CORES)) return LIPFIT_E_PARAM;
    if (info) *info = lipfit_knn_info{0, 0.0, 0, 0};
    Xform xf;
    rc = make_xform(d, mono_mask, weights, side == 0, side < 0, &xf);
    if (rc) return rc;
    if (!X) return LIPFIT_E_NULL;
    if (Q == 0) return LIPFIT_OK;
    if (!Xq || !idx || !dist) return LIPFIT_E_NULL;
    Ctx c;
    rc = make_ctx(cuda_stream, &c);
    if (rc) return rc;
    return launch_knn(c, X, N, Xq, Q, xf, norm, k, idx, dist, !(flags & LIPFIT_KNN_NO_TENSOR_CORES), info);
}

int lipfit_knn_host(const float* X, int64_t N, int32_t d, const float* Xq, int64_t Q,
                    const int32_t* mono_mask, int32_t side, int32_t norm, const float* weights,
                    int32_t k, int32_t* idx, float* dist, void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_knn_host");
    int rc = check_sizes(N, d, Q);
    if (rc) return rc;
    if (k < 1 || k > N || k > LIPFIT_MAX_K) return LIPFIT_E_SIZE;
    if (check_norm(norm) || side < -1 || side > 1) return LIPFIT_E_PARAM;
    Xform xf;
    if ((rc = make_xform(d, mono_mask, weights, side == 0, side < 0, &xf))) return rc;
    if (!X || (Q > 0 && (!Xq || !idx || !dist))) return LIPFIT_E_NULL;
    if (Q == 0) return LIPFIT_OK;
    cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);
    Workspace dX, dXq, di, dd;
    if ((rc = to_device(dX, X, static_cast<size_t>(N) * d, s))) return rc;
    if ((rc = to_device(dXq, Xq, static_cast<size_t>(Q) * d, s))) return rc;
    const size_t n = static_cast<size_t>(Q) * k;
    if ((rc = di.alloc(n * sizeof(int32_t), s))) return rc;
    if ((rc = dd.alloc(n * sizeof(float), s))) return rc;
    rc = lipfit_knn(dX.as<float>(), N, d, dXq.as<float>(), Q, mono_mask, side, norm, weights, k,
                    di.as<int32_t>(), dd.as<float>(), cuda_stream);
    if (rc) return rc;
    if (n) {
        LIPFIT_CUDA(cudaMemcpyAsync(idx, di.p, n * sizeof(int32_t), cudaMemcpyDeviceToHost, s));
        LIPFIT_CUDA(cudaMemcpyAsync(dist, dd.p, n * sizeof(float), cudaMemcpyDeviceToHost, s));
    }
    LIPFIT_CUDA(cudaStreamSynchronize(s));
    return LIPFIT_OK;
}

// ---- local Lipschitz interpolation ----
int lipfit_distance_quantiles(const float* X, int64_t N, int32_t d, int32_t norm, const float* weights,
                              const int32_t* pair_i, const int32_t* pair_k, int64_t S, int32_t J, float* knots,
                              void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_distance_quantiles");
    int rc = check_sizes(N, d, 0);
    if (rc) return rc;
    if (check_norm(norm)) return LIPFIT_E_PARAM;
    if (S < 1 || S > 0x7fffffffLL || J < 1 || J > 1024 || J > S) return LIPFIT_E_SIZE;
    Xform xf;
    if ((rc = make_xform(d, nullptr, weights, true, false, &xf))) return rc;
    if (!X || !pair_i || !pair_k || !knots) return LIPFIT_E_NULL;
    Ctx c;
    if ((rc = make_ctx(cuda_stream, &c))) return rc;
    Workspace wk;
    if ((rc = wk.alloc(sizeof(float) * 1024 + sizeof(int), c.stream))) return rc;
    int* bad = reinterpret_cast<int*>(wk.as<float>() + 1024);
    LIPFIT_CUDA(cudaMemsetAsync(bad, 0, sizeof(int), c.stream));
    if ((rc = launch_distance_quantiles(c, X, N, xf, norm, pair_i, pair_k, S, J, wk.as<float>(), bad))) return rc;
    int bad_h = 0;
    LIPFIT_CUDA(cudaMemcpyAsync(knots, wk.p, sizeof(float) * J, cudaMemcpyDeviceToHost, c.stream));
    LIPFIT_CUDA(cudaMemcpyAsync(&bad_h, bad, sizeof(int), cudaMemcpyDeviceToHost, c.stream));
    LIPFIT_CUDA(cudaStreamSynchronize(c.stream));
    return bad_h ? LIPFIT_E_SIZE : LIPFIT_OK;  // an index pair outside [0, N)
}

static int check_knots(const float* knots, int32_t J) {
    if (!knots) return LIPFIT_E_NULL;
    if (J != LIPFIT_LOCAL_KNOTS) return LIPFIT_E_SIZE;
    for (int j = 0; j < J; ++j) {
        if (!(knots[j] >= 0.f) || (j > 0 && knots[j] < knots[j - 1])) return LIPFIT_E_PARAM;  // also rejects NaN
    }
    return LIPFIT_OK;
}

int lipfit_local_lipschitz(const float* X, const float* y, int64_t N, int32_t d, int32_t norm,
                           const float* weights, const float* knots, int32_t J, float* table,
                           void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_local_lipschitz");
    int rc = check_sizes(N, d, 0);
    if (rc) return rc;
    if (check_norm(norm)) return LIPFIT_E_PARAM;
    if ((rc = check_knots(knots, J))) return rc;
    Xform xf;
    if ((rc = make_xform(d, nullptr, weights, true, false, &xf))) return rc;
    if (!X || !y || !table) return LIPFIT_E_NULL;
    if (N * static_cast<int64_t>(J) > 0x7fffffffLL) return LIPFIT_E_SIZE;
    Ctx c;
    if ((rc = make_ctx(cuda_stream, &c))) return rc;
    return launch_local_lipschitz(c, X, y, N, xf, norm, knots, table);
}

int lipfit_values_local(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                        int32_t norm, const float* weights, const float* knots, int32_t J, const float* table,
                        float* upper, float* lower, float* g, void* cuda_stream) {
    NvtxRange nvtx_range("lipfit_values_local");
    int rc = check_sizes(N, d, Q);
    if (rc) return rc;
    if (check_norm(norm)) return LIPFIT_E_PARAM;
    if ((rc = check_knots(knots, J))) return rc;
    Xform xf;
    if ((rc = make_xform(d, nullptr, weights, true, false, &xf))) return rc;
    if (!X || !y || !table) return LIPFIT_E_NULL;
    if (Q == 0) return LIPFIT_OK;
    if (!Xq || (!upper && !lower && !g)) return LIPFIT_E_NULL;
    Ctx c;
    if ((rc = make_ctx(cuda_stream, &c))) return rc;
    return launch_values_local(c, X, y, N, Xq, Q, xf, norm, knots, table, upper, lower, g);
}

}  // extern "C"
