// prepack.cu -- step a1: build the packed data records once per call so that
// the mask, the weights and the coordinate order never reach the hot loops
// ("a suitable modification to distance calculation, which avoids branching").
// Pure streaming kernels (HBM-bound, microseconds).
#include <cmath>
#include <map>
#include <mutex>

#include "kernels.h"

namespace lipfit {

std::atomic<int64_t> g_launches{0};

std::atomic<int> g_timing_on{0};
static std::mutex g_timing_mu;
static double g_timing_ms[TK_COUNT] = {};
static long long g_timing_n[TK_COUNT] = {};

KernelTimer::KernelTimer(int which_, cudaStream_t s_) : which(which_), s(s_) {
    if (!g_timing_on.load()) return;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        (void)cudaGetLastError();
        return;
    }
    on = true;
    cudaEventRecord(e0, s);
}
void KernelTimer::stop() {
    if (!on) return;
    cudaEventRecord(e1, s);
    if (cudaEventSynchronize(e1) == cudaSuccess) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess) {
            std::lock_guard<std::mutex> lk(g_timing_mu);
            g_timing_ms[which] += ms;
            g_timing_n[which] += 1;
        }
    }
    (void)cudaGetLastError();
}
KernelTimer::~KernelTimer() {
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
}
void timing_set(int on) {
    g_timing_on.store(on ? 1 : 0);
    std::lock_guard<std::mutex> lk(g_timing_mu);
    for (int i = 0; i < TK_COUNT; ++i) {
        g_timing_ms[i] = 0;
        g_timing_n[i] = 0;
    }
}
int timing_get(int which, double* ms, long long* n) {
    if (which < 0 || which >= TK_COUNT) return LIPFIT_E_PARAM;
    std::lock_guard<std::mutex> lk(g_timing_mu);
    if (ms) *ms = g_timing_ms[which];
    if (n) *n = g_timing_n[which];
    return LIPFIT_OK;
}

int make_ctx(void* cuda_stream, Ctx* ctx) {
    ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    int dev = 0;
    LIPFIT_CUDA(cudaGetDevice(&dev));
    static std::atomic<int> sm_cache[64];  // SM count per device ordinal (0 = not asked yet)
    int sms = (dev >= 0 && dev < 64) ? sm_cache[dev].load() : 0;
    if (sms == 0) {  // first call on this device
        LIPFIT_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        if (dev >= 0 && dev < 64) sm_cache[dev].store(sms);
    }
    ctx->device = dev;
    ctx->num_sms = sms;
    return LIPFIT_OK;
}

// Workspaces come from a pool of the library's own (common.cuh: Workspace).  A pool's default release
// threshold is 0: every synchronisation would hand the freed workspaces back to the driver and the next
// call would pay for mapping them again (0.2-0.6 ms on the 25 us config 1 step, tens of ms for the 0.5 GB
// of kNN pools), so this pool keeps them until lipfit_release_workspace().
namespace {
std::mutex g_pool_mu;
cudaMemPool_t g_pools[64] = {};
}  // namespace

cudaError_t workspace_pool(cudaMemPool_t* pool) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(g_pool_mu);
    if (!g_pools[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t p = nullptr;
        e = cudaMemPoolCreate(&p, &props);
        if (e != cudaSuccess) return e;
        unsigned long long keep = ~0ull;
        (void)cudaMemPoolSetAttribute(p, cudaMemPoolAttrReleaseThreshold, &keep);
        g_pools[dev] = p;
    }
    *pool = g_pools[dev];
    return cudaSuccess;
}

int workspace_release() {
    int dev = 0;
    LIPFIT_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return LIPFIT_E_CUDA;
    std::lock_guard<std::mutex> lk(g_pool_mu);
    if (g_pools[dev]) LIPFIT_CUDA(cudaMemPoolTrimTo(g_pools[dev], 0));
    return LIPFIT_OK;
}

cudaError_t occupancy_cached(const void* func, int threads, size_t smem, int* occ) {
    struct Key {
        const void* f;
        int t;
        size_t s;
        int dev;
        bool operator<(const Key& o) const {
            if (f != o.f) return f < o.f;
            if (t != o.t) return t < o.t;
            if (s != o.s) return s < o.s;
            return dev < o.dev;
        }
    };
    static std::mutex mu;
    static std::map<Key, int> cache;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const Key k{func, threads, smem, dev};
    {
        std::lock_guard<std::mutex> lk(mu);
        auto it = cache.find(k);
        if (it != cache.end()) {
            *occ = it->second;
            return cudaSuccess;
        }
    }
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, func, threads, smem);
    if (e == cudaSuccess) {
        std::lock_guard<std::mutex> lk(mu);
        cache[k] = *occ;
    }
    return e;
}

int make_xform(int32_t d, const int32_t* mono_mask, const float* weights, bool symmetric, bool flip,
               Xform* xf) {
    if (d < 1 || d > kMaxDim) return LIPFIT_E_DIM;
    int32_t s[kMaxDim];
    for (int i = 0; i < d; ++i) {
        int32_t m = mono_mask ? mono_mask[i] : 0;
        if (m < -1 || m > 1) return LIPFIT_E_PARAM;
        if (weights && !(weights[i] >= 0.f && std::isfinite(weights[i]))) return LIPFIT_E_PARAM;
        s[i] = symmetric ? 0 : (flip ? -m : m);
    }
    int n = 0;
    for (int i = 0; i < d; ++i)
        if (s[i] == 0) {
            xf->perm[n] = i;
            xf->sw[n] = weights ? weights[i] : 1.f;
            ++n;
        }
    xf->dU = n;
    for (int i = 0; i < d; ++i)
        if (s[i] != 0) {
            xf->perm[n] = i;
            xf->sw[n] = (weights ? weights[i] : 1.f) * (s[i] < 0 ? -1.f : 1.f);
            ++n;
        }
    xf->dC = n - xf->dU;
    xf->d = d;
    xf->dsrc = d;
    for (int i = d; i < kMaxDim; ++i) {
        xf->perm[i] = 0;
        xf->sw[i] = 0.f;
    }
    return LIPFIT_OK;
}

Xform scale_xform(const Xform& xf, float s) {
    Xform o = xf;
    for (int j = 0; j < kMaxDim; ++j) o.sw[j] = xf.sw[j] * s;
    return o;
}

FreeFlags make_free_flags(const Xform& xf) {
    FreeFlags ff;
    for (int j = 0; j < kMaxDim; ++j) ff.fr[j] = (j < xf.dU) ? 1.f : 0.f;
    ff.nfree4 = xf.dU / 4;
    ff.nall4 = (xf.d + 3) / 4;
    return ff;
}

// One thread per record; the record is assembled in registers and written as float4s.
__global__ void __launch_bounds__(256)
prepack_kernel(const float* __restrict__ X, const float* __restrict__ y,
               const float* __restrict__ eps, int N, Xform xf, int rf, int vslot, int cslot,
               const float* __restrict__ centre, float* __restrict__ rec) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const float* src = X + static_cast<size_t>(k) * xf.dsrc;
    float* dst = rec + static_cast<size_t>(k) * rf;
    float v = y ? y[k] : 0.f;
    if (eps) v += eps[k];
    // packed coordinate j = sw_j (x_perm(j) - centre_perm(j)); centre == NULL: no translation
    auto coord = [&](int j) {
        const int o = xf.perm[j];
        return xf.sw[j] * (centre ? src[o] - __ldg(centre + o) : src[o]);
    };
    float cval = 0.f;
    if (cslot >= 0) {  // folded L1 records (bounds.cu FoldL1Core): with sx = sum of the constrained (packed)
        float sc = 0.f;  // coordinates, the value slot holds y - sx and the c' slot 2 y - sx
        for (int j = xf.dU; j < xf.d; ++j) sc += coord(j);
        cval = 2.f * v - sc;
        v -= sc;
    }
    for (int j0 = 0; j0 < rf; j0 += 4) {
        float t[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            int j = j0 + c;
            t[c] = (j < xf.d) ? coord(j) : (j == vslot ? v : (j == cslot ? cval : 0.f));
        }
        *reinterpret_cast<float4*>(dst + j0) = make_float4(t[0], t[1], t[2], t[3]);
    }
}

// Duplicated layout for the packed-f32x2 kernels: logical record [x'_0..x'_{d-1}, value, c', 0..] of rf/2
// floats, each stored twice, so that an LDS.128 yields two (x, x) register pairs ready for FADD2.
__global__ void __launch_bounds__(256)
prepack_dup_kernel(const float* __restrict__ X, const float* __restrict__ y, int N, Xform xf, int rf, int vslot,
                   int cslot, const float* __restrict__ centre, float* __restrict__ rec) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const float* src = X + static_cast<size_t>(k) * xf.dsrc;
    float* dst = rec + static_cast<size_t>(k) * rf;
    float v = y ? y[k] : 0.f;
    auto coord = [&](int j) {
        const int o = xf.perm[j];
        return xf.sw[j] * (centre ? src[o] - __ldg(centre + o) : src[o]);
    };
    float cval = 0.f;
    if (cslot >= 0) {  // as prepack_kernel: value slot y - sx, c' slot 2 y - sx
        float sc = 0.f;
        for (int j = xf.dU; j < xf.d; ++j) sc += coord(j);
        cval = 2.f * v - sc;
        v -= sc;
    }
    for (int j0 = 0; j0 < rf / 2; j0 += 2) {
        float t[2];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            int j = j0 + c;
            t[c] = (j < xf.d) ? coord(j) : (j == vslot ? v : (j == cslot ? cval : 0.f));
        }
        *reinterpret_cast<float4*>(dst + 2 * j0) = make_float4(t[0], t[0], t[1], t[1]);
    }
}

__global__ void __launch_bounds__(256)
set_values_kernel(float* __restrict__ rec, int rf, int vslot, const float* __restrict__ y,
                  const float* __restrict__ eps, int N) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    rec[static_cast<size_t>(k) * rf + vslot] = y[k] + (eps ? eps[k] : 0.f);
}

__global__ void __launch_bounds__(256)
axpy_kernel(float* __restrict__ y, const float* __restrict__ eps, int N) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < N) y[k] += eps[k];
}

int launch_prepack(const Ctx& c, const float* X, const float* y, const float* eps, int64_t N,
                   const Xform& xf, RecLayout lay, float* rec, const float* centre) {
    int n = static_cast<int>(N);
    if (lay.dup) {
        prepack_dup_kernel<<<(n + 255) / 256, 256, 0, c.stream>>>(X, y, n, xf, lay.rf, lay.vslot, lay.cslot, centre,
                                                                  rec);
        ++g_launches;
        LIPFIT_CUDA(cudaGetLastError());
        return LIPFIT_OK;
    }
    prepack_kernel<<<(n + 255) / 256, 256, 0, c.stream>>>(X, y, eps, n, xf, lay.rf, lay.vslot, lay.cslot, centre,
                                                          rec);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

int launch_set_values(const Ctx& c, float* rec, RecLayout lay, const float* y, const float* eps,
                      int64_t N) {
    int n = static_cast<int>(N);
    set_values_kernel<<<(n + 255) / 256, 256, 0, c.stream>>>(rec, lay.rf, lay.vslot, y, eps, n);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

int launch_axpy(const Ctx& c, float* y, const float* eps, int64_t N) {
    int n = static_cast<int>(N);
    axpy_kernel<<<(n + 255) / 256, 256, 0, c.stream>>>(y, eps, n);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

}  // namespace lipfit
