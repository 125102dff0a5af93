// noalloc.cu -- lipfit_bounds_noalloc: Eq.(2),(3) PAPER.md:103-116 (distance of Eq.(4)) for callers
// that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc).  A variant of the generic fused bounds kernel of bounds.cu whose scratch -- the packed data
// records of step a1 and the order-preserving keys through which the partial extrema of data chunks meet --
// lives in ONE file-scope device array of a fixed size instead of stream-ordered workspaces:
//     g_scratch : kScratchBytes = 8 MiB, held by every GPU that loads the library until the process exits.
// The entry point calls no cudaMalloc / cudaFree / cudaMallocAsync and no allocating library routine, only kernel
// launches on the caller's stream.  Sizes beyond the array are rejected with LIPFIT_E_LIMIT.
//
// Every call shares the array, and it keeps the last call's contents: each call rewrites the records it reads
// and re-initialises the keys it uses (inside its pack kernel) before the bounds kernel runs -- nothing relies on
// zeros.  Calls that overlap on the GPU (two streams, two threads) RACE on it: callers serialise them.
//
// In host code `g_scratch` is a host-side stand-in for the symbol, not a device address: the address the kernels
// get comes from cudaGetSymbolAddress, taken once per device with that device current (scratch_of_current_device).
#include <mutex>

#include "kernels.h"

namespace lipfit {

namespace {

constexpr size_t kRecFloats = LIPFIT_NOALLOC_MAX_RECORD_FLOATS;  // records region: 4 MiB
constexpr size_t kMaxQ = LIPFIT_NOALLOC_MAX_Q;                   // keys region: 2 x 4 B x Q = 4 MiB
constexpr size_t kScratchBytes = kRecFloats * sizeof(float) + 2 * kMaxQ * sizeof(uint32_t);
static_assert(kScratchBytes == (8u << 20), "stated size of the fixed scratch: 8 MiB");

static __device__ __align__(256) unsigned char g_scratch[kScratchBytes];

// device address of g_scratch on the CURRENT device, looked up once per device ordinal
int scratch_of_current_device(unsigned char** out) {
    static std::mutex mu;
    static unsigned char* addr[64] = {};
    int dev = 0;
    LIPFIT_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return LIPFIT_E_CUDA;
    std::lock_guard<std::mutex> lk(mu);
    if (!addr[dev]) {
        unsigned char* p = nullptr;
        LIPFIT_CUDA(cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_scratch));
        if (!p) return LIPFIT_E_CUDA;
        addr[dev] = p;
    }
    *out = addr[dev];
    return LIPFIT_OK;
}

struct NoAllocArgs {
    const float* X;
    const float* y;
    const float* Xq;
    float* rec;      // scratch: [N][DP + 4] records [x'_0 .. x'_{DP-1}, y, 0, 0, 0]
    uint32_t* keyU;  // scratch: [Q] running minimum of the upper candidates (order-preserving keys)
    uint32_t* keyL;  // scratch: [Q] running maximum of the lower candidates
    float *upper, *lower, *g;
    int N, Q, nqb, nch, chunk;
    float M;
    Xform xf;
};

// step a1 into the fixed scratch + (re)initialisation of the keys this call uses
__global__ void __launch_bounds__(256)
noalloc_pack_kernel(const NoAllocArgs a, int dp) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < a.N) {
        const float* src = a.X + static_cast<size_t>(k) * a.xf.dsrc;
        float4* dst = reinterpret_cast<float4*>(a.rec + static_cast<size_t>(k) * (dp + 4));
        for (int j0 = 0; j0 < dp; j0 += 4) {
            float t[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const int j = j0 + c;
                t[c] = j < a.xf.d ? a.xf.sw[j] * src[a.xf.perm[j]] : 0.f;
            }
            dst[j0 >> 2] = make_float4(t[0], t[1], t[2], t[3]);
        }
        dst[dp >> 2] = make_float4(a.y[k], 0.f, 0.f, 0.f);
    }
    if (k < a.Q) {
        a.keyU[k] = 0xFFFFFFFFu;
        a.keyL[k] = 0u;
    }
}

constexpr int kThreads = 128;

template <int DP>
__host__ __device__ constexpr int noalloc_tile() {
    return DP <= 4 ? 512 : (DP <= 8 ? 256 : (DP <= 16 ? 128 : 64));
}

// the generic fused bounds kernel (flag arithmetic of dist.cuh: any mask, d <= DP), R queries per thread
template <int NORM, int DP, int R>
__global__ void __launch_bounds__(kThreads, 2)
bounds_noalloc_kernel(const NoAllocArgs a, const FreeFlags ff) {
    constexpr int RF = DP + 4;
    constexpr int TILE = noalloc_tile<DP>();
    __shared__ __align__(128) float sbuf[2 * TILE * RF];
    __shared__ __align__(8) uint64_t bars[2];
    if (threadIdx.x == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    uint32_t phase = 0;
    const int ntiles = a.nqb * a.nch;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int qb = tile / a.nch;
        const int ch = tile - qb * a.nch;
        float q[R][DP], U[R], L[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            int qi = (qb * R + r) * kThreads + static_cast<int>(threadIdx.x);
            qi = qi < a.Q ? qi : a.Q - 1;
            const float* src = a.Xq + static_cast<size_t>(qi) * a.xf.dsrc;
#pragma unroll
            for (int j = 0; j < DP; ++j) q[r][j] = (j < a.xf.d) ? a.xf.sw[j] * __ldg(src + a.xf.perm[j]) : 0.f;
            U[r] = __int_as_float(0x7f800000);
            L[r] = __int_as_float(0xff800000);
        }
        const int begin = ch * a.chunk;
        const int end = min(a.N, begin + a.chunk);
        RecordStream<TILE> rs(a.rec, RF, begin, end, sbuf, bars, &phase);
        for (int t = 0; t < rs.ntiles; ++t) {
            const float* s = rs.acquire(t);
            const int n = rs.count(t);
            for (int j = 0; j < n; ++j) {
                float x[RF];
#pragma unroll
                for (int c = 0; c < RF / 4; ++c) {
                    const float4 v = reinterpret_cast<const float4*>(s + j * RF)[c];
                    x[4 * c] = v.x;
                    x[4 * c + 1] = v.y;
                    x[4 * c + 2] = v.z;
                    x[4 * c + 3] = v.w;
                }
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    float au, al;
                    PairAccGeneric<NORM, DP>::run(q[r], x, ff, au, al);
                    U[r] = fminf(U[r], fmaf(a.M, PairAccGeneric<NORM, DP>::finish(au), x[DP]));
                    L[r] = fmaxf(L[r], fmaf(-a.M, PairAccGeneric<NORM, DP>::finish(al), x[DP]));
                }
            }
            rs.release(t);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int qi = (qb * R + r) * kThreads + static_cast<int>(threadIdx.x);
            if (qi < a.Q) {
                atomicMin(a.keyU + qi, f2key(U[r]));
                atomicMax(a.keyL + qi, f2key(L[r]));
            }
        }
    }
}

template <int NORM, int DP>
int launch_noalloc(const Ctx& c, NoAllocArgs& a, const FreeFlags& ff) {
    constexpr int R = DP <= 8 ? 4 : (DP <= 16 ? 2 : 1);
    constexpr int TILE = noalloc_tile<DP>();
    const int slots = 2 * c.num_sms;  // __launch_bounds__(128, 2)
    a.nqb = (a.Q + kThreads * R - 1) / (kThreads * R);
    // as bounds.cu: cut the data into chunks until there are ~16 tiles per resident CTA, chunks >= 4 smem tiles
    int want = (16 * slots + a.nqb - 1) / a.nqb;
    const int max_ch = (a.N + 4 * TILE - 1) / (4 * TILE);
    int nch = want < 1 ? 1 : want;
    if (nch > max_ch) nch = max_ch;
    if (nch < 1) nch = 1;
    int chunk = (a.N + nch - 1) / nch;
    chunk = ((chunk + TILE - 1) / TILE) * TILE;
    nch = (a.N + chunk - 1) / chunk;
    a.nch = nch;
    a.chunk = chunk;
    const int big = a.N > a.Q ? a.N : a.Q;
    noalloc_pack_kernel<<<(big + 255) / 256, 256, 0, c.stream>>>(a, DP);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    const long long ntiles = static_cast<long long>(a.nqb) * nch;
    bounds_noalloc_kernel<NORM, DP, R><<<static_cast<int>(ntiles < slots ? ntiles : slots), kThreads, 0, c.stream>>>(a, ff);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return launch_bounds_finalize(c, a.keyU, a.keyL, a.Q, a.upper, a.lower, a.g);
}

template <int NORM>
int launch_noalloc_n(const Ctx& c, NoAllocArgs& a, const FreeFlags& ff, int dp) {
    switch (dp) {
        case 4: return launch_noalloc<NORM, 4>(c, a, ff);
        case 8: return launch_noalloc<NORM, 8>(c, a, ff);
        case 16: return launch_noalloc<NORM, 16>(c, a, ff);
        default: return launch_noalloc<NORM, 32>(c, a, ff);
    }
}

}  // namespace

int launch_bounds_noalloc(const Ctx& c, const float* X, const float* y, int64_t N, const float* Xq, int64_t Q,
                          const Xform& xf, int norm, float M, float* upper, float* lower, float* g) {
    const int dp = xf.d <= 4 ? 4 : (xf.d <= 8 ? 8 : (xf.d <= 16 ? 16 : 32));
    if (static_cast<size_t>(N) * static_cast<size_t>(dp + 4) > kRecFloats || static_cast<size_t>(Q) > kMaxQ)
        return LIPFIT_E_LIMIT;
    unsigned char* scratch = nullptr;
    int rc = scratch_of_current_device(&scratch);
    if (rc) return rc;
    NoAllocArgs a{};
    a.X = X;
    a.y = y;
    a.Xq = Xq;
    a.rec = reinterpret_cast<float*>(scratch);
    a.keyU = reinterpret_cast<uint32_t*>(scratch + kRecFloats * sizeof(float));
    a.keyL = a.keyU + kMaxQ;
    a.upper = upper;
    a.lower = lower;
    a.g = g;
    a.N = static_cast<int>(N);
    a.Q = static_cast<int>(Q);
    a.M = M;
    a.xf = xf;
    const FreeFlags ff = make_free_flags(xf);
    if (norm == 1) return launch_noalloc_n<1>(c, a, ff, dp);
    if (norm == 2) return launch_noalloc_n<2>(c, a, ff, dp);
    return launch_noalloc_n<3>(c, a, ff, dp);
}

}  // namespace lipfit
