// small.cu -- step a2 for SMALL data sets (BASELINE.json configs[0]: N = 1000, Q = 10000, 1e7 pairs): Eq.(2),(3)
// PAPER.md:103-116 in ONE kernel launch.  Such a call is bound by launch latency, not by arithmetic (1e7 pairs are
// ~3 us of work for the chip): the general path costs five stream operations (prepack, two key
// memsets, the chunked bounds kernel, finalize).  Here every CTA packs ALL N data into its own shared memory
// (step a1 inside the kernel: N records of DP + 4 floats, at most 46 KB), then 32 queries (lane = query) meet
// the data in 8 interleaved slices (warp = slice, broadcast LDS.128), the eight partial extrema meet through
// shared memory and the outputs are written directly: no workspace, no atomics, no second kernel.
#include "kernels.h"

namespace lipfit {

namespace {

constexpr int kSmallThreads = 256;  // 8 warps = 8 data slices
constexpr int kSmallQueries = 32;   // queries per CTA (lane = query)
constexpr int kSmallBytes = 46 * 1024;  // records; + 2 KB of static shared memory = the 48 KB a CTA gets without opting in

struct SmallArgs {
    const float* X;
    const float* y;
    const float* Xq;
    float *upper, *lower, *g;
    int N, Q;
    float M;
    Xform xf;
};

// DA > 0: symmetric distance (no constrained coordinate) over exactly DA coordinates (compile time, d <= 8);
// DA == 0: any mask, flag arithmetic over the DP padded coordinates.
template <int NORM, int DP, int DA>
__global__ void __launch_bounds__(kSmallThreads)
bounds_small_kernel(const SmallArgs a, const FreeFlags ff) {
    constexpr int RF = DP + 4;
    constexpr int DQ = DA > 0 ? DA : DP;
    extern __shared__ __align__(16) float srec[];  // [N][RF]
    __shared__ float sU[kSmallThreads / 32][kSmallQueries], sL[kSmallThreads / 32][kSmallQueries];
    // ---- a1 inside the kernel: packed records [x'_0 .. x'_{DP-1}, y, 0, 0, 0] ----
#pragma unroll 4  // (the non-coherent loads of four records are in flight together: cold data, ~1 us each)
    for (int k = threadIdx.x; k < a.N; k += kSmallThreads) {
        const float* src = a.X + static_cast<size_t>(k) * a.xf.dsrc;
        float4* dst = reinterpret_cast<float4*>(srec + k * RF);
#pragma unroll
        for (int j0 = 0; j0 < DP; j0 += 4) {
            float t[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const int j = j0 + c;
                t[c] = j < a.xf.d ? a.xf.sw[j] * __ldg(src + a.xf.perm[j]) : 0.f;
            }
            dst[j0 >> 2] = make_float4(t[0], t[1], t[2], t[3]);
        }
        dst[DP >> 2] = make_float4(__ldg(a.y + k), 0.f, 0.f, 0.f);
    }
    const int lane = threadIdx.x & 31, slice = threadIdx.x >> 5;
    const int qi = blockIdx.x * kSmallQueries + lane;
    float q[DQ];
    {
        const float* src = a.Xq + static_cast<size_t>(qi < a.Q ? qi : a.Q - 1) * a.xf.dsrc;
#pragma unroll
        for (int j = 0; j < DQ; ++j) q[j] = j < a.xf.d ? a.xf.sw[j] * __ldg(src + a.xf.perm[j]) : 0.f;
    }
    __syncthreads();
    float U = __int_as_float(0x7f800000), L = __int_as_float(0xff800000);
#pragma unroll 4
    for (int k = slice; k < a.N; k += kSmallThreads / 32) {
        float x[RF];
#pragma unroll
        for (int c = 0; c < RF / 4; ++c) {
            const float4 v = reinterpret_cast<const float4*>(srec + k * RF)[c];
            x[4 * c] = v.x;
            x[4 * c + 1] = v.y;
            x[4 * c + 2] = v.z;
            x[4 * c + 3] = v.w;
        }
        float au, al;
        if (DA > 0) {
            au = al = PairAccU<NORM, DQ, 0>::run(q, x);
        } else {
            PairAccGeneric<NORM, DP>::run(q, x, ff, au, al);
        }
        const float du = NORM == 2 ? fast_sqrt(au) : au;
        const float dl = (DA > 0) ? du : (NORM == 2 ? fast_sqrt(al) : al);
        U = fminf(U, fmaf(a.M, du, x[DP]));
        L = fmaxf(L, fmaf(-a.M, dl, x[DP]));
    }
    sU[slice][lane] = U;
    sL[slice][lane] = L;
    __syncthreads();
    if (slice == 0 && qi < a.Q) {
#pragma unroll
        for (int s = 1; s < kSmallThreads / 32; ++s) {
            U = fminf(U, sU[s][lane]);
            L = fmaxf(L, sL[s][lane]);
        }
        if (a.upper) a.upper[qi] = U;
        if (a.lower) a.lower[qi] = L;
        if (a.g) a.g[qi] = 0.5f * (U + L);
    }
}

template <int NORM, int DP, int DA>
int launch_small_t(const Ctx& c, const SmallArgs& a, const FreeFlags& ff) {
    const size_t smem = sizeof(float) * static_cast<size_t>(a.N) * (DP + 4);
    const int grid = (a.Q + kSmallQueries - 1) / kSmallQueries;
    KernelTimer kt(TK_BOUNDS, c.stream);
    bounds_small_kernel<NORM, DP, DA><<<grid, kSmallThreads, smem, c.stream>>>(a, ff);
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

template <int NORM>
int launch_small_n(const Ctx& c, const SmallArgs& a, const FreeFlags& ff) {
    const int d = a.xf.d;
    if (a.xf.dC == 0) {  // symmetric: exact-d arithmetic for d <= 8
        switch (d) {
            case 1: return launch_small_t<NORM, 4, 1>(c, a, ff);
            case 2: return launch_small_t<NORM, 4, 2>(c, a, ff);
            case 3: return launch_small_t<NORM, 4, 3>(c, a, ff);
            case 4: return launch_small_t<NORM, 4, 4>(c, a, ff);
            case 5: return launch_small_t<NORM, 8, 5>(c, a, ff);
            case 6: return launch_small_t<NORM, 8, 6>(c, a, ff);
            case 7: return launch_small_t<NORM, 8, 7>(c, a, ff);
            case 8: return launch_small_t<NORM, 8, 8>(c, a, ff);
            default: break;
        }
    }
    if (d <= 4) return launch_small_t<NORM, 4, 0>(c, a, ff);
    if (d <= 8) return launch_small_t<NORM, 8, 0>(c, a, ff);
    if (d <= 16) return launch_small_t<NORM, 16, 0>(c, a, ff);
    return launch_small_t<NORM, 32, 0>(c, a, ff);
}

int small_dp(int d) { return d <= 4 ? 4 : (d <= 8 ? 8 : (d <= 16 ? 16 : 32)); }

}  // namespace

// the whole data set fits the shared memory a CTA gets without opting in, and the call is small enough
// (<= 2^25 pairs: tens of microseconds) for launch latency to dominate over the tuned pair arithmetic of the
// general path
bool bounds_small_applies(const Xform& xf, int64_t N, int64_t Q) {
    return static_cast<size_t>(N) * (small_dp(xf.d) + 4) * sizeof(float) <= static_cast<size_t>(kSmallBytes) &&
           N * Q <= (1LL << 25);
}

int launch_bounds_small(const Ctx& c, const float* X, const float* y, int64_t N, const float* Xq, int64_t Q,
                        const Xform& xf, int norm, float M, float* upper, float* lower, float* g) {
    SmallArgs a{};
    a.X = X;
    a.y = y;
    a.Xq = Xq;
    a.upper = upper;
    a.lower = lower;
    a.g = g;
    a.N = static_cast<int>(N);
    a.Q = static_cast<int>(Q);
    a.M = M;
    a.xf = xf;
    const FreeFlags ff = make_free_flags(xf);
    if (norm == 1) return launch_small_n<1>(c, a, ff);
    if (norm == 2) return launch_small_n<2>(c, a, ff);
    return launch_small_n<3>(c, a, ff);
}

}  // namespace lipfit
