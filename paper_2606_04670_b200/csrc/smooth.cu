// smooth.cu -- step a4: all-pairs objective and gradient of Eq.(7) PAPER.md:197,
// distances recomputed on the fly: nothing of size N x N is ever stored (the paper's precomputed
// d_ik / y_k - y_i matrices are its memory wall).
//
// With z = y + eps, D_ik = d_s(x^k, x^i) and V_ik = (z_i - z_k - M D_ik)_+ (reading R12):
//   F = ||eps||^2 / p + 2 sum_{i != k} V_ik^2 = ||eps||^2/p + sum_i sum_k (V_ik^2 + V_ki^2)
//   dF/deps_i = 2 eps_i / p + 4 sum_k (V_ik - V_ki).
// Row formulation: a thread owns R rows i (coordinates + z_i in registers) and sweeps the data k
// through shared memory exactly like the bounds kernel; the pair (i,k) yields both V_ik (from D^u of
// datum k seen from x^i) and V_ki (from D^l).  The k = i term is 0 by itself (D = 0, z_i - z_i = 0).
// fp32 pair arithmetic; sums leave the shared-memory tile in fp64; (row block, chunk) partials are
// combined in a fixed order, so an evaluation is bit-reproducible.
#include "kernels.h"

namespace lipfit {

struct SmoothArgs {
    const float* rec;
    double* gpart;  // [nch][N]   sum_k (V_ik - V_ki) over the chunk
    double* fpart;  // [ntiles]   sum of (V_ik^2 + V_ki^2) over the tile
    double* vpart;  // [ntiles]   max violation over the tile
    int N, nrb, nch, chunk;
    float M;
};

template <int RF>
__host__ __device__ constexpr int smooth_tile_records() {
    return RF <= 8 ? 512 : (RF <= 16 ? 256 : (RF <= 24 ? 128 : 96));
}

template <class Acc, int R, int THREADS>
__global__ void __launch_bounds__(THREADS, 2)
smooth_pairs_kernel(const SmoothArgs a, const FreeFlags ff) {
    constexpr int D = Acc::D;
    constexpr int RF = Acc::RF;
    constexpr int TILE = smooth_tile_records<RF>();
    __shared__ __align__(128) float sbuf[2 * TILE * RF];
    __shared__ __align__(8) uint64_t bars[2];
    __shared__ double redf[THREADS / 32];
    __shared__ float redv[THREADS / 32];
    if (threadIdx.x == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    uint32_t phase = 0;
    const int ntiles = a.nrb * a.nch;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int rb = tile / a.nch;
        const int ch = tile - rb * a.nch;
        float xi[R][D], zi[R];
        double fd[R], gd[R];
        float vmax = 0.f;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            int i = (rb * R + r) * THREADS + static_cast<int>(threadIdx.x);
            int ic = i < a.N ? i : a.N - 1;
            const float* src = a.rec + static_cast<size_t>(ic) * RF;
#pragma unroll
            for (int j = 0; j < D; ++j) xi[r][j] = __ldg(src + j);
            zi[r] = __ldg(src + Acc::VSLOT);
            fd[r] = 0.0;
            gd[r] = 0.0;
        }
        const int begin = ch * a.chunk;
        const int end = min(a.N, begin + a.chunk);
        RecordStream<TILE> rs(a.rec, RF, begin, end, sbuf, bars, &phase);
        for (int t = 0; t < rs.ntiles; ++t) {
            const float* s = rs.acquire(t);
            const int n = rs.count(t);
            float ft[R], gt[R];
#pragma unroll
            for (int r = 0; r < R; ++r) ft[r] = gt[r] = 0.f;
#pragma unroll 2
            for (int j = 0; j < n; ++j) {
                float x[RF];
#pragma unroll
                for (int c = 0; c < RF / 4; ++c) {
                    float4 v = reinterpret_cast<const float4*>(s + j * RF)[c];
                    x[4 * c + 0] = v.x;
                    x[4 * c + 1] = v.y;
                    x[4 * c + 2] = v.z;
                    x[4 * c + 3] = v.w;
                }
                const float zk = x[Acc::VSLOT];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    float au, al;
                    Acc::run(xi[r], x, ff, au, al);
                    float dz = zi[r] - zk;
                    float vik = fmaxf(fmaf(-a.M, Acc::finish(au), dz), 0.f);
                    float vki = fmaxf(fmaf(-a.M, Acc::finish(al), -dz), 0.f);
                    ft[r] = fmaf(vik, vik, ft[r]);
                    ft[r] = fmaf(vki, vki, ft[r]);
                    gt[r] += vik - vki;
                    vmax = fmaxf(vmax, fmaxf(vik, vki));
                }
            }
#pragma unroll
            for (int r = 0; r < R; ++r) {
                fd[r] += static_cast<double>(ft[r]);
                gd[r] += static_cast<double>(gt[r]);
            }
            rs.release(t);
        }
        // ---- per-row gradient partials, per-tile objective partial ----
        double fsum = 0.0;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            int i = (rb * R + r) * THREADS + static_cast<int>(threadIdx.x);
            if (i < a.N) {
                a.gpart[static_cast<size_t>(ch) * a.N + i] = gd[r];
                fsum += fd[r];
            }  // rows past N are clamped duplicates of row N-1: not counted (their vmax is harmless)
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            fsum += __shfl_xor_sync(0xffffffffu, fsum, o);
            vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
        }
        if ((threadIdx.x & 31) == 0) {
            redf[threadIdx.x >> 5] = fsum;
            redv[threadIdx.x >> 5] = vmax;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            double f = 0.0;
            float v = 0.f;
            for (int w = 0; w < THREADS / 32; ++w) {
                f += redf[w];
                v = fmaxf(v, redv[w]);
            }
            a.fpart[tile] = f;
            a.vpart[tile] = static_cast<double>(v);
        }
        __syncthreads();
    }
}

// grad[i] = 2 eps_i / p + 4 sum_ch gpart[ch][i]; per-block partial of sum eps^2.
__global__ void __launch_bounds__(256)
smooth_grad_kernel(const double* __restrict__ gpart, int nch, int N, const float* __restrict__ eps,
                   float p, float* __restrict__ grad, double* __restrict__ e2part) {
    __shared__ double red[8];
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    double e = 0.0;
    if (i < N) {
        double s = 0.0;
        for (int c = 0; c < nch; ++c) s += gpart[static_cast<size_t>(c) * N + i];
        e = eps ? static_cast<double>(eps[i]) : 0.0;
        if (grad) grad[i] = static_cast<float>(2.0 * e / static_cast<double>(p) + 4.0 * s);
    }
    double e2 = e * e;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e2 += __shfl_xor_sync(0xffffffffu, e2, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = e2;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += red[w];
        e2part[blockIdx.x] = t;
    }
}

// Single block, fixed order: F = sum(e2part)/p + sum(fpart); maxviol = max(vpart).
__global__ void __launch_bounds__(256)
smooth_final_kernel(const double* __restrict__ fpart, const double* __restrict__ vpart, int ntiles,
                    const double* __restrict__ e2part, int nblk, float p, double* __restrict__ F,
                    double* __restrict__ maxviol) {
    __shared__ double rf_[256], re_[256], rv_[256];
    double f = 0.0, e = 0.0, v = 0.0;
    for (int t = threadIdx.x; t < ntiles; t += 256) {
        f += fpart[t];
        v = fmax(v, vpart[t]);
    }
    for (int b = threadIdx.x; b < nblk; b += 256) e += e2part[b];
    rf_[threadIdx.x] = f;
    re_[threadIdx.x] = e;
    rv_[threadIdx.x] = v;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) {
            rf_[threadIdx.x] += rf_[threadIdx.x + o];
            re_[threadIdx.x] += re_[threadIdx.x + o];
            rv_[threadIdx.x] = fmax(rv_[threadIdx.x], rv_[threadIdx.x + o]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        if (F) *F = re_[0] / static_cast<double>(p) + rf_[0];
        if (maxviol) *maxviol = rv_[0];
    }
}

namespace {

template <class Acc, int R>
int launch_pairs(const Ctx& c, SmoothArgs& a, const FreeFlags& ff, const float* eps, float p,
                 double* F_dev, float* grad, double* maxviol_dev) {
    constexpr int THREADS = 128;
    auto kern = smooth_pairs_kernel<Acc, R, THREADS>;
    int occ = 0;
    LIPFIT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, THREADS, 0));
    if (occ < 1) occ = 1;
    const int slots = c.num_sms * occ;
    constexpr int TILE = smooth_tile_records<Acc::RF>();
    a.nrb = (a.N + THREADS * R - 1) / (THREADS * R);
    int want = (16 * slots + a.nrb - 1) / a.nrb;
    int max_ch = (a.N + 2 * TILE - 1) / (2 * TILE);
    int nch = want < 1 ? 1 : want;
    if (nch > max_ch) nch = max_ch;
    if (nch > 64) nch = 64;
    if (nch < 1) nch = 1;
    int chunk = (a.N + nch - 1) / nch;
    chunk = ((chunk + TILE - 1) / TILE) * TILE;
    nch = (a.N + chunk - 1) / chunk;
    a.nch = nch;
    a.chunk = chunk;
    const int ntiles = a.nrb * nch;
    const int nblk = (a.N + 255) / 256;

    Workspace w;
    size_t bytes = sizeof(double) * (static_cast<size_t>(nch) * a.N + 2 * static_cast<size_t>(ntiles) + nblk);
    int rc = w.alloc(bytes, c.stream);
    if (rc) return rc;
    a.gpart = w.as<double>();
    a.fpart = a.gpart + static_cast<size_t>(nch) * a.N;
    a.vpart = a.fpart + ntiles;
    double* e2part = a.vpart + ntiles;

    int grid = ntiles < slots ? ntiles : slots;
    KernelTimer kt(TK_SMOOTH_PAIRS, c.stream);
    kern<<<grid, THREADS, 0, c.stream>>>(a, ff);
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    smooth_grad_kernel<<<nblk, 256, 0, c.stream>>>(a.gpart, nch, a.N, eps, p, grad, e2part);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    if (F_dev || maxviol_dev) {
        smooth_final_kernel<<<1, 256, 0, c.stream>>>(a.fpart, a.vpart, ntiles, e2part, nblk, p, F_dev,
                                                     maxviol_dev);
        ++g_launches;
        LIPFIT_CUDA(cudaGetLastError());
    }
    return LIPFIT_OK;
}

int smooth_dp(int d) { return d <= 4 ? 4 : (d <= 8 ? 8 : (d <= 16 ? 16 : 32)); }
bool is_spec(const Xform& xf, int norm) {
    return (norm == 2 && xf.dU == 0 && xf.dC == 5) || (norm == 2 && xf.dU == 2 && xf.dC == 0);
}

}  // namespace

RecLayout smooth_layout(const Xform& xf, int norm) {
    if (is_spec(xf, norm)) return RecLayout{record_floats(xf.d), xf.d};
    int dp = smooth_dp(xf.d);
    return RecLayout{dp + 4, dp};
}

int launch_smooth_objective(const Ctx& c, const float* rec, int64_t N, const Xform& xf, int norm,
                            float M, float p, const float* eps, double* F_dev, float* grad,
                            double* maxviol_dev) {
    SmoothArgs a{};
    a.rec = rec;
    a.N = static_cast<int>(N);
    a.M = M;
    FreeFlags ff = make_free_flags(xf);
#define GO(ACC, R) return launch_pairs<ACC, R>(c, a, ff, eps, p, F_dev, grad, maxviol_dev)
    using S205 = SpecAcc<2, 0, 5>;
    using S220 = SpecAcc<2, 2, 0>;
    using G14 = GenAcc<1, 4>;
    using G18 = GenAcc<1, 8>;
    using G116 = GenAcc<1, 16>;
    using G132 = GenAcc<1, 32>;
    using G24 = GenAcc<2, 4>;
    using G28 = GenAcc<2, 8>;
    using G216 = GenAcc<2, 16>;
    using G232 = GenAcc<2, 32>;
    using G34 = GenAcc<3, 4>;
    using G38 = GenAcc<3, 8>;
    using G316 = GenAcc<3, 16>;
    using G332 = GenAcc<3, 32>;
    if (norm == 2 && xf.dU == 0 && xf.dC == 5) GO(S205, 8);
    if (norm == 2 && xf.dU == 2 && xf.dC == 0) GO(S220, 8);
    const int dp = smooth_dp(xf.d);
    if (norm == 1) {
        if (dp == 4) GO(G14, 4);
        if (dp == 8) GO(G18, 4);
        if (dp == 16) GO(G116, 2);
        GO(G132, 1);
    } else if (norm == 2) {
        if (dp == 4) GO(G24, 4);
        if (dp == 8) GO(G28, 4);
        if (dp == 16) GO(G216, 2);
        GO(G232, 1);
    } else {
        if (dp == 4) GO(G34, 4);
        if (dp == 8) GO(G38, 4);
        if (dp == 16) GO(G316, 2);
        GO(G332, 1);
    }
#undef GO
}

}  // namespace lipfit
