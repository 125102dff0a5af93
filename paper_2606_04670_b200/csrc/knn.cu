// knn.cu -- step a3: fused distance + per-query top-k.
// Neighbours by distance d_(1) <= d_(2) <= ... without the cdist matrix + topk of
// PAPER.md:206.  Two device passes:
//   (1) selection in fp32: every thread keeps R queries in registers, streams packed records through
//       shared memory (TMA bulk copies) and compares each pair's accumulated distance (squared for
//       L2) with the query's current threshold tau = worst distance of its candidate list; only the
//       rare pair that passes (k ln(N/k) of N) touches the list, a sorted array of ksel = k + margin
//       entries kept in an L2-resident workspace laid out [slot][query] so that a warp's accesses
//       coalesce;
//   (2) re-rank in fp64: the candidates' distances are recomputed in double from the ORIGINAL fp32
//       inputs, ordered by (distance, index), and the first k are emitted (this makes
//       the result independent of the fp32 selection arithmetic as long as the pool is a superset).
#include <cfloat>

#include "kernels.h"

namespace lipfit {

constexpr int kKnnMargin = 8;

struct KnnArgs {
    const float* rec;
    const float* Xq;
    float* Ld;   // [nch][ksel][Qp]
    int32_t* Li; // [nch][ksel][Qp]
    int N, Q, Qp, d, ksel;
    int nqb, nch, chunk;
    Xform xf;
};

__device__ __noinline__ float knn_insert(float* Ld, int32_t* Li, size_t stride, int ksel, float dv,
                                         int32_t iv) {
    int p = ksel - 1;
    while (p > 0) {
        float prev = Ld[(p - 1) * stride];
        if (!(prev > dv)) break;
        Ld[p * stride] = prev;
        Li[p * stride] = Li[(p - 1) * stride];
        --p;
    }
    Ld[p * stride] = dv;
    Li[p * stride] = iv;
    return Ld[(ksel - 1) * stride];
}

template <int DP>
__host__ __device__ constexpr int knn_tile_records() {
    return DP <= 8 ? 512 : (DP <= 16 ? 256 : 128);
}

template <int NORM, int DP, bool ONESIDED, int R, int THREADS>
__global__ void __launch_bounds__(THREADS, 2)
knn_select_kernel(const KnnArgs a, const FreeFlags ff) {
    constexpr int TILE = knn_tile_records<DP>();
    __shared__ __align__(128) float sbuf[2 * TILE * DP];
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
        float q[R][DP];
        float tau[R];
        int qidx[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            int qi = (qb * R + r) * THREADS + static_cast<int>(threadIdx.x);
            qidx[r] = qi;
            int qc = qi < a.Q ? qi : a.Q - 1;
            const float* src = a.Xq + static_cast<size_t>(qc) * a.d;
#pragma unroll
            for (int j = 0; j < DP; ++j)
                q[r][j] = (j < a.d) ? a.xf.sw[j] * __ldg(src + a.xf.perm[j]) : 0.f;
            tau[r] = __int_as_float(0x7f800000);
        }
        const size_t stride = static_cast<size_t>(a.Qp);
        float* Ld = a.Ld + static_cast<size_t>(ch) * a.ksel * stride;
        int32_t* Li = a.Li + static_cast<size_t>(ch) * a.ksel * stride;

        const int begin = ch * a.chunk;
        const int end = min(a.N, begin + a.chunk);
        RecordStream<TILE> rs(a.rec, DP, begin, end, sbuf, bars, &phase);
        for (int t = 0; t < rs.ntiles; ++t) {
            const float* s = rs.acquire(t);
            const int n = rs.count(t);
            const int base = begin + t * TILE;
            for (int j = 0; j < n; ++j) {
                float x[DP];
#pragma unroll
                for (int c = 0; c < DP / 4; ++c) {
                    float4 v = reinterpret_cast<const float4*>(s + j * DP)[c];
                    x[4 * c + 0] = v.x;
                    x[4 * c + 1] = v.y;
                    x[4 * c + 2] = v.z;
                    x[4 * c + 3] = v.w;
                }
                float sv[R];
                bool any = false;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    sv[r] = ONESIDED ? PairAccGeneric<NORM, DP>::run_u(q[r], x, ff)
                                     : PairAccU<NORM, DP, 0>::run(q[r], x);
                    any |= (sv[r] < tau[r]);
                }
                if (any) {
#pragma unroll
                    for (int r = 0; r < R; ++r)
                        if (sv[r] < tau[r] && qidx[r] < a.Q)
                            tau[r] = knn_insert(Ld + qidx[r], Li + qidx[r], stride, a.ksel, sv[r],
                                                base + j);
                }
            }
            rs.release(t);
        }
    }
}

__global__ void __launch_bounds__(256)
knn_fill_kernel(float* __restrict__ Ld, int32_t* __restrict__ Li, size_t n) {
    size_t i = static_cast<size_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i < n) {
        Ld[i] = __int_as_float(0x7f800000);
        Li[i] = -1;
    }
}

// One warp per query.  Pool = nch * ksel candidates (index -1 = empty slot).
struct RerankArgs {
    const float* X;
    const float* Xq;
    const int32_t* Li;
    int32_t* idx;
    float* dist;
    int N, Q, Qp, d, pool, k, norm;
    Xform xf;  // perm/sw of the ORIGINAL coordinates; dU tells which packed coords are free
};

constexpr int kRerankWarps = 4;
constexpr int kMaxPool = 768;

__global__ void __launch_bounds__(kRerankWarps * 32)
knn_rerank_kernel(const RerankArgs a) {
    __shared__ double sd[kRerankWarps][kMaxPool];
    __shared__ int32_t si[kRerankWarps][kMaxPool];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int qi = blockIdx.x * kRerankWarps + warp;
    if (qi >= a.Q) return;
    const float* xq = a.Xq + static_cast<size_t>(qi) * a.d;
    for (int c = lane; c < a.pool; c += 32) {
        int32_t id = a.Li[static_cast<size_t>(c) * a.Qp + qi];
        double acc = 0.0;
        if (id >= 0) {
            const float* xk = a.X + static_cast<size_t>(id) * a.d;
            for (int j = 0; j < a.d; ++j) {
                int o = a.xf.perm[j];
                double sw = static_cast<double>(a.xf.sw[j]);
                double dlt = sw * (static_cast<double>(xq[o]) - static_cast<double>(xk[o]));
                double comp = (j < a.xf.dU) ? fabs(dlt) : fmax(dlt, 0.0);
                if (a.norm == 1) acc += comp;
                else if (a.norm == 2) acc += comp * comp;
                else acc = fmax(acc, comp);
            }
            if (a.norm == 2) acc = sqrt(acc);
        } else {
            acc = __longlong_as_double(0x7ff0000000000000LL);
            id = 0x7fffffff;
        }
        sd[warp][c] = acc;
        si[warp][c] = id;
    }
    __syncwarp();
    for (int c = lane; c < a.pool; c += 32) {
        double dc = sd[warp][c];
        int32_t ic = si[warp][c];
        int rank = 0;
        for (int o = 0; o < a.pool; ++o) {
            double d2 = sd[warp][o];
            int32_t i2 = si[warp][o];
            rank += (d2 < dc) || (d2 == dc && i2 < ic);
        }
        if (rank < a.k) {
            a.idx[static_cast<size_t>(qi) * a.k + rank] = ic;
            a.dist[static_cast<size_t>(qi) * a.k + rank] = static_cast<float>(dc);
        }
    }
}

namespace {

template <int NORM, int DP, bool ONESIDED>
int launch_select(const Ctx& c, KnnArgs& a, const FreeFlags& ff) {
    constexpr int R = (DP <= 8) ? 8 : (DP <= 16 ? 4 : 2);
    constexpr int THREADS = 128;
    auto kern = knn_select_kernel<NORM, DP, ONESIDED, R, THREADS>;
    int occ = 0;
    LIPFIT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, THREADS, 0));
    if (occ < 1) occ = 1;
    const int slots = c.num_sms * occ;
    long long ntiles = static_cast<long long>(a.nqb) * a.nch;
    int grid = static_cast<int>(ntiles < slots ? ntiles : slots);
    KernelTimer kt(TK_KNN_SELECT, c.stream);
    kern<<<grid, THREADS, 0, c.stream>>>(a, ff);
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

template <int NORM, bool ONESIDED>
int dispatch_dp(const Ctx& c, KnnArgs& a, const FreeFlags& ff, int dp) {
    switch (dp) {
        case 4: return launch_select<NORM, 4, ONESIDED>(c, a, ff);
        case 8: return launch_select<NORM, 8, ONESIDED>(c, a, ff);
        case 16: return launch_select<NORM, 16, ONESIDED>(c, a, ff);
        default: return launch_select<NORM, 32, ONESIDED>(c, a, ff);
    }
}

int knn_dp(int d) { return d <= 4 ? 4 : (d <= 8 ? 8 : (d <= 16 ? 16 : 32)); }
int knn_r(int dp) { return dp <= 8 ? 8 : (dp <= 16 ? 4 : 2); }

}  // namespace

RecLayout knn_layout(const Xform& xf, int) { return RecLayout{knn_dp(xf.d), -1}; }

int launch_knn(const Ctx& c, const float* X, const float* rec, int64_t N, const float* Xq, int64_t Q,
               const Xform& xf, int norm, int k, int32_t* idx, float* dist) {
    KnnArgs a{};
    const int dp = knn_dp(xf.d);
    a.rec = rec;
    a.Xq = Xq;
    a.N = static_cast<int>(N);
    a.Q = static_cast<int>(Q);
    a.d = xf.d;
    a.xf = xf;
    a.ksel = static_cast<int>(N < k + kKnnMargin ? N : k + kKnnMargin);
    const int qper = 128 * knn_r(dp);
    a.nqb = (a.Q + qper - 1) / qper;
    a.Qp = a.nqb * qper;
    // Data chunks: only when the query blocks alone cannot fill the chip (small Q, large N).
    int nch = 1;
    const int slots = c.num_sms * 2;
    if (a.nqb < slots) {
        nch = (slots + a.nqb - 1) / a.nqb;
        int max_ch = kMaxPool / a.ksel;
        if (nch > max_ch) nch = max_ch;
        int by_n = a.N / (4 * a.ksel);
        if (nch > by_n) nch = by_n;
        if (nch < 1) nch = 1;
    }
    const int tile = dp <= 8 ? 512 : (dp <= 16 ? 256 : 128);
    int chunk = (a.N + nch - 1) / nch;
    chunk = ((chunk + tile - 1) / tile) * tile;
    nch = (a.N + chunk - 1) / chunk;
    a.nch = nch;
    a.chunk = chunk;

    const size_t entries = static_cast<size_t>(nch) * a.ksel * a.Qp;
    Workspace wd, wi;
    int rc = wd.alloc(entries * sizeof(float), c.stream);
    if (rc) return rc;
    rc = wi.alloc(entries * sizeof(int32_t), c.stream);
    if (rc) return rc;
    a.Ld = wd.as<float>();
    a.Li = wi.as<int32_t>();
    knn_fill_kernel<<<static_cast<unsigned>((entries + 255) / 256), 256, 0, c.stream>>>(a.Ld, a.Li,
                                                                                       entries);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());

    FreeFlags ff = make_free_flags(xf);
    const bool onesided = xf.dC > 0;
    if (norm == 1)
        rc = onesided ? dispatch_dp<1, true>(c, a, ff, dp) : dispatch_dp<1, false>(c, a, ff, dp);
    else if (norm == 2)
        rc = onesided ? dispatch_dp<2, true>(c, a, ff, dp) : dispatch_dp<2, false>(c, a, ff, dp);
    else
        rc = onesided ? dispatch_dp<3, true>(c, a, ff, dp) : dispatch_dp<3, false>(c, a, ff, dp);
    if (rc) return rc;

    RerankArgs r{};
    r.X = X;
    r.Xq = Xq;
    r.Li = a.Li;
    r.idx = idx;
    r.dist = dist;
    r.N = a.N;
    r.Q = a.Q;
    r.Qp = a.Qp;
    r.d = a.d;
    r.pool = nch * a.ksel;
    r.k = k;
    r.norm = norm;
    r.xf = xf;
    knn_rerank_kernel<<<(a.Q + kRerankWarps - 1) / kRerankWarps, kRerankWarps * 32, 0, c.stream>>>(r);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

}  // namespace lipfit
