// knn.cu -- step a3: fused distance + per-query top-k.
// Neighbours by distance d_(1) <= d_(2) <= ... without the cdist matrix + topk of
// PAPER.md:206.  Two device passes:
//   (1) selection in fp32.  Every thread keeps R queries in registers and streams packed records
//       through shared memory (TMA bulk copies), exactly like the bounds kernel.  Per query it holds a
//       threshold tau and a fill count in registers; a pair whose accumulated distance (squared for
//       L2) is below tau is APPENDED (one 8-byte fire-and-forget store) to the query's candidate pool
//       of P = 2*ksel entries, ksel = k + margin, in an L2-resident workspace.  When a pool is full
//       the whole warp compacts it (rank by counting in shared memory), keeps the ksel best in sorted
//       order and lowers tau to the ksel-th best.  tau only decreases, so the pool always contains
//       the ksel best of the data seen so far, for ANY data order; a pool is compacted about
//       log2(N/ksel) times, so the hot loop is the distance arithmetic plus one compare.
//   (2) re-rank in fp64: the candidates' distances are recomputed in double from the ORIGINAL fp32
//       inputs, ordered by (distance, index), and the first k are emitted (the result
//       does not depend on the fp32 selection arithmetic as long as the pool is a superset).
#include "kernels.h"

namespace lipfit {

constexpr int kKnnMargin = 8;
constexpr int kSelThreads = 128;
constexpr int kSelWarps = kSelThreads / 32;
constexpr int kMaxP = 2 * (LIPFIT_MAX_K + kKnnMargin);  // 272 pool entries per (chunk, query)

struct KnnArgs {
    const float* rec;
    const float* Xq;
    int2* pool;     // [nch][Qp][P]  (x = distance bits, y = datum index)
    int32_t* fill;  // [nch][Qp]     valid entries of each pool at kernel end
    int N, Q, Qp, d, ksel, P;
    int nqb, nch, chunk;
    Xform xf;
};

// Warp-cooperative compaction of one pool of n entries: keeps the ksel smallest (distance, index)
// in slots [0, ksel) in ascending order and returns the ksel-th smallest distance (the new tau).
// All 32 lanes must call it; `scr` is this warp's shared scratch of >= n + 1 entries.
__device__ __forceinline__ float knn_compact(int2* pool, int n, int ksel, int2* scr, int lane) {
    for (int c = lane; c < n; c += 32) scr[c] = pool[c];
    __syncwarp();
    for (int c = lane; c < n; c += 32) {
        const int2 e = scr[c];
        const float de = __int_as_float(e.x);
        int rank = 0;
        for (int o = 0; o < n; ++o) {
            const int2 f = scr[o];
            const float df = __int_as_float(f.x);
            rank += (df < de) || (df == de && f.y < e.y);
        }
        if (rank < ksel) pool[rank] = e;
        if (rank == ksel - 1) scr[kMaxP] = e;
    }
    __syncwarp();
    const float tau = __int_as_float(scr[kMaxP].x);
    __syncwarp();
    return tau;
}

template <int DP>
__host__ __device__ constexpr int knn_tile_records() {
    return DP <= 8 ? 512 : (DP <= 16 ? 256 : 128);
}

template <int NORM, int DP, bool ONESIDED, int R>
__global__ void __launch_bounds__(kSelThreads, 3)
knn_select_kernel(const KnnArgs a, const FreeFlags ff) {
    constexpr int THREADS = kSelThreads;
    constexpr int TILE = knn_tile_records<DP>();
    __shared__ __align__(128) float sbuf[2 * TILE * DP];
    __shared__ __align__(8) uint64_t bars[2];
    __shared__ int2 scratch[kSelWarps][kMaxP + 1];
    if (threadIdx.x == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    uint32_t phase = 0;
    const int lane = threadIdx.x & 31;
    int2* scr = scratch[threadIdx.x >> 5];
    const int P = a.P, ksel = a.ksel;

    const int ntiles = a.nqb * a.nch;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int qb = tile / a.nch;
        const int ch = tile - qb * a.nch;
        float q[R][DP];
        float tau[R];
        int fill[R];
        const int q0 = qb * R * THREADS + static_cast<int>(threadIdx.x);  // query of r: q0 + r*THREADS
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int qi = q0 + r * THREADS;
            const int qc = qi < a.Q ? qi : a.Q - 1;
            const float* src = a.Xq + static_cast<size_t>(qc) * a.d;
#pragma unroll
            for (int j = 0; j < DP; ++j)
                q[r][j] = (j < a.d) ? a.xf.sw[j] * __ldg(src + a.xf.perm[j]) : 0.f;
            // padding lanes (qi >= Q) never accept a candidate
            tau[r] = (qi < a.Q) ? __int_as_float(0x7f800000) : __int_as_float(0xff800000);
            fill[r] = 0;
        }
        int2* pool0 = a.pool + (static_cast<size_t>(ch) * a.Qp + q0) * P;  // pool of r: + r*THREADS*P

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
                bool hit = false;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    sv[r] = ONESIDED ? PairAccGeneric<NORM, DP>::run_u(q[r], x, ff)
                                     : PairAccU<NORM, DP, 0>::run(q[r], x);
                    hit |= (sv[r] < tau[r]);
                }
                if (__any_sync(0xffffffffu, hit)) {  // warp-uniform: rare after the first records
                    bool full = false;
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        if (sv[r] < tau[r]) {
                            pool0[static_cast<size_t>(r) * THREADS * P + fill[r]] =
                                make_int2(__float_as_int(sv[r]), base + j);
                            ++fill[r];
                            full |= (fill[r] == P);
                        }
                    }
                    if (__any_sync(0xffffffffu, full)) {
                        __syncwarp();  // orders the appends above before the cooperative reads below
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            unsigned m = __ballot_sync(0xffffffffu, fill[r] == P);
                            while (m) {
                                const int src = __ffs(m) - 1;
                                m &= m - 1;
                                int2* pq = a.pool + (static_cast<size_t>(ch) * a.Qp + q0 - lane + src +
                                                     static_cast<size_t>(r) * THREADS) * P;
                                const float nt = knn_compact(pq, P, ksel, scr, lane);
                                if (lane == src) {
                                    tau[r] = nt;
                                    fill[r] = ksel;
                                }
                            }
                        }
                    }
                }
            }
            rs.release(t);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int qi = q0 + r * THREADS;
            a.fill[static_cast<size_t>(ch) * a.Qp + qi] = fill[r];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// (2) fp64 re-rank.  One warp per query; candidates = the valid entries of its nch pools.
// ---------------------------------------------------------------------------------------------
struct RerankArgs {
    const float* X;
    const float* Xq;
    const int2* pool;
    const int32_t* fill;
    int32_t* idx;
    float* dist;
    int N, Q, Qp, d, P, nch, k, norm;
    Xform xf;  // perm/sw of the ORIGINAL coordinates; dU tells which packed coords are free
};

constexpr int kRerankWarps = 4;
constexpr int kMaxCand = 768;

__global__ void __launch_bounds__(kRerankWarps * 32)
knn_rerank_kernel(const RerankArgs a) {
    __shared__ double sd[kRerankWarps][kMaxCand];
    __shared__ int32_t si[kRerankWarps][kMaxCand];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int qi = blockIdx.x * kRerankWarps + warp;
    if (qi >= a.Q) return;
    const float* xq = a.Xq + static_cast<size_t>(qi) * a.d;
    int total = 0;
    for (int ch = 0; ch < a.nch; ++ch) {
        const int nf = a.fill[static_cast<size_t>(ch) * a.Qp + qi];
        const int2* pq = a.pool + (static_cast<size_t>(ch) * a.Qp + qi) * a.P;
        for (int c = lane; c < nf; c += 32) {
            const int32_t id = pq[c].y;
            const float* xk = a.X + static_cast<size_t>(id) * a.d;
            double acc = 0.0;
            for (int j = 0; j < a.d; ++j) {
                const int o = a.xf.perm[j];
                const double sw = static_cast<double>(a.xf.sw[j]);
                const double dlt = sw * (static_cast<double>(xq[o]) - static_cast<double>(xk[o]));
                const double comp = (j < a.xf.dU) ? fabs(dlt) : fmax(dlt, 0.0);
                if (a.norm == 1) acc += comp;
                else if (a.norm == 2) acc += comp * comp;
                else acc = fmax(acc, comp);
            }
            if (a.norm == 2) acc = sqrt(acc);
            sd[warp][total + c] = acc;
            si[warp][total + c] = id;
        }
        total += nf;
    }
    __syncwarp();
    for (int c = lane; c < total; c += 32) {
        const double dc = sd[warp][c];
        const int32_t ic = si[warp][c];
        int rank = 0;
        for (int o = 0; o < total; ++o) {
            const double d2 = sd[warp][o];
            const int32_t i2 = si[warp][o];
            rank += (d2 < dc) || (d2 == dc && i2 < ic);
        }
        if (rank < a.k) {
            a.idx[static_cast<size_t>(qi) * a.k + rank] = ic;
            a.dist[static_cast<size_t>(qi) * a.k + rank] = static_cast<float>(dc);
        }
    }
}

namespace {

int knn_dp(int d) { return d <= 4 ? 4 : (d <= 8 ? 8 : (d <= 16 ? 16 : 32)); }
constexpr int knn_r(int dp) { return dp <= 8 ? 8 : (dp <= 16 ? 4 : 2); }

template <int NORM, int DP, bool ONESIDED>
int launch_select(const Ctx& c, KnnArgs& a, const FreeFlags& ff, int slots_hint, bool query_only) {
    constexpr int R = knn_r(DP);
    auto kern = knn_select_kernel<NORM, DP, ONESIDED, R>;
    if (query_only) {  // occupancy query used by the host to size the decomposition
        int occ = 0;
        LIPFIT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, kSelThreads, 0));
        return occ < 1 ? 1 : occ;
    }
    long long ntiles = static_cast<long long>(a.nqb) * a.nch;
    int grid = static_cast<int>(ntiles < slots_hint ? ntiles : slots_hint);
    KernelTimer kt(TK_KNN_SELECT, c.stream);
    kern<<<grid, kSelThreads, 0, c.stream>>>(a, ff);
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

template <int NORM, bool ONESIDED>
int dispatch_dp(const Ctx& c, KnnArgs& a, const FreeFlags& ff, int dp, int slots, bool query_only) {
    switch (dp) {
        case 4: return launch_select<NORM, 4, ONESIDED>(c, a, ff, slots, query_only);
        case 8: return launch_select<NORM, 8, ONESIDED>(c, a, ff, slots, query_only);
        case 16: return launch_select<NORM, 16, ONESIDED>(c, a, ff, slots, query_only);
        default: return launch_select<NORM, 32, ONESIDED>(c, a, ff, slots, query_only);
    }
}

int dispatch(const Ctx& c, KnnArgs& a, const FreeFlags& ff, int norm, bool onesided, int dp, int slots,
             bool query_only) {
    if (norm == 1)
        return onesided ? dispatch_dp<1, true>(c, a, ff, dp, slots, query_only)
                        : dispatch_dp<1, false>(c, a, ff, dp, slots, query_only);
    if (norm == 2)
        return onesided ? dispatch_dp<2, true>(c, a, ff, dp, slots, query_only)
                        : dispatch_dp<2, false>(c, a, ff, dp, slots, query_only);
    return onesided ? dispatch_dp<3, true>(c, a, ff, dp, slots, query_only)
                    : dispatch_dp<3, false>(c, a, ff, dp, slots, query_only);
}

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
    a.P = 2 * a.ksel;
    const int qper = kSelThreads * knn_r(dp);
    a.nqb = (a.Q + qper - 1) / qper;
    a.Qp = a.nqb * qper;
    FreeFlags ff = make_free_flags(xf);
    const bool onesided = xf.dC > 0;
    const int occ = dispatch(c, a, ff, norm, onesided, dp, 0, true);
    if (occ < 0) return occ;
    const int slots = c.num_sms * occ;

    // Data chunks: the fewest (<= 8, pools must fit the re-rank) that keep the last wave of the
    // persistent grid >= 94 % full; every chunk keeps its own pools, merged by the re-rank.
    const int tile = dp <= 8 ? 512 : (dp <= 16 ? 256 : 128);
    int max_ch = kMaxCand / a.P;
    if (max_ch > 8) max_ch = 8;
    int by_n = a.N / (8 * a.P);
    if (max_ch > by_n) max_ch = by_n;
    if (max_ch < 1) max_ch = 1;
    int best = 1;
    double best_eff = 0.0;
    for (int nch = 1; nch <= max_ch; ++nch) {
        long long tiles = static_cast<long long>(a.nqb) * nch;
        long long waves = (tiles + slots - 1) / slots;
        double eff = static_cast<double>(tiles) / static_cast<double>(waves * slots);
        if (eff > best_eff + 1e-9) {
            best_eff = eff;
            best = nch;
        }
        if (eff >= 0.94) break;
    }
    int nch = best;
    int chunk = (a.N + nch - 1) / nch;
    chunk = ((chunk + tile - 1) / tile) * tile;
    nch = (a.N + chunk - 1) / chunk;
    a.nch = nch;
    a.chunk = chunk;

    Workspace wp, wf;
    int rc = wp.alloc(sizeof(int2) * static_cast<size_t>(nch) * a.Qp * a.P, c.stream);
    if (rc) return rc;
    rc = wf.alloc(sizeof(int32_t) * static_cast<size_t>(nch) * a.Qp, c.stream);
    if (rc) return rc;
    a.pool = wp.as<int2>();
    a.fill = wf.as<int32_t>();
    rc = dispatch(c, a, ff, norm, onesided, dp, slots, false);
    if (rc) return rc;

    RerankArgs r{};
    r.X = X;
    r.Xq = Xq;
    r.pool = a.pool;
    r.fill = a.fill;
    r.idx = idx;
    r.dist = dist;
    r.N = a.N;
    r.Q = a.Q;
    r.Qp = a.Qp;
    r.d = a.d;
    r.P = a.P;
    r.nch = nch;
    r.k = k;
    r.norm = norm;
    r.xf = xf;
    knn_rerank_kernel<<<(a.Q + kRerankWarps - 1) / kRerankWarps, kRerankWarps * 32, 0, c.stream>>>(r);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

}  // namespace lipfit
