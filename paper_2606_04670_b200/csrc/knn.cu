// knn.cu -- step a3: fused distance + per-query top-k.
// Neighbours by distance d_(1) <= d_(2) <= ... without the cdist matrix + topk of
// PAPER.md:206.  Device passes:
//   (0) pack: records [x'_0..x'_{DP-1}, ||x'||^2, 0,0,0] (x' = weighted / mirrored coordinates) and two
//       data statistics (max |x'_j|, max ||x'||^2) that the error bounds of pass (2) need.
//   (1) selection in fp32.  Every thread keeps R queries in registers and streams packed records
//       through shared memory (TMA bulk copies), exactly like the bounds kernel.  Per query it holds a
//       threshold tau and a fill count in registers; a pair whose selection key is below tau is
//       APPENDED (one 8-byte fire-and-forget store) to the query's candidate pool of P = 2*ksel
//       entries, ksel = k + margin, in an L2-resident workspace.  When a pool is full the whole warp
//       compacts it (rank by counting in shared memory), keeps the ksel best in sorted order and
//       lowers tau to the ksel-th best.  tau only decreases, so every datum that is NOT in the pool
//       has key >= tau_final, for ANY data order; a pool is compacted about log2(N/ksel) times, so
//       the hot loop is the key arithmetic plus one compare.  Two key flavours:
//         * dot  (symmetric L2): key = ||x'||^2 - 2 q'.x'  (= d^2 - ||q'||^2): d FFMA per pair;
//         * diff (everything else): key = the accumulated |.| / (.)_+ distance (squared for L2).
//   (2) re-rank in fp64: the candidates' distances are recomputed in double from the ORIGINAL fp32
//       inputs, ordered by (distance, index), and the first k are emitted -- IF the certificate holds:
//       exact k-th candidate distance < min_chunks(tau_final) - E, E a rigorous bound of the fp32 key
//       error.  Then no datum outside the pools can belong to the answer.
//   (3) exact fallback for the (rare) queries whose certificate fails (ties beyond the margin,
//       adversarial inputs): one CTA per such query scans all data in fp64.
// The result therefore never depends on the fp32 selection arithmetic.
#include "kernels.h"
#include "knn_common.cuh"

#include <cstring>

namespace lipfit {

#ifndef LIPFIT_KNN_NREC
#define LIPFIT_KNN_NREC 2  // records consumed per loop iteration
#endif
#ifndef LIPFIT_KNN_MINB
#define LIPFIT_KNN_MINB 3  // resident CTAs per SM the selection kernel is compiled for
#endif
// ---------------------------------------------------------------------------------------------
// (0) pack
// ---------------------------------------------------------------------------------------------
// stats[0] = bits of max_k max_j |x'_kj|, stats[1] = bits of max_k fl(||x'_k||^2)  (non-negative
// floats order like their bit patterns).
__global__ void __launch_bounds__(256)
knn_pack_kernel(const float* __restrict__ X, int N, Xform xf, int rf, int x2slot,
                float* __restrict__ rec, uint32_t* __restrict__ stats) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    float amax = 0.f, x2 = 0.f;
    if (k < N) {
        const float* src = X + static_cast<size_t>(k) * xf.d;
        float* dst = rec + static_cast<size_t>(k) * rf;
        double s2 = 0.0;
        for (int j0 = 0; j0 < rf; j0 += 4) {
            float t[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                int j = j0 + c;
                t[c] = (j < xf.d) ? xf.sw[j] * src[xf.perm[j]] : 0.f;
                amax = fmaxf(amax, fabsf(t[c]));
                s2 += static_cast<double>(t[c]) * static_cast<double>(t[c]);
            }
            if (j0 + 4 <= x2slot || x2slot < 0)
                *reinterpret_cast<float4*>(dst + j0) = make_float4(t[0], t[1], t[2], t[3]);
            else {  // the float4 holding the ||x'||^2 slot: s2 is complete (all coordinates are before it)
                x2 = static_cast<float>(s2);
                t[x2slot - j0] = x2;
                *reinterpret_cast<float4*>(dst + j0) = make_float4(t[0], t[1], t[2], t[3]);
            }
        }
        if (x2slot < 0) x2 = static_cast<float>(s2);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
        x2 = fmaxf(x2, __shfl_xor_sync(0xffffffffu, x2, o));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMax(stats + 0, __float_as_uint(amax));
        atomicMax(stats + 1, __float_as_uint(x2));
    }
}

// ---------------------------------------------------------------------------------------------
// (1) selection
// ---------------------------------------------------------------------------------------------
// Slow path of the selection loop, entered warp-uniformly when some lane has a key below its
// threshold: append (NREC records at once), and compact the pools that are (nearly) full.  A pool
// is compacted as soon as fewer than NREC free entries are left, so NREC appends always fit.
template <int R, int NREC>
__device__ __forceinline__ void knn_hit(const KnnArgs& a, const float (&sv)[NREC][R], float (&tau)[R],
                                        int (&fill)[R], int2* pool0, int index, int2* scr, int lane) {
    const int P = a.P;
    bool full = false;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        int2* pr = pool0 + static_cast<size_t>(r) * kSelThreads * P;
#pragma unroll
        for (int e = 0; e < NREC; ++e) {
            if (sv[e][r] < tau[r]) {
                pr[fill[r]] = make_int2(__float_as_int(sv[e][r]), index + e);
                ++fill[r];
            }
        }
        full |= (fill[r] > P - NREC);
    }
    if (__any_sync(0xffffffffu, full)) {
        __syncwarp();  // orders the appends above before the cooperative reads below
#pragma unroll
        for (int r = 0; r < R; ++r) {
            unsigned m = __ballot_sync(0xffffffffu, fill[r] > P - NREC);
            while (m) {
                const int src = __ffs(m) - 1;
                m &= m - 1;
                // pool0 is this lane's pool of r = 0; lane `src`'s pool of query r is a fixed offset away
                int2* pq = pool0 + (static_cast<ptrdiff_t>(src - lane) +
                                    static_cast<ptrdiff_t>(r) * kSelThreads) * P;
                const int n = __shfl_sync(0xffffffffu, fill[r], src);
                const float nt = knn_compact(pq, n, a.ksel, scr, lane);
                if (lane == src) {
                    tau[r] = nt;
                    fill[r] = a.ksel;
                }
            }
        }
    }
}

constexpr int kKnnStages = 4;
template <int RF>
__host__ __device__ constexpr int knn_tile_records() {
    return RF <= 8 ? 256 : (RF <= 20 ? 128 : 64);
}

template <int RF>
__device__ __forceinline__ void knn_load_record(const float* s, float* x) {
#pragma unroll
    for (int c = 0; c < RF / 4; ++c) {
        float4 v = reinterpret_cast<const float4*>(s)[c];
        x[4 * c + 0] = v.x;
        x[4 * c + 1] = v.y;
        x[4 * c + 2] = v.z;
        x[4 * c + 3] = v.w;
    }
}

// Key policies.  load_q() turns the caller's query into the registers the key needs.
template <int NORM, int DP, bool ONESIDED>
struct DiffKey {
    static constexpr int RF = DP + 4;  // only the DP coordinates are read; the stride is shared with DotKey
    static constexpr int NLOAD = DP;
    static __device__ __forceinline__ float qscale() { return 1.f; }
    static __device__ __forceinline__ float key(const float* q, const float* x, const FreeFlags& ff) {
        return ONESIDED ? PairAccGeneric<NORM, DP>::run_u(q, x, ff) : PairAccU<NORM, DP, 0>::run(q, x);
    }
};
template <int DP>
struct DotKey {
    static constexpr int RF = DP + 4;
    static constexpr int NLOAD = DP + 4;
    static __device__ __forceinline__ float qscale() { return -2.f; }
    // 2 coordinates per FFMA2 (packed fp32, sm_100): half the issue slots of DP scalar FFMAs.
    static __device__ __forceinline__ float key(const float* q, const float* x, const FreeFlags&) {
        float2 s = make_float2(x[DP], 0.f);  // ||x'||^2
#pragma unroll
        for (int j = 0; j < DP; j += 2)
            s = __ffma2_rn(make_float2(q[j], q[j + 1]), make_float2(x[j], x[j + 1]), s);
        return s.x + s.y;
    }
};

template <class Key, int DP, int R, int NREC, int MINB>
__global__ void __launch_bounds__(kSelThreads, MINB)
knn_select_kernel(const KnnArgs a, const FreeFlags ff) {
    constexpr int THREADS = kSelThreads;
    constexpr int RF = Key::RF;
    constexpr int NL = Key::NLOAD;
    constexpr int TILE = knn_tile_records<RF>();
    constexpr int ST = kKnnStages;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* sbuf = reinterpret_cast<float*>(smem_raw);                                    // ST*TILE*RF floats
    int2* scratch = reinterpret_cast<int2*>(smem_raw + sizeof(float) * ST * TILE * RF);  // [warps][kMaxP+1]
    __shared__ __align__(8) uint64_t bars[ST];
    __shared__ int done[ST];
    if (threadIdx.x == 0) {
#pragma unroll
        for (int b = 0; b < ST; ++b) {
            mbar_init(&bars[b], 1);
            done[b] = 0;
        }
        mbar_fence_init();
    }
    __syncthreads();
    uint32_t phase = 0;
    const int lane = threadIdx.x & 31;
    int2* scr = scratch + (threadIdx.x >> 5) * (kMaxP + 1);
    const int P = a.P;
    const float qs = Key::qscale();

    const int ntiles = a.nfull + a.ntail * a.T;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        int qb, ch, begin, end;
        if (tile < a.nfull) {
            qb = tile;
            ch = 0;
            begin = 0;
            end = a.N;
        } else {
            const int t = tile - a.nfull;
            qb = a.nfull + t / a.T;
            ch = t - (qb - a.nfull) * a.T;
            begin = ch * a.chunk;
            end = min(a.N, begin + a.chunk);
        }
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
                q[r][j] = (j < a.d) ? qs * (a.xf.sw[j] * __ldg(src + a.xf.perm[j])) : 0.f;
            // padding lanes (qi >= Q) never accept a candidate
            tau[r] = (qi < a.Q) ? __int_as_float(0x7f800000) : __int_as_float(0xff800000);
            fill[r] = 0;
        }
        const size_t slot0 = knn_pool_slot(q0, ch, a.Qp, a.Qtp, a.nfullq);  // slot of r: + r*THREADS
        int2* pool0 = a.pool + slot0 * P;                                   // pool of r: + r*THREADS*P

        RecordPipe<TILE, ST, kSelWarps> rs(a.rec, RF, begin, end, sbuf, bars, done, &phase);
        for (int t = 0; t < rs.ntiles; ++t) {
            const float* s = rs.acquire(t);
            const int n = rs.count(t);
            const int base = begin + t * TILE;
            int j = 0;
            for (; j + NREC <= n; j += NREC) {
                float x[NREC][NL];
                float sv[NREC][R];
#pragma unroll
                for (int e = 0; e < NREC; ++e) knn_load_record<NL>(s + (j + e) * RF, x[e]);
                bool hit = false;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    float m = __int_as_float(0x7f800000);
#pragma unroll
                    for (int e = 0; e < NREC; ++e) {
                        sv[e][r] = Key::key(q[r], x[e], ff);
                        m = fminf(m, sv[e][r]);
                    }
                    hit |= (m < tau[r]);
                }
                if (__any_sync(0xffffffffu, hit)) {  // warp-uniform: rare after the first records
#pragma unroll
                    for (int e = 0; e < NREC; ++e) {  // one record at a time: measured faster than merged
                        float s1[1][R];
#pragma unroll
                        for (int r = 0; r < R; ++r) s1[0][r] = sv[e][r];
                        knn_hit<R, 1>(a, s1, tau, fill, pool0, base + j + e, scr, lane);
                    }
                }
            }
            for (; j < n; ++j) {  // ragged end of the tile
                float x[1][NL];
                float sv[1][R];
                knn_load_record<NL>(s + j * RF, x[0]);
                bool hit = false;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    sv[0][r] = Key::key(q[r], x[0], ff);
                    hit |= (sv[0][r] < tau[r]);
                }
                if (__any_sync(0xffffffffu, hit))
                    knn_hit<R, 1>(a, sv, tau, fill, pool0, base + j, scr, lane);
            }
            rs.release(t);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            a.fill[slot0 + static_cast<size_t>(r) * THREADS] = fill[r];
            a.tau[slot0 + static_cast<size_t>(r) * THREADS] = tau[r];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// (2) fp64 re-rank + certificate.  One warp per query; candidates = the valid entries of its pools.
// ---------------------------------------------------------------------------------------------
struct RerankArgs {
    const float* X;
    const float* Xq;
    const int2* pool;
    const int32_t* fill;
    const float* tau;
    const uint32_t* stats;  // [0] max |x'|, [1] max ||x'||^2, [2] flagged count, [4] max observed key error / E
    const float* mu;        // tensor-core path: centre of the coordinates
    int32_t* idx;
    float* dist;
    int32_t* flagged;   // [Q] queries whose certificate failed
    double* flagged_T;  // [Q] their exact k-th candidate key (an upper bound of the true one)
    int32_t* nflagged;
    int N, Q, Qp, Qtp, nfullq, T, d, P, k, norm, dot;
    Xform xf;  // perm/sw of the ORIGINAL coordinates; dU tells which packed coords are free
};

// Exact key of (query, datum) in fp64 from the original fp32 inputs: squared distance for L2, the
// distance itself for L1 / Linf.
__device__ __forceinline__ double knn_exact_key(const float* xq, const float* xk, const Xform& xf,
                                                int norm) {
    double acc = 0.0;
    for (int j = 0; j < xf.d; ++j) {
        const int o = xf.perm[j];
        const double sw = static_cast<double>(xf.sw[j]);
        const double dlt = sw * (static_cast<double>(xq[o]) - static_cast<double>(xk[o]));
        const double comp = (j < xf.dU) ? fabs(dlt) : fmax(dlt, 0.0);
        if (norm == 1) acc += comp;
        else if (norm == 2) acc += comp * comp;
        else acc = fmax(acc, comp);
    }
    return acc;
}

// Bound E of |fp32 selection key - exact key| for one query, any datum, and the
// shift that maps selection keys to exact keys (exact = key + shift for the dot flavour).
//   a   = max_j |x'_j| over the data + max_j |q'_j|        (coordinate scale)
//   dot : E = (d + 8) u (sqrt(max ||x'||^2) + ||q'||)^2
//   diff: L1  E = u a (4 d + 2 d^2),  Linf  E = 4 u a,  L2 (squared)  E = u a^2 (20 d + 4 d^2)
// u = 2^-24; every formula is then doubled as slack for the fp32-rounded statistics themselves.
//   tc  : key from the bf16-split GEMM on coordinates centred at mu (knn_tc.cu); qn = ||q_c||,
//         xn = sqrt(max ||x_c||^2):  E = 10.5 2^-16 qn xn          (1.5 x the split residue 7 2^-16 qn xn)
//                                      + 2^-17 (6 qn xn + xn^2)    (fp32 accumulation of <= 64 terms)
//                                      + 4 (qn + xn) sqrt(d) 2^-23 (amax + qinf + qn + xn)   (centring in fp32)
__device__ __forceinline__ void knn_error_bound(const float* xq, const Xform& xf, int norm, int dot,
                                                const uint32_t* stats, const float* mu, double* E,
                                                double* shift) {
    const double u = 5.9604644775390625e-08;
    const double amax = static_cast<double>(__uint_as_float(stats[0]));
    const double x2max = static_cast<double>(__uint_as_float(stats[1]));
    if (dot == 2) {
        double qinf = 0.0, qc2 = 0.0;
        for (int j = 0; j < xf.d; ++j) {
            const double v = static_cast<double>(xf.sw[j]) * static_cast<double>(xq[xf.perm[j]]);
            const double vc = v - static_cast<double>(mu[j]);
            qinf = fmax(qinf, fabs(v));
            qc2 += vc * vc;
        }
        const double qn = sqrt(qc2), xn = sqrt(x2max);
        *E = 10.5 * 1.52587890625e-05 * qn * xn + 7.62939453125e-06 * (6.0 * qn * xn + x2max) +
             4.0 * (qn + xn) * sqrt(static_cast<double>(xf.d)) * 2.0 * u * (amax + qinf + qn + xn);
        *shift = qc2;
        return;
    }
    double qinf = 0.0, q2 = 0.0;
    for (int j = 0; j < xf.d; ++j) {
        const double v = fabs(static_cast<double>(xf.sw[j]) * static_cast<double>(xq[xf.perm[j]]));
        qinf = fmax(qinf, v);
        q2 += v * v;
    }
    const double d = static_cast<double>(xf.d);
    if (dot) {
        const double b = sqrt(x2max) + sqrt(q2);
        *E = 2.0 * (d + 8.0) * u * b * b;
        *shift = q2;
    } else {
        const double a = amax + qinf;
        if (norm == 1) *E = 2.0 * u * a * (4.0 * d + 2.0 * d * d);
        else if (norm == 2) *E = 2.0 * u * a * a * (20.0 * d + 4.0 * d * d);
        else *E = 8.0 * u * a;
        *shift = 0.0;
    }
}

constexpr int kRerankWarps = 4;
constexpr int kMaxCand = 768;

__global__ void __launch_bounds__(kRerankWarps * 32)
knn_rerank_kernel(const RerankArgs a) {
    __shared__ double sd[kRerankWarps][kMaxCand];
    __shared__ int32_t si[kRerankWarps][kMaxCand];
    __shared__ double skth[kRerankWarps];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int qi = blockIdx.x * kRerankWarps + warp;
    if (qi >= a.Q) return;
    const float* xq = a.Xq + static_cast<size_t>(qi) * a.d;
    int total = 0;
    float tmin = __int_as_float(0x7f800000);
    // certificate: every datum outside the pools has exact key >= tmin + shift - E
    double E, shift, worst = 0.0;
    knn_error_bound(xq, a.xf, a.norm, a.dot, a.stats, a.mu, &E, &shift);
    const int nch = qi >= a.nfullq ? a.T : 1;
    for (int ch = 0; ch < nch; ++ch) {
        const size_t slot = knn_pool_slot(qi, ch, a.Qp, a.Qtp, a.nfullq);
        const int nf = a.fill[slot];
        tmin = fminf(tmin, a.tau[slot]);
        const int2* pq = a.pool + slot * a.P;
        for (int c = lane; c < nf; c += 32) {
            const int2 e = pq[c];
            const double ex = knn_exact_key(xq, a.X + static_cast<size_t>(e.y) * a.d, a.xf, a.norm);
            sd[warp][total + c] = ex;
            si[warp][total + c] = e.y;
            worst = fmax(worst, fabs(static_cast<double>(__int_as_float(e.x)) + shift - ex));
        }
        total += nf;
    }
    __syncwarp();
    // diagnostic (lipfit_knn_key_error_ratio): largest observed |selection key - exact key| over E
    {
        float ratio = E > 0.0 ? static_cast<float>(worst / E) : 0.f;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) ratio = fmaxf(ratio, __shfl_xor_sync(0xffffffffu, ratio, o));
        if (lane == 0 && ratio > 0.f) atomicMax(const_cast<uint32_t*>(a.stats) + 4, __float_as_uint(ratio));
    }
    const bool all_in = !(tmin < __int_as_float(0x7f800000));  // no pool was ever compacted
    const double lb = static_cast<double>(tmin) + shift - E;
    int myrank[kMaxCand / 32];
#pragma unroll
    for (int s = 0; s < kMaxCand / 32; ++s) {
        const int c = lane + 32 * s;
        int rank = 0x7fffffff;
        if (c < total) {
            const double dc = sd[warp][c];
            const int32_t ic = si[warp][c];
            rank = 0;
            for (int o = 0; o < total; ++o) {
                const double d2 = sd[warp][o];
                const int32_t i2 = si[warp][o];
                rank += (d2 < dc) || (d2 == dc && i2 < ic);
            }
            if (rank == a.k - 1) skth[warp] = dc;
        }
        myrank[s] = rank;
    }
    __syncwarp();
    // fewer than k candidates cannot happen by construction (seeded thresholds keep >= ksel data below
    // them); if it ever did, the query goes to the exact fallback with an unbounded candidate set
    const double kth = total >= a.k ? skth[warp] : static_cast<double>(__int_as_float(0x7f800000));
    if (all_in || kth < lb) {
#pragma unroll
        for (int s = 0; s < kMaxCand / 32; ++s) {
            const int c = lane + 32 * s;
            if (c < total && myrank[s] < a.k) {
                const double dc = sd[warp][c];
                a.idx[static_cast<size_t>(qi) * a.k + myrank[s]] = si[warp][c];
                a.dist[static_cast<size_t>(qi) * a.k + myrank[s]] =
                    static_cast<float>(a.norm == 2 ? sqrt(dc) : dc);
            }
        }
    } else if (lane == 0) {
        const int slot = atomicAdd(a.nflagged, 1);
        a.flagged[slot] = qi;
        a.flagged_T[slot] = kth;
    }
}

// ---------------------------------------------------------------------------------------------
// (3) exact fallback: one CTA per flagged query, everything in fp64 from the original inputs.
// T = exact key of the k-th pool candidate >= the true k-th key, so the answer lies in
// C = {datum : key <= T}.  |C| <= kMaxCand: rank C by (key, index).  Otherwise (massive ties):
// k rounds of "next smallest (key, index) after the previous one" -- slow, correct, deterministic.
// ---------------------------------------------------------------------------------------------
constexpr int kExactThreads = 256;

__global__ void __launch_bounds__(kExactThreads)
knn_exact_kernel(const RerankArgs a) {
    __shared__ double sd[kMaxCand];
    __shared__ int32_t si[kMaxCand];
    __shared__ int scount;
    __shared__ double rk[kExactThreads / 32];
    __shared__ int32_t ri[kExactThreads / 32];
    const int nfl = *a.nflagged;
    for (int slot = blockIdx.x; slot < nfl; slot += gridDim.x) {
        const int qi = a.flagged[slot];
        const double T = a.flagged_T[slot];
        const float* xq = a.Xq + static_cast<size_t>(qi) * a.d;
        if (threadIdx.x == 0) scount = 0;
        __syncthreads();
        for (int k = threadIdx.x; k < a.N; k += kExactThreads) {
            const double key = knn_exact_key(xq, a.X + static_cast<size_t>(k) * a.d, a.xf, a.norm);
            if (key <= T) {
                const int c = atomicAdd(&scount, 1);
                if (c < kMaxCand) {
                    sd[c] = key;
                    si[c] = k;
                }
            }
        }
        __syncthreads();
        const int total = scount;
        if (total <= kMaxCand) {
            for (int c = threadIdx.x; c < total; c += kExactThreads) {
                const double dc = sd[c];
                const int32_t ic = si[c];
                int rank = 0;
                for (int o = 0; o < total; ++o) rank += (sd[o] < dc) || (sd[o] == dc && si[o] < ic);
                if (rank < a.k) {
                    a.idx[static_cast<size_t>(qi) * a.k + rank] = ic;
                    a.dist[static_cast<size_t>(qi) * a.k + rank] =
                        static_cast<float>(a.norm == 2 ? sqrt(dc) : dc);
                }
            }
        } else {
            double pk = -1.0;  // keys are >= 0
            int32_t pi = -1;
            for (int r = 0; r < a.k; ++r) {
                double bk = __longlong_as_double(0x7ff0000000000000LL);
                int32_t bi = 0x7fffffff;
                for (int k = threadIdx.x; k < a.N; k += kExactThreads) {
                    const double key = knn_exact_key(xq, a.X + static_cast<size_t>(k) * a.d, a.xf, a.norm);
                    const bool after = (key > pk) || (key == pk && k > pi);
                    const bool better = (key < bk) || (key == bk && k < bi);
                    if (after && better) {
                        bk = key;
                        bi = k;
                    }
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    const double ok = __shfl_xor_sync(0xffffffffu, bk, o);
                    const int32_t oi = __shfl_xor_sync(0xffffffffu, bi, o);
                    if (ok < bk || (ok == bk && oi < bi)) {
                        bk = ok;
                        bi = oi;
                    }
                }
                if ((threadIdx.x & 31) == 0) {
                    rk[threadIdx.x >> 5] = bk;
                    ri[threadIdx.x >> 5] = bi;
                }
                __syncthreads();
                bk = rk[0];
                bi = ri[0];
                for (int w = 1; w < kExactThreads / 32; ++w)
                    if (rk[w] < bk || (rk[w] == bk && ri[w] < bi)) {
                        bk = rk[w];
                        bi = ri[w];
                    }
                __syncthreads();
                if (threadIdx.x == 0) {
                    a.idx[static_cast<size_t>(qi) * a.k + r] = bi;
                    a.dist[static_cast<size_t>(qi) * a.k + r] =
                        static_cast<float>(a.norm == 2 ? sqrt(bk) : bk);
                }
                pk = bk;
                pi = bi;
            }
        }
        __syncthreads();
    }
}

namespace {

int knn_dp(int d) { return d <= 4 ? 4 : (d <= 8 ? 8 : (d <= 16 ? 16 : 32)); }
constexpr int knn_r(int dp) { return dp <= 8 ? 8 : (dp <= 16 ? 4 : 2); }

template <int RF>
constexpr size_t knn_smem_bytes() {
    return sizeof(float) * kKnnStages * knn_tile_records<RF>() * RF +
           sizeof(int2) * kSelWarps * (kMaxP + 1);
}

template <class Key, int DP>
int launch_select(const Ctx& c, KnnArgs& a, const FreeFlags& ff, int slots_hint, bool query_only) {
    constexpr int R = knn_r(DP);
    constexpr int NREC = LIPFIT_KNN_NREC;
    constexpr int MINB = DP <= 16 ? LIPFIT_KNN_MINB : 2;
    auto kern = knn_select_kernel<Key, DP, R, NREC, MINB>;
    constexpr size_t smem = knn_smem_bytes<Key::RF>();
    LIPFIT_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     static_cast<int>(smem)));
    if (query_only) {  // occupancy query used by the host to size the decomposition
        int occ = 0;
        LIPFIT_CUDA(occupancy_of(&occ, kern, kSelThreads, smem));
        return occ < 1 ? 1 : occ;
    }
    long long ntiles = static_cast<long long>(a.nfull) + static_cast<long long>(a.ntail) * a.T;
    int grid = static_cast<int>(ntiles < slots_hint ? ntiles : slots_hint);
    KernelTimer kt(TK_KNN_SELECT, c.stream);
    kern<<<grid, kSelThreads, smem, c.stream>>>(a, ff);
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

template <int NORM, bool ONESIDED>
int dispatch_dp(const Ctx& c, KnnArgs& a, const FreeFlags& ff, int dp, int slots, bool query_only) {
    switch (dp) {
        case 4: return launch_select<DiffKey<NORM, 4, ONESIDED>, 4>(c, a, ff, slots, query_only);
        case 8: return launch_select<DiffKey<NORM, 8, ONESIDED>, 8>(c, a, ff, slots, query_only);
        case 16: return launch_select<DiffKey<NORM, 16, ONESIDED>, 16>(c, a, ff, slots, query_only);
        default: return launch_select<DiffKey<NORM, 32, ONESIDED>, 32>(c, a, ff, slots, query_only);
    }
}

int dispatch_dot(const Ctx& c, KnnArgs& a, const FreeFlags& ff, int dp, int slots, bool query_only) {
    switch (dp) {
        case 4: return launch_select<DotKey<4>, 4>(c, a, ff, slots, query_only);
        case 8: return launch_select<DotKey<8>, 8>(c, a, ff, slots, query_only);
        case 16: return launch_select<DotKey<16>, 16>(c, a, ff, slots, query_only);
        default: return launch_select<DotKey<32>, 32>(c, a, ff, slots, query_only);
    }
}

int dispatch(const Ctx& c, KnnArgs& a, const FreeFlags& ff, int norm, bool onesided, bool dot, int dp,
             int slots, bool query_only) {
    if (dot) return dispatch_dot(c, a, ff, dp, slots, query_only);
    if (norm == 1)
        return onesided ? dispatch_dp<1, true>(c, a, ff, dp, slots, query_only)
                        : dispatch_dp<1, false>(c, a, ff, dp, slots, query_only);
    if (norm == 2)
        return onesided ? dispatch_dp<2, true>(c, a, ff, dp, slots, query_only)
                        : dispatch_dp<2, false>(c, a, ff, dp, slots, query_only);
    return onesided ? dispatch_dp<3, true>(c, a, ff, dp, slots, query_only)
                    : dispatch_dp<3, false>(c, a, ff, dp, slots, query_only);
}

bool use_tc(const Xform& xf, int norm, bool allow_tc) {
    return allow_tc && norm == 2 && xf.dC == 0 && xf.d <= 16;
}

}  // namespace

const char* knn_variant_name(const Xform& xf, int norm, bool allow_tc) {
    if (use_tc(xf, norm, allow_tc)) {  // K = 16 bf16 per K step, ceil((3 d + 3) / 16) steps (knn_tc.cu)
        static const char* const names[4] = {"knn_tc_select<bf16x3,K16>", "knn_tc_select<bf16x3,K32>",
                                             "knn_tc_select<bf16x3,K48>", "knn_tc_select<bf16x3,K64>"};
        return names[(3 * xf.d + 3 + 15) / 16 - 1];
    }
    return (norm == 2 && xf.dC == 0) ? "knn_select<dot>" : "knn_select<diff>";
}

int launch_knn(const Ctx& c, const float* X, int64_t N, const float* Xq, int64_t Q, const Xform& xf,
               int norm, int k, int32_t* idx, float* dist, bool allow_tc, lipfit_knn_info* info) {
    KnnArgs a{};
    const int dp = knn_dp(xf.d);
    const int rf = dp + 4;
    const bool onesided = xf.dC > 0;
    const bool dot = (norm == 2) && !onesided;  // symmetric L2: cross-term key
    a.Xq = Xq;
    a.N = static_cast<int>(N);
    a.Q = static_cast<int>(Q);
    a.d = xf.d;
    a.xf = xf;
    a.ksel = static_cast<int>(N < k + kKnnMargin ? N : k + kKnnMargin);
    a.P = 2 * a.ksel;
    const bool tc = use_tc(xf, norm, allow_tc);  // tensor-core selection (knn_tc.cu)
    if (tc) a.P = a.ksel + kTcPoolExtra;
    const int qper = tc ? kTcQueries : kSelThreads * knn_r(dp);
    a.nqb = (a.Q + qper - 1) / qper;
    a.Qp = a.nqb * qper;
    FreeFlags ff = make_free_flags(xf);
    int slots = knn_tc_slots(c);
    if (!tc) {
        const int occ = dispatch(c, a, ff, norm, onesided, dot, dp, 0, true);
        if (occ < 0) return occ;
        slots = c.num_sms * occ;
    }

    // Schedule (KnnArgs): whole waves of query blocks sweep the data unsplit; the blocks of the last,
    // partial wave are cut into T <= 8 data chunks (pools must fit the re-rank) to keep it full.
    const int tile = tc ? kTcBN : (rf <= 8 ? 256 : (rf <= 20 ? 128 : 64));
    int maxT = kMaxCand / a.P;
    if (maxT > 8) maxT = 8;
    const int by_n = a.N / (8 * a.P);
    if (maxT > by_n) maxT = by_n;
    if (maxT < 1) maxT = 1;
    a.nfull = (a.nqb / slots) * slots;
    a.ntail = a.nqb - a.nfull;
    int T = a.ntail > 0 ? slots / a.ntail : 1;
    if (T > maxT) T = maxT;
    if (T < 1) T = 1;
    int chunk = (a.N + T - 1) / T;
    chunk = ((chunk + tile - 1) / tile) * tile;
    T = (a.N + chunk - 1) / chunk;
    a.T = T;
    a.chunk = chunk;
    a.nfullq = a.nfull * qper;
    a.Qtp = a.ntail * qper;

    // workspace: records | stats + flagged counter | pools | fill | tau | flagged list
    const size_t nq = static_cast<size_t>(a.Qp) + static_cast<size_t>(T - 1) * a.Qtp;
    Workspace wrec, wp, wf, wt, wfl, wflT, wst, wmu;
    int rc;
    if ((rc = wrec.alloc(tc ? 16 : sizeof(float) * static_cast<size_t>(N) * rf, c.stream))) return rc;
    if ((rc = wst.alloc(sizeof(uint32_t) * 8, c.stream))) return rc;
    if ((rc = wmu.alloc(sizeof(float) * kMaxDim, c.stream))) return rc;
    if ((rc = wp.alloc(sizeof(int2) * nq * a.P, c.stream))) return rc;
    if ((rc = wf.alloc(sizeof(int32_t) * nq, c.stream))) return rc;
    if ((rc = wt.alloc(sizeof(float) * nq, c.stream))) return rc;
    if ((rc = wfl.alloc(sizeof(int32_t) * static_cast<size_t>(a.Q), c.stream))) return rc;
    if ((rc = wflT.alloc(sizeof(double) * static_cast<size_t>(a.Q), c.stream))) return rc;
    LIPFIT_CUDA(cudaMemsetAsync(wst.p, 0, sizeof(uint32_t) * 8, c.stream));
    uint32_t* stats = wst.as<uint32_t>();
    a.rec = wrec.as<float>();
    a.pool = wp.as<int2>();
    a.fill = wf.as<int32_t>();
    a.tau = wt.as<float>();
    if (tc) {
        rc = launch_knn_tc_select(c, X, Xq, a, wmu.as<float>(), stats);
    } else {
        knn_pack_kernel<<<(a.N + 255) / 256, 256, 0, c.stream>>>(X, a.N, xf, rf, dp, wrec.as<float>(), stats);
        ++g_launches;
        LIPFIT_CUDA(cudaGetLastError());
        rc = dispatch(c, a, ff, norm, onesided, dot, dp, slots, false);
    }
    if (rc) return rc;

    RerankArgs r{};
    r.X = X;
    r.Xq = Xq;
    r.pool = a.pool;
    r.fill = a.fill;
    r.tau = a.tau;
    r.stats = stats;
    r.mu = wmu.as<float>();
    r.idx = idx;
    r.dist = dist;
    r.flagged = wfl.as<int32_t>();
    r.flagged_T = wflT.as<double>();
    r.nflagged = reinterpret_cast<int32_t*>(stats + 2);
    r.N = a.N;
    r.Q = a.Q;
    r.Qp = a.Qp;
    r.Qtp = a.Qtp;
    r.nfullq = a.nfullq;
    r.T = T;
    r.d = a.d;
    r.P = a.P;
    r.k = k;
    r.norm = norm;
    r.dot = tc ? 2 : (dot ? 1 : 0);
    r.xf = xf;
    {
        KernelTimer kt(TK_KNN_RERANK, c.stream);
        knn_rerank_kernel<<<(a.Q + kRerankWarps - 1) / kRerankWarps, kRerankWarps * 32, 0, c.stream>>>(r);
        kt.stop();
    }
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    int egrid = a.Q < 2 * c.num_sms ? a.Q : 2 * c.num_sms;
    knn_exact_kernel<<<egrid, kExactThreads, 0, c.stream>>>(r);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    if (info) {  // per-call diagnostics: the caller asked for them, so this call synchronises
        uint32_t h[8] = {};
        LIPFIT_CUDA(cudaMemcpyAsync(h, stats, sizeof(h), cudaMemcpyDeviceToHost, c.stream));
        LIPFIT_CUDA(cudaStreamSynchronize(c.stream));
        float ratio;
        memcpy(&ratio, &h[4], sizeof(ratio));
        info->fallbacks = static_cast<int64_t>(static_cast<int32_t>(h[2]));
        info->key_error_ratio = static_cast<double>(ratio);
        info->tensor_cores = tc ? 1 : 0;
        info->reserved = 0;
    }
    return LIPFIT_OK;
}

}  // namespace lipfit
