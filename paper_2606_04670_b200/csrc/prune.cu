// prune.cu -- NEXT-4(ii): Eq.(2),(3) PAPER.md:103-116 evaluated EXACTLY with spatial pruning.
//
// The paper visits all N data per query and prunes only heuristically (the M/3 pair
// removal of smoothing).  Here the pruning is exact: data and queries are sorted along a Morton curve of the packed coordinates;
// 32 consecutive data form a tile with a bounding box [lo, hi] and the range [ymin, ymax] of its
// values, 32 consecutive queries form a warp with a bounding box.  For a tile t and a set of
// queries B
//     y^k + M D^u(q, x^k) >= ymin_t + M dlb^u(B, t)      for every q in B, k in t
//     y^k - M D^l(q, x^k) <= ymax_t - M dlb^l(B, t)
// where dlb is the norm of the componentwise smallest possible |delta| / relu(+-delta) between
// the two boxes.  A tile whose first quantity is not below the largest running upper bound of B
// and whose second is not above the smallest running lower bound of B cannot change any running
// extremum and is skipped.  Two stages: (1) lane = tile, warp box against tile box with the
// warp-wide extrema; (2) per surviving tile, lane = query, the query point against the tile box
// with the lane's own running bounds, the tile is evaluated if any lane needs it.  Running bounds
// are seeded from the tile(s) at the queries' own Morton position.
//
// Exactness in fp32: a pair is evaluated as fmaf(M, D, y) with D the rounded norm; the box
// distance is scaled by (1 - 1e-5), which covers the rounding of both norms ((DP + 3) 2^-24 each),
// and fmaf is monotone in its addend and multiplicand, so the computed tile bound never exceeds a
// computed pair value of that tile: the result is the min / max over all N data of the same
// per-pair arithmetic, whatever was skipped.
#include <cub/device/device_radix_sort.cuh>

#include "kernels.h"

namespace lipfit {

namespace {

constexpr int kTile = 32;  // data per tile = lanes per warp

// ---- coordinate ranges of the packed data -----------------------------------------------------
__global__ void prune_range_init_kernel(uint32_t* keys) {
    int j = threadIdx.x;
    if (j < kMaxDim) {
        keys[j] = 0xFFFFFFFFu;      // running minimum
        keys[kMaxDim + j] = 0u;     // running maximum
    }
}

__global__ void __launch_bounds__(256)
prune_range_kernel(const float* __restrict__ X, int N, Xform xf, uint32_t* __restrict__ keys) {
    __shared__ uint32_t smin[kMaxDim], smax[kMaxDim];
    if (threadIdx.x < kMaxDim) {
        smin[threadIdx.x] = 0xFFFFFFFFu;
        smax[threadIdx.x] = 0u;
    }
    __syncthreads();
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < N; k += gridDim.x * blockDim.x) {
        const float* src = X + static_cast<size_t>(k) * xf.d;
        for (int j = 0; j < xf.d; ++j) {
            uint32_t key = f2key(xf.sw[j] * src[xf.perm[j]]);
            atomicMin(&smin[j], key);
            atomicMax(&smax[j], key);
        }
    }
    __syncthreads();
    if (threadIdx.x < xf.d) {
        atomicMin(&keys[threadIdx.x], smin[threadIdx.x]);
        atomicMax(&keys[kMaxDim + threadIdx.x], smax[threadIdx.x]);
    }
}

// Morton key of one point: cell index per coordinate inside the data range (clamped), bits
// interleaved, coordinate 0 most significant within a level.
__device__ __forceinline__ uint64_t morton_key(const float* __restrict__ src, const Xform& xf,
                                               const uint32_t* __restrict__ keys, int bits) {
    uint32_t cell[kMaxDim];
    const float cells = static_cast<float>(1u << bits);
    for (int j = 0; j < xf.d; ++j) {
        float lo = key2f(keys[j]), hi = key2f(keys[kMaxDim + j]);
        float v = xf.sw[j] * src[xf.perm[j]];
        float w = hi - lo;
        float t = w > 0.f ? (v - lo) / w * cells : 0.f;
        t = fminf(fmaxf(t, 0.f), cells - 1.f);
        cell[j] = static_cast<uint32_t>(t);
    }
    uint64_t key = 0;
    for (int b = bits - 1; b >= 0; --b)
        for (int j = 0; j < xf.d; ++j) key = (key << 1) | ((cell[j] >> b) & 1u);
    return key;
}

__global__ void __launch_bounds__(256)
prune_keys_kernel(const float* __restrict__ P, int n, Xform xf, const uint32_t* __restrict__ keys, int bits,
                  uint64_t* __restrict__ out, int32_t* __restrict__ ids) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    out[k] = morton_key(P + static_cast<size_t>(k) * xf.d, xf, keys, bits);
    ids[k] = k;
}

// ---- sorted records and tile boxes: one warp per tile, lane = record --------------------------
// rec : ntiles * 32 records of RF = DP + 4 floats [x'_0 .. x'_{DP-1}, y, 0, 0, 0]; the last tile is
//       filled up with copies of the last datum (they change no minimum or maximum)
// box : ntiles * (2 DP + 4) floats [lo_0 .. lo_{DP-1}, hi_0 .. hi_{DP-1}, ymin, ymax, 0, 0]
// xfp: the PADDED transform of launch_bounds_pruned (DP packed coordinates), dsrc: floats per source row.
template <int DP>
__global__ void __launch_bounds__(128)
prune_gather_kernel(const float* __restrict__ X, const float* __restrict__ y, const float* __restrict__ eps,
                    int N, Xform xfp, int dsrc, const int32_t* __restrict__ order, int ntiles,
                    float* __restrict__ rec, float* __restrict__ box) {
    constexpr int RF = DP + 4, BF = 2 * DP + 4;
    const int lane = threadIdx.x & 31;
    const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (t >= ntiles) return;
    int pos = t * kTile + lane;
    if (pos >= N) pos = N - 1;
    const int k = order[pos];
    const float* src = X + static_cast<size_t>(k) * dsrc;
    float v[DP];
#pragma unroll
    for (int j = 0; j < DP; ++j) v[j] = xfp.sw[j] * src[xfp.perm[j]];
    const float yv = eps ? y[k] + eps[k] : y[k];  // smoothing: z = y + eps
    float4* dst = reinterpret_cast<float4*>(rec + (static_cast<size_t>(t) * kTile + lane) * RF);
#pragma unroll
    for (int j = 0; j < DP; j += 4) dst[j >> 2] = make_float4(v[j], v[j + 1], v[j + 2], v[j + 3]);
    dst[DP >> 2] = make_float4(yv, 0.f, 0.f, 0.f);
    float* b = box + static_cast<size_t>(t) * BF;
#pragma unroll
    for (int j = 0; j < DP; ++j) {
        float lo = v[j], hi = v[j];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, o));
            hi = fmaxf(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        }
        if (lane == 0) {
            b[j] = lo;
            b[DP + j] = hi;
        }
    }
    float ylo = yv, yhi = yv;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        ylo = fminf(ylo, __shfl_xor_sync(0xffffffffu, ylo, o));
        yhi = fmaxf(yhi, __shfl_xor_sync(0xffffffffu, yhi, o));
    }
    if (lane == 0) {
        b[2 * DP] = ylo;
        b[2 * DP + 1] = yhi;
        b[2 * DP + 2] = 0.f;
        b[2 * DP + 3] = 0.f;
    }
}

// ---- box distances -----------------------------------------------------------------------------
// Smallest possible D^u and D^l between a query box [qlo, qhi] and a tile box [tlo, thi]
// (delta = q - x):  a = qlo - thi <= delta <= qhi - tlo = -b.
//   unconstrained: |delta| >= max(a, b, 0) on both sides
//   constrained  : relu(delta) >= max(a, 0),  relu(-delta) >= max(b, 0)
// DC >= 0: the last DC packed coordinates are the constrained ones (compile time); DC < 0: runtime flags.
template <int NORM, int DP, int DC>
__device__ __forceinline__ void box_lb(const float* __restrict__ qlo, const float* __restrict__ qhi,
                                       const float* __restrict__ tb, const FreeFlags& ff, float& du,
                                       float& dl) {
    float pu = 0.f, pl = 0.f;
#pragma unroll
    for (int j = 0; j < DP; ++j) {
        float a = qlo[j] - tb[DP + j];
        float b = tb[j] - qhi[j];
        float u, l;
        if (DC < 0) {
            u = fmaxf(fmaxf(a, ff.fr[j] * b), 0.f);
            l = fmaxf(fmaxf(b, ff.fr[j] * a), 0.f);
        } else if (j < DP - DC) {
            u = l = fmaxf(fmaxf(a, b), 0.f);
        } else {
            u = fmaxf(a, 0.f);
            l = fmaxf(b, 0.f);
        }
        if (NORM == 1) {
            pu += u;
            pl += l;
        }
        if (NORM == 2) {
            pu = fmaf(u, u, pu);
            pl = fmaf(l, l, pl);
        }
        if (NORM == 3) {
            pu = fmaxf(pu, u);
            pl = fmaxf(pl, l);
        }
    }
    constexpr float kShrink = 1.f - 1e-5f;  // covers the rounding of this norm and of the pair's norm
    du = (NORM == 2 ? fast_sqrt(pu) : pu) * kShrink;
    dl = (NORM == 2 ? fast_sqrt(pl) : pl) * kShrink;
}

struct PruneArgs {
    const float* Xq;
    const int32_t* qorder;     // sorted position -> original query
    const uint64_t* qkeys;     // sorted Morton keys of the queries
    const uint64_t* dkeys;     // sorted Morton keys of the data
    const float* rec;
    const float* box;
    int N, Q, ntiles, dsrc;
    float M;
    Xform xfp;                 // padded transform: [unconstrained, zero padding, constrained], DP coordinates
    FreeFlags ff;
    float *upper, *lower, *g;
    unsigned long long* stats;  // [0] tiles evaluated (x 1024 pairs), [1] stage-1 survivors, [2] lanes that needed them
    // Guard of LIPFIT_BOUNDS_AUTO (NULL: none).  guard[0] += tiles evaluated by FINISHED query groups,
    // guard[1] += finished groups, guard[2] = 1 once the finished groups have evaluated more than guard_limit
    // of their pairs (checked from guard_min finished groups on, while fewer than half of all groups are done):
    // groups that have not started yet then return at once, and the caller runs the all-pairs kernels.
    unsigned long long* guard;
    float guard_limit;
    int guard_min;
};

template <int NORM, int DP, int DC>
__device__ __forceinline__ void pair_acc(const float* q, const float* x, const FreeFlags& ff, float& au, float& al) {
    if (DC < 0) PairAccGeneric<NORM, DP>::run(q, x, ff, au, al);
    else PairAcc<NORM, DP - (DC < 0 ? 0 : DC), (DC < 0 ? 0 : DC)>::run(q, x, au, al);
}

// One tile against the warp's 32 queries.  Every lane fetches ONE record of the tile (coalesced, a single
// L2 round trip per tile), the warp parks the 32 records in its own shared-memory slab as float4 columns
// (sm[c * 32 + r] = 16-byte word c of record r: conflict-free stores, broadcast loads), then every lane
// runs its query against all 32 records.
template <int NORM, int DP, int DC>
__device__ __forceinline__ void eval_tile(const float* __restrict__ rec, int t, float4* __restrict__ sm,
                                          const float* q, const FreeFlags& ff, float M, float& U, float& L) {
    constexpr int RF = DP + 4, W = RF / 4;
    const int lane = threadIdx.x & 31;
    const float4* g = reinterpret_cast<const float4*>(rec + static_cast<size_t>(t) * kTile * RF) + lane * W;
    float4 v[W];
#pragma unroll
    for (int c = 0; c < W; ++c) v[c] = __ldg(g + c);
    __syncwarp();  // every lane has finished reading the previous tile
#pragma unroll
    for (int c = 0; c < W - 1; ++c) sm[c * 32 + lane] = v[c];
    // the 32 values packed into eight 16-byte words: one load serves four records
    reinterpret_cast<float*>(sm + (W - 1) * 32)[lane] = v[W - 1].x;
    __syncwarp();
#pragma unroll 2
    for (int r0 = 0; r0 < kTile; r0 += 4) {
        const float4 y4 = sm[(W - 1) * 32 + (r0 >> 2)];
        const float yv4[4] = {y4.x, y4.y, y4.z, y4.w};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int r = r0 + u;
            float x[DP];
#pragma unroll
            for (int j = 0; j < DP; j += 4) {
                const float4 xv = sm[(j >> 2) * 32 + r];
                x[j] = xv.x;
                x[j + 1] = xv.y;
                x[j + 2] = xv.z;
                x[j + 3] = xv.w;
            }
            float au, al;
            pair_acc<NORM, DP, DC>(q, x, ff, au, al);
            U = fminf(U, fmaf(M, PairAccGeneric<NORM, DP>::finish(au), yv4[u]));
            L = fmaxf(L, fmaf(-M, PairAccGeneric<NORM, DP>::finish(al), yv4[u]));
        }
    }
}

__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ float warp_min(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

template <int NORM, int DP, int DC>
__global__ void __launch_bounds__(128)
bounds_pruned_kernel(const PruneArgs a) {
    constexpr int BF = 2 * DP + 4;
    __shared__ float4 slab[4][(DP + 4) / 4 * 32];
    float4* sm = slab[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const int nwarps = (a.Q + 31) >> 5;
    const int nchunks = (a.ntiles + 31) >> 5;
    unsigned long long n_eval = 0, n_surv = 0, n_mine = 0;
    for (int w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); w < nwarps;
         w += gridDim.x * (blockDim.x >> 5)) {
        if (a.guard && *reinterpret_cast<volatile unsigned long long*>(a.guard + 2) != 0ull) break;  // warp-uniform
        const unsigned long long n_eval_before = n_eval;
        const int pos = min(w * 32 + lane, a.Q - 1);
        const bool live = (w * 32 + lane) < a.Q;
        const int qi = a.qorder[pos];
        const float* src = a.Xq + static_cast<size_t>(qi) * a.dsrc;
        float q[DP];
#pragma unroll
        for (int j = 0; j < DP; ++j) q[j] = a.xfp.sw[j] * src[a.xfp.perm[j]];
        float qlo[DP], qhi[DP];
#pragma unroll
        for (int j = 0; j < DP; ++j) {
            qlo[j] = warp_min(q[j]);
            qhi[j] = warp_max(q[j]);
        }
        // seed: the tile at the lane's own Morton position among the data
        int mytile;
        {
            const uint64_t key = a.qkeys[pos];
            int lo = 0, hi = a.N;  // first datum with key >= the query's
            while (lo < hi) {
                int mid = (lo + hi) >> 1;
                if (a.dkeys[mid] < key) lo = mid + 1;
                else hi = mid;
            }
            mytile = min(lo, a.N - 1) / kTile;
        }
        float U = __int_as_float(0x7f800000), L = __int_as_float(0xff800000);
        {
            unsigned todo = 0xffffffffu;
            while (todo) {
                const int t = __shfl_sync(0xffffffffu, mytile, __ffs(todo) - 1);
                eval_tile<NORM, DP, DC>(a.rec, t, sm, q, a.ff, a.M, U, L);
                ++n_eval;
                todo &= ~__ballot_sync(0xffffffffu, mytile == t);
            }
        }
        float Umax = warp_max(U), Lmin = warp_min(L);
        // chunks of 32 tiles, from the chunk of the seed outwards along the curve (near tiles first: the
        // running bounds tighten early; a separate first pass over the tiles that touch the warp's box was
        // measured and changes the number of evaluated tiles by < 2 %: the seeds already give tight bounds)
        const int c0 = __shfl_sync(0xffffffffu, mytile, 0) >> 5;
        int up = c0, down = c0 - 1;
        for (int i = 0; i < nchunks; ++i) {
            int chunk;
            if (down < 0 || (up < nchunks && (i & 1) == 0)) chunk = up++;
            else chunk = down--;
            const int tb = chunk << 5;
            const int t = tb + lane;
            bool need = false;
            if (t < a.ntiles) {
                const float* b = a.box + static_cast<size_t>(t) * BF;
                float tbx[2 * DP];
#pragma unroll
                for (int j = 0; j < 2 * DP; j += 4) {
                    float4 v = __ldg(reinterpret_cast<const float4*>(b + j));
                    tbx[j] = v.x;
                    tbx[j + 1] = v.y;
                    tbx[j + 2] = v.z;
                    tbx[j + 3] = v.w;
                }
                const float4 yy = __ldg(reinterpret_cast<const float4*>(b + 2 * DP));
                float du, dl;
                box_lb<NORM, DP, DC>(qlo, qhi, tbx, a.ff, du, dl);
                need = (fmaf(a.M, du, yy.x) < Umax) || (fmaf(-a.M, dl, yy.y) > Lmin);
            }
            unsigned surv = __ballot_sync(0xffffffffu, need);
            if (!surv) continue;
            bool any_eval = false;
            while (surv) {
                const int s = __ffs(surv) - 1;
                surv &= surv - 1;
                const int ts = tb + s;
                ++n_surv;
                if (__any_sync(0xffffffffu, mytile == ts)) continue;  // evaluated as a seed
                // stage 2: the lane's own query against the tile box, with its own running bounds
                const float* b = a.box + static_cast<size_t>(ts) * BF;
                float tbx[2 * DP];
#pragma unroll
                for (int j = 0; j < 2 * DP; j += 4) {
                    float4 v = __ldg(reinterpret_cast<const float4*>(b + j));
                    tbx[j] = v.x;
                    tbx[j + 1] = v.y;
                    tbx[j + 2] = v.z;
                    tbx[j + 3] = v.w;
                }
                const float4 yy = __ldg(reinterpret_cast<const float4*>(b + 2 * DP));
                float du, dl;
                box_lb<NORM, DP, DC>(q, q, tbx, a.ff, du, dl);
                const bool mine = (fmaf(a.M, du, yy.x) < U) || (fmaf(-a.M, dl, yy.y) > L);
                const unsigned who = __ballot_sync(0xffffffffu, mine);
                if (!who) continue;
                eval_tile<NORM, DP, DC>(a.rec, ts, sm, q, a.ff, a.M, U, L);
                ++n_eval;
                n_mine += __popc(who);
                any_eval = true;
            }
            if (any_eval) {
                Umax = warp_max(U);
                Lmin = warp_min(L);
            }
        }
        if (live) {
            if (a.upper) a.upper[qi] = U;
            if (a.lower) a.lower[qi] = L;
            if (a.g) a.g[qi] = 0.5f * (U + L);
        }
        if (a.guard && lane == 0) {
            const unsigned long long tiles = atomicAdd(a.guard, n_eval - n_eval_before) + (n_eval - n_eval_before);
            const unsigned long long done = atomicAdd(a.guard + 1, 1ull) + 1ull;
            // fraction of their pairs the finished groups evaluated = tiles * 32 / (done * N)
            if (done >= static_cast<unsigned long long>(a.guard_min) && 2ull * done < static_cast<unsigned long long>(nwarps) &&
                static_cast<float>(tiles) * static_cast<float>(kTile) >
                    a.guard_limit * static_cast<float>(done) * static_cast<float>(a.N))
                atomicExch(a.guard + 2, 1ull);
        }
    }
    if (a.stats && lane == 0) {
        atomicAdd(&a.stats[0], n_eval);
        atomicAdd(&a.stats[1], n_surv);
        atomicAdd(&a.stats[2], n_mine);
    }
}

struct PruneLaunch {
    const float *X, *y;
    const int32_t* dorder;
    float *rec, *box;
};

template <int NORM, int DP, int DC>
int launch_pruned_t(const Ctx& c, const PruneLaunch& pl, const PruneArgs& a) {
    prune_gather_kernel<DP><<<(a.ntiles + 3) / 4, 128, 0, c.stream>>>(pl.X, pl.y, nullptr, a.N, a.xfp, a.dsrc,
                                                                     pl.dorder, a.ntiles, pl.rec, pl.box);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    // one warp per group of 32 queries, every CTA launched: the groups differ in the number of surviving
    // tiles, the hardware scheduler balances them
    const int grid = ((a.Q + 31) / 32 + 3) / 4;
    KernelTimer kt(TK_BOUNDS_PRUNED, c.stream);
    bounds_pruned_kernel<NORM, DP, DC><<<grid, 128, 0, c.stream>>>(a);
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

template <int NORM, int DP, int DC>
struct PruneDispatchDC {
    static int run(int dc, const Ctx& c, const PruneLaunch& pl, const PruneArgs& a) {
        if (dc == DC) return launch_pruned_t<NORM, DP, DC>(c, pl, a);
        return PruneDispatchDC<NORM, DP, DC - 1>::run(dc, c, pl, a);
    }
};
template <int NORM, int DP>
struct PruneDispatchDC<NORM, DP, -1> {
    static int run(int, const Ctx& c, const PruneLaunch& pl, const PruneArgs& a) {
        return launch_pruned_t<NORM, DP, -1>(c, pl, a);
    }
};

// DP <= 8: the number of constrained coordinates is a compile-time constant of the kernel (no flag
// arithmetic per pair); DP = 16, 32: runtime flags.
template <int NORM>
int launch_pruned_n(int dp, int dc, const Ctx& c, const PruneLaunch& pl, const PruneArgs& a) {
    switch (dp) {
        case 4: return PruneDispatchDC<NORM, 4, 4>::run(dc, c, pl, a);
        case 8: return PruneDispatchDC<NORM, 8, 8>::run(dc, c, pl, a);
        case 16: return launch_pruned_t<NORM, 16, -1>(c, pl, a);
        default: return launch_pruned_t<NORM, 32, -1>(c, pl, a);
    }
}

// Morton keys of n points, sorted; order[i] = original index of the i-th point along the curve.
int sorted_keys(const Ctx& c, const float* P, int n, const Xform& xf, const uint32_t* range, int bits,
                Workspace& keys_sorted, Workspace& order) {
    Workspace keys_in, ids_in, tmp;
    int rc = keys_in.alloc(sizeof(uint64_t) * n, c.stream);
    if (rc) return rc;
    if ((rc = ids_in.alloc(sizeof(int32_t) * n, c.stream))) return rc;
    if ((rc = keys_sorted.alloc(sizeof(uint64_t) * n, c.stream))) return rc;
    if ((rc = order.alloc(sizeof(int32_t) * n, c.stream))) return rc;
    prune_keys_kernel<<<(n + 255) / 256, 256, 0, c.stream>>>(P, n, xf, range, bits, keys_in.as<uint64_t>(),
                                                             ids_in.as<int32_t>());
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    size_t tmp_bytes = 0;
    const int end_bit = bits * xf.d > 0 ? bits * xf.d : 1;
    LIPFIT_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, keys_in.as<uint64_t>(),
                                                keys_sorted.as<uint64_t>(), ids_in.as<int32_t>(),
                                                order.as<int32_t>(), n, 0, end_bit, c.stream));
    if ((rc = tmp.alloc(tmp_bytes, c.stream))) return rc;
    LIPFIT_CUDA(cub::DeviceRadixSort::SortPairs(tmp.p, tmp_bytes, keys_in.as<uint64_t>(),
                                                keys_sorted.as<uint64_t>(), ids_in.as<int32_t>(),
                                                order.as<int32_t>(), n, 0, end_bit, c.stream));
    return LIPFIT_OK;
}


// ---------------------------------------------------------------------------------------------
// Smoothing objective / gradient, Eq.(5)-(7) PAPER.md:189-198, with the same exact pruning.
// From datum i's side (reading R12):  V_ik = (z_i - (z_k + M D^u(x^i, k)))_+  is i's violation of the
// upper bound set by k, V_ki = ((z_k - M D^l(x^i, k)) - z_i)_+  its violation of the lower bound, so
//   F = ||eps||^2 / p + sum_i sum_k (V_ik^2 + V_ki^2),   dF/deps_i = 2 eps_i / p + 4 sum_k (V_ik - V_ki),
// i.e. the bounds pass with the data as queries and a different reduction.  A tile B is skipped for
// the data of tile A when  zmin_B + M dlb^u >= zmax_A  and  zmax_B - M dlb^l <= zmin_A : then every
// V_ik and V_ki with i in A, k in B is exactly 0 in the kernel's own arithmetic (same argument as above).
// One warp per tile A, lane = datum i (coordinates and z_i in registers); pair terms in fp32, the sums
// of a tile's 32 terms go into fp64 accumulators.
struct SmoothPruneArgs {
    const float* rec;
    const float* box;
    const int32_t* order;
    const float* eps;  // original order, may be NULL
    int N, ntiles;
    float M, p;
    FreeFlags ff;
    double* fpart;     // [ntiles] per-tile share of F (reduced in tile order by smooth_pruned_final_kernel)
    float* vpart;      // [ntiles] per-tile max over pairs of V_ik
    float* grad;       // original order, may be NULL
    unsigned long long* stats;
};

template <int NORM, int DP, int DC>
__global__ void __launch_bounds__(128)
smooth_pruned_kernel(const SmoothPruneArgs a) {
    constexpr int RF = DP + 4, W = RF / 4, BF = 2 * DP + 4;
    __shared__ float4 slab[4][W * 32];
    float4* sm = slab[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const int nchunks = (a.ntiles + 31) >> 5;
    const int A = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (A >= a.ntiles) return;
    const int pos = A * kTile + lane;
    const bool live = pos < a.N;
    float q[DP], zi;
    {
        const float4* g = reinterpret_cast<const float4*>(a.rec + static_cast<size_t>(pos) * RF);
#pragma unroll
        for (int j = 0; j < DP; j += 4) {
            const float4 v = __ldg(g + (j >> 2));
            q[j] = v.x;
            q[j + 1] = v.y;
            q[j + 2] = v.z;
            q[j + 3] = v.w;
        }
        zi = __ldg(g + (W - 1)).x;
    }
    float qlo[DP], qhi[DP];
    const float* ba = a.box + static_cast<size_t>(A) * BF;
#pragma unroll
    for (int j = 0; j < DP; ++j) {
        qlo[j] = __ldg(ba + j);
        qhi[j] = __ldg(ba + DP + j);
    }
    const float zminA = __ldg(ba + 2 * DP), zmaxA = __ldg(ba + 2 * DP + 1);
    double Fi = 0.0, gi = 0.0;
    float vmax = 0.f;
    unsigned long long n_eval = 0;
    for (int chunk = 0; chunk < nchunks; ++chunk) {
        const int tb = chunk << 5;
        const int t = tb + lane;
        bool need = false;
        if (t < a.ntiles) {
            const float* b = a.box + static_cast<size_t>(t) * BF;
            float tbx[2 * DP];
#pragma unroll
            for (int j = 0; j < 2 * DP; j += 4) {
                float4 v = __ldg(reinterpret_cast<const float4*>(b + j));
                tbx[j] = v.x;
                tbx[j + 1] = v.y;
                tbx[j + 2] = v.z;
                tbx[j + 3] = v.w;
            }
            const float4 zz = __ldg(reinterpret_cast<const float4*>(b + 2 * DP));
            float du, dl;
            box_lb<NORM, DP, DC>(qlo, qhi, tbx, a.ff, du, dl);
            need = (fmaf(a.M, du, zz.x) < zmaxA) || (fmaf(-a.M, dl, zz.y) > zminA);
        }
        unsigned surv = __ballot_sync(0xffffffffu, need);
        while (surv) {
            const int s = __ffs(surv) - 1;
            surv &= surv - 1;
            const int ts = tb + s;
            const float* b = a.box + static_cast<size_t>(ts) * BF;
            float tbx[2 * DP];
#pragma unroll
            for (int j = 0; j < 2 * DP; j += 4) {
                float4 v = __ldg(reinterpret_cast<const float4*>(b + j));
                tbx[j] = v.x;
                tbx[j + 1] = v.y;
                tbx[j + 2] = v.z;
                tbx[j + 3] = v.w;
            }
            const float4 zz = __ldg(reinterpret_cast<const float4*>(b + 2 * DP));
            float du, dl;
            box_lb<NORM, DP, DC>(q, q, tbx, a.ff, du, dl);
            const bool mine = (fmaf(a.M, du, zz.x) < zi) || (fmaf(-a.M, dl, zz.y) > zi);
            if (!__any_sync(0xffffffffu, mine)) continue;
            // evaluate tile ts (only its real records: the filled-up tail of the last tile is left out)
            const float4* g = reinterpret_cast<const float4*>(a.rec + static_cast<size_t>(ts) * kTile * RF) + lane * W;
            float4 v[W];
#pragma unroll
            for (int c = 0; c < W; ++c) v[c] = __ldg(g + c);
            __syncwarp();
#pragma unroll
            for (int c = 0; c < W; ++c) sm[c * 32 + lane] = v[c];
            __syncwarp();
            const int n = min(kTile, a.N - ts * kTile);
            float fs = 0.f, gs = 0.f;
#pragma unroll 4
            for (int r = 0; r < n; ++r) {
                float x[DP];
#pragma unroll
                for (int j = 0; j < DP; j += 4) {
                    const float4 xv = sm[(j >> 2) * 32 + r];
                    x[j] = xv.x;
                    x[j + 1] = xv.y;
                    x[j + 2] = xv.z;
                    x[j + 3] = xv.w;
                }
                const float zk = sm[(W - 1) * 32 + r].x;
                float au, al;
                pair_acc<NORM, DP, DC>(q, x, a.ff, au, al);
                const float v1 = fmaxf(zi - fmaf(a.M, PairAccGeneric<NORM, DP>::finish(au), zk), 0.f);
                const float v2 = fmaxf(fmaf(-a.M, PairAccGeneric<NORM, DP>::finish(al), zk) - zi, 0.f);
                fs = fmaf(v1, v1, fs);
                fs = fmaf(v2, v2, fs);
                gs += v1 - v2;
                vmax = fmaxf(vmax, fmaxf(v1, v2));
            }
            Fi += static_cast<double>(fs);
            gi += static_cast<double>(gs);
            ++n_eval;
        }
    }
    if (live) {
        const int orig = a.order[pos];
        const double e = a.eps ? static_cast<double>(a.eps[orig]) : 0.0;
        Fi += e * e / static_cast<double>(a.p);
        if (a.grad) a.grad[orig] = static_cast<float>(2.0 * e / static_cast<double>(a.p) + 4.0 * gi);
    } else {
        Fi = 0.0;
        vmax = 0.f;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) Fi += __shfl_xor_sync(0xffffffffu, Fi, o);
    vmax = warp_max(vmax);
    if (lane == 0) {
        a.fpart[A] = Fi;  // fixed summation order inside the warp (xor tree) and over the tiles: reproducible
        a.vpart[A] = vmax;
        if (a.stats) atomicAdd(&a.stats[0], n_eval);
    }
}

// Single block, fixed order: F = sum of the per-tile shares, maxviol = their maximum.
__global__ void __launch_bounds__(256)
smooth_pruned_final_kernel(const double* __restrict__ fpart, const float* __restrict__ vpart, int ntiles,
                           double* __restrict__ F, double* __restrict__ maxviol) {
    __shared__ double rf_[256], rv_[256];
    double f = 0.0, v = 0.0;
    for (int t = threadIdx.x; t < ntiles; t += 256) {
        f += fpart[t];
        v = fmax(v, static_cast<double>(vpart[t]));
    }
    rf_[threadIdx.x] = f;
    rv_[threadIdx.x] = v;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) {
            rf_[threadIdx.x] += rf_[threadIdx.x + o];
            rv_[threadIdx.x] = fmax(rv_[threadIdx.x], rv_[threadIdx.x + o]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        *F = rf_[0];
        if (maxviol) *maxviol = rv_[0];
    }
}

template <int NORM, int DP, int DC>
int launch_smooth_pruned_t(const Ctx& c, const PruneLaunch& pl, const Xform& xfp, int dsrc, const float* eps,
                           const SmoothPruneArgs& a) {
    prune_gather_kernel<DP><<<(a.ntiles + 3) / 4, 128, 0, c.stream>>>(pl.X, pl.y, eps, a.N, xfp, dsrc, pl.dorder,
                                                                     a.ntiles, pl.rec, pl.box);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    KernelTimer kt(TK_SMOOTH_PRUNED, c.stream);
    smooth_pruned_kernel<NORM, DP, DC><<<(a.ntiles + 3) / 4, 128, 0, c.stream>>>(a);
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

template <int NORM, int DP, int DC>
struct SmoothDispatchDC {
    static int run(int dc, const Ctx& c, const PruneLaunch& pl, const Xform& xfp, int dsrc, const float* eps,
                   const SmoothPruneArgs& a) {
        if (dc == DC) return launch_smooth_pruned_t<NORM, DP, DC>(c, pl, xfp, dsrc, eps, a);
        return SmoothDispatchDC<NORM, DP, DC - 1>::run(dc, c, pl, xfp, dsrc, eps, a);
    }
};
template <int NORM, int DP>
struct SmoothDispatchDC<NORM, DP, -1> {
    static int run(int, const Ctx& c, const PruneLaunch& pl, const Xform& xfp, int dsrc, const float* eps,
                   const SmoothPruneArgs& a) {
        return launch_smooth_pruned_t<NORM, DP, -1>(c, pl, xfp, dsrc, eps, a);
    }
};

template <int NORM>
int launch_smooth_pruned_n(int dp, int dc, const Ctx& c, const PruneLaunch& pl, const Xform& xfp, int dsrc,
                           const float* eps, const SmoothPruneArgs& a) {
    switch (dp) {
        case 4: return SmoothDispatchDC<NORM, 4, 4>::run(dc, c, pl, xfp, dsrc, eps, a);
        case 8: return SmoothDispatchDC<NORM, 8, 8>::run(dc, c, pl, xfp, dsrc, eps, a);
        case 16: return launch_smooth_pruned_t<NORM, 16, -1>(c, pl, xfp, dsrc, eps, a);
        default: return launch_smooth_pruned_t<NORM, 32, -1>(c, pl, xfp, dsrc, eps, a);
    }
}

// padded transform: unconstrained coordinates, zero padding up to dp, constrained coordinates last
Xform padded_xform(const Xform& xf, int dp) {
    Xform xfp = xf;
    xfp.d = dp;
    const int npad = dp - xf.d;
    for (int j = 0; j < dp; ++j) {
        if (j < xf.dU) continue;
        if (j < xf.dU + npad) {
            xfp.perm[j] = 0;
            xfp.sw[j] = 0.f;
        } else {
            xfp.perm[j] = xf.perm[j - npad];
            xfp.sw[j] = xf.sw[j - npad];
        }
    }
    xfp.dU = xf.dU + npad;
    return xfp;
}

}  // namespace

int launch_bounds_pruned(const Ctx& c, const float* X, const float* y, int64_t N64, const float* Xq,
                         int64_t Q64, const Xform& xf, int norm, float M, float* upper, float* lower,
                         float* g, unsigned long long* stats_dev, float guard_limit, bool* declined) {
    const int N = static_cast<int>(N64), Q = static_cast<int>(Q64);
    const int dp = xf.d <= 4 ? 4 : xf.d <= 8 ? 8 : xf.d <= 16 ? 16 : 32;
    if (declined) *declined = false;
    int bits = 32 / xf.d;  // <= 32 key bits in all: four radix passes; 2^32 cells >> any N
    if (bits > 16) bits = 16;
    const int ntiles = (N + kTile - 1) / kTile;

    Workspace range, dkeys, dorder, qkeys, qorder, rec, box;
    int rc = range.alloc(sizeof(uint32_t) * 2 * kMaxDim, c.stream);
    if (rc) return rc;
    prune_range_init_kernel<<<1, 32, 0, c.stream>>>(range.as<uint32_t>());
    int rgrid = (N + 255) / 256;
    if (rgrid > c.num_sms * 8) rgrid = c.num_sms * 8;
    prune_range_kernel<<<rgrid, 256, 0, c.stream>>>(X, N, xf, range.as<uint32_t>());
    g_launches += 2;
    LIPFIT_CUDA(cudaGetLastError());
    if ((rc = sorted_keys(c, X, N, xf, range.as<uint32_t>(), bits, dkeys, dorder))) return rc;
    if ((rc = sorted_keys(c, Xq, Q, xf, range.as<uint32_t>(), bits, qkeys, qorder))) return rc;
    if ((rc = rec.alloc(sizeof(float) * static_cast<size_t>(ntiles) * kTile * (dp + 4), c.stream))) return rc;
    if ((rc = box.alloc(sizeof(float) * static_cast<size_t>(ntiles) * (2 * dp + 4), c.stream))) return rc;

    const Xform xfp = padded_xform(xf, dp);

    PruneArgs a;
    a.Xq = Xq;
    a.qorder = qorder.as<int32_t>();
    a.qkeys = qkeys.as<uint64_t>();
    a.dkeys = dkeys.as<uint64_t>();
    a.rec = rec.as<float>();
    a.box = box.as<float>();
    a.N = N;
    a.Q = Q;
    a.ntiles = ntiles;
    a.dsrc = xf.d;
    a.M = M;
    a.xfp = xfp;
    a.ff = make_free_flags(xfp);
    a.upper = upper;
    a.lower = lower;
    a.g = g;
    a.stats = stats_dev;
    a.guard = nullptr;
    a.guard_limit = 0.f;
    a.guard_min = 0;
    PruneLaunch pl{X, y, dorder.as<int32_t>(), rec.as<float>(), box.as<float>()};
    auto launch = [&]() {
        switch (norm) {
            case LIPFIT_L1: return launch_pruned_n<1>(dp, xf.dC, c, pl, a);
            case LIPFIT_L2: return launch_pruned_n<2>(dp, xf.dC, c, pl, a);
            default: return launch_pruned_n<3>(dp, xf.dC, c, pl, a);
        }
    };
    // LIPFIT_BOUNDS_AUTO: the kernel watches the fraction of pairs its finished query groups evaluated and stops
    // handing out groups once that exceeds guard_limit; ONE read-back + stream synchronisation after the kernel
    // tells the caller whether the outputs are complete.  The first finishers report when every resident warp
    // (~24 per SM) is about to finish its first group, so stopping only saves work when there are many waves of
    // groups: below 6 waves the guard stays off (measured on an adversarial config 2 shaped workload, nothing
    // prunable: Q = 1e6, 8.8 waves: guarded 46 ms, pruned pass alone 65 ms, all-pairs 32 ms; Q = 2.6e5, 2.3 waves:
    // 4.6 / 3.1 / 2.1 ms -- the guard would only add the all-pairs pass on top of a finished pruned one).
    if (!(guard_limit > 0.f && declined) || (Q + 31) / 32 < 6 * 24 * c.num_sms) return launch();
    Workspace guard;
    if ((rc = guard.alloc(4 * sizeof(unsigned long long), c.stream))) return rc;
    LIPFIT_CUDA(cudaMemsetAsync(guard.p, 0, 4 * sizeof(unsigned long long), c.stream));
    const int nwarps = (Q + 31) / 32;
    a.guard = guard.as<unsigned long long>();
    a.guard_limit = guard_limit;
    a.guard_min = nwarps / 64 > 64 ? nwarps / 64 : 64;
    if ((rc = launch())) return rc;
    unsigned long long h[4] = {0, 0, 0, 0};
    LIPFIT_CUDA(cudaMemcpyAsync(h, guard.p, sizeof(h), cudaMemcpyDeviceToHost, c.stream));
    LIPFIT_CUDA(cudaStreamSynchronize(c.stream));
    *declined = h[2] != 0ull;
    return LIPFIT_OK;
}

// Morton order of the data (coordinate ranges, keys, radix sort): depends on X only, so lipfit_smooth computes
// it once and reuses it for every evaluation of the LBFGS loop.
int smooth_pruned_order(const Ctx& c, const float* X, int64_t N64, const Xform& xf, Workspace& dorder) {
    const int N = static_cast<int>(N64);
    int bits = 32 / xf.d;
    if (bits > 16) bits = 16;
    Workspace range, dkeys;
    int rc = range.alloc(sizeof(uint32_t) * 2 * kMaxDim, c.stream);
    if (rc) return rc;
    prune_range_init_kernel<<<1, 32, 0, c.stream>>>(range.as<uint32_t>());
    int rgrid = (N + 255) / 256;
    if (rgrid > c.num_sms * 8) rgrid = c.num_sms * 8;
    prune_range_kernel<<<rgrid, 256, 0, c.stream>>>(X, N, xf, range.as<uint32_t>());
    g_launches += 2;
    LIPFIT_CUDA(cudaGetLastError());
    return sorted_keys(c, X, N, xf, range.as<uint32_t>(), bits, dkeys, dorder);
}

int launch_smooth_objective_pruned(const Ctx& c, const float* X, const float* y, const float* eps, int64_t N64,
                                   const Xform& xf, int norm, float M, float p, double* F_dev, float* grad,
                                   unsigned long long* stats_dev, double* maxviol_dev, const int32_t* order_dev) {
    const int N = static_cast<int>(N64);
    const int dp = xf.d <= 4 ? 4 : xf.d <= 8 ? 8 : xf.d <= 16 ? 16 : 32;
    const int ntiles = (N + kTile - 1) / kTile;
    Workspace dorder, rec, box, fpart, vpart;
    int rc;
    if (!order_dev) {
        if ((rc = smooth_pruned_order(c, X, N64, xf, dorder))) return rc;
        order_dev = dorder.as<int32_t>();
    }
    if ((rc = rec.alloc(sizeof(float) * static_cast<size_t>(ntiles) * kTile * (dp + 4), c.stream))) return rc;
    if ((rc = box.alloc(sizeof(float) * static_cast<size_t>(ntiles) * (2 * dp + 4), c.stream))) return rc;
    if ((rc = fpart.alloc(sizeof(double) * static_cast<size_t>(ntiles), c.stream))) return rc;
    if ((rc = vpart.alloc(sizeof(float) * static_cast<size_t>(ntiles), c.stream))) return rc;
    const Xform xfp = padded_xform(xf, dp);
    SmoothPruneArgs a;
    a.rec = rec.as<float>();
    a.box = box.as<float>();
    a.order = order_dev;
    a.eps = eps;
    a.N = N;
    a.ntiles = ntiles;
    a.M = M;
    a.p = p;
    a.ff = make_free_flags(xfp);
    a.fpart = fpart.as<double>();
    a.vpart = vpart.as<float>();
    a.grad = grad;
    a.stats = stats_dev;
    PruneLaunch pl{X, y, order_dev, rec.as<float>(), box.as<float>()};
    switch (norm) {
        case LIPFIT_L1: rc = launch_smooth_pruned_n<1>(dp, xf.dC, c, pl, xfp, xf.d, eps, a); break;
        case LIPFIT_L2: rc = launch_smooth_pruned_n<2>(dp, xf.dC, c, pl, xfp, xf.d, eps, a); break;
        default: rc = launch_smooth_pruned_n<3>(dp, xf.dC, c, pl, xfp, xf.d, eps, a); break;
    }
    if (rc) return rc;
    smooth_pruned_final_kernel<<<1, 256, 0, c.stream>>>(a.fpart, a.vpart, ntiles, F_dev, maxviol_dev);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}


}  // namespace lipfit
