// knn_common.cuh -- pieces shared by the CUDA-core selection kernels (knn.cu) and the tensor-core
// selection kernel (knn_tc.cu): candidate-pool layout, schedule, warp-cooperative compaction.
#pragma once
#include "kernels.h"

namespace lipfit {

constexpr int kKnnMargin = 8;
constexpr int kSelThreads = 128;
constexpr int kSelWarps = kSelThreads / 32;
constexpr int kMaxP = 2 * (LIPFIT_MAX_K + kKnnMargin);  // 272 pool entries per (chunk, query)

struct KnnArgs {
    const float* rec;
    const float* Xq;
    int2* pool;     // [nch][Qp][P]  (x = key bits, y = datum index)
    int32_t* fill;  // [nch][Qp]     valid entries of each pool at kernel end
    float* tau;     // [nch][Qp]     final threshold: every datum of the chunk outside the pool has key >= tau
    int N, Q, Qp, d, ksel, P;
    // Work items: query blocks [0, nfull) sweep all N data as ONE chunk (fewest pool insertions);
    // the remaining ntail blocks (the last, partial wave of the persistent grid) are cut into T
    // data chunks of `chunk` records each so that the wave stays full.  Pools: chunk 0 of query slot
    // q lives at pool slot q; chunk c >= 1 of a tail query at Qp + (c-1)*Qtp + (q - nfullq).
    int nqb, nfull, ntail, T, chunk, nfullq, Qtp;
    Xform xf;
};

__host__ __device__ __forceinline__ size_t knn_pool_slot(int qslot, int c, int Qp, int Qtp, int nfullq) {
    return c == 0 ? static_cast<size_t>(qslot)
                  : static_cast<size_t>(Qp) + static_cast<size_t>(c - 1) * Qtp + (qslot - nfullq);
}

// The rank-th smallest (1-based) of the 32 NE order-preserving integer keys a warp holds (NE per lane),
// found bit by bit with warp votes; `need` = how many of the keys equal to it belong to the rank
// smallest.  All 32 lanes must call it.
template <int NE>
__device__ __forceinline__ uint32_t knn_rank_select(const uint32_t (&key)[NE], int rank, int& need) {
    uint32_t prefix = 0;
    need = rank;  // rank still wanted among the keys that agree with `prefix` on the decided bits
#pragma unroll 1
    for (int bit = 31; bit >= 0; --bit) {
        int cnt0 = 0;  // keys that agree with prefix above `bit` and have a 0 at `bit`
#pragma unroll
        for (int i = 0; i < NE; ++i)
            cnt0 += __popc(__ballot_sync(0xffffffffu, ((key[i] ^ prefix) >> bit) == 0u));
        if (need > cnt0) {
            need -= cnt0;
            prefix |= 1u << bit;
        }
    }
    return prefix;
}

// Warp-cooperative compaction of one pool of n entries: keeps exactly the ksel entries with the
// smallest keys in slots [0, ksel) (unordered; the re-rank sorts) and returns the ksel-th smallest key
// (the new tau).  Register-resident radix select: every lane holds NE entries (n <= 32 NE), the
// ksel-th smallest order-preserving integer key is found bit by bit with warp votes (no shared
// memory, no data-dependent loads), then the kept entries are written back at their ballot-prefix
// positions; ties at the threshold are kept in pool order.  All 32 lanes must call it.
template <int NE>
__device__ __forceinline__ float knn_compact_regs(int2* pool, int n, int ksel, int lane) {
    uint32_t key[NE];
    int2 e[NE];
#pragma unroll
    for (int i = 0; i < NE; ++i) {
        const int c = lane + 32 * i;
        e[i] = c < n ? pool[c] : make_int2(0, 0);
        key[i] = c < n ? f2key(__int_as_float(e[i].x)) : 0xFFFFFFFFu;  // padding sorts last
    }
    int need;
    const uint32_t prefix = knn_rank_select<NE>(key, ksel, need);
    // prefix = the ksel-th smallest key; `need` of the entries equal to it are kept
    const unsigned below = (1u << lane) - 1u;
    int base = 0, eqbase = 0;
#pragma unroll
    for (int i = 0; i < NE; ++i) {
        const bool lt = key[i] < prefix;
        const bool eq = key[i] == prefix;
        const unsigned be = __ballot_sync(0xffffffffu, eq);
        const bool keep = lt || (eq && eqbase + __popc(be & below) < need);
        const unsigned bk = __ballot_sync(0xffffffffu, keep);
        if (keep) pool[base + __popc(bk & below)] = e[i];
        base += __popc(bk);
        eqbase += __popc(be);
    }
    __syncwarp();
    return key2f(prefix);
}

__device__ __forceinline__ float knn_compact(int2* pool, int n, int ksel, int2*, int lane) {
    if (n <= 128) return knn_compact_regs<4>(pool, n, ksel, lane);
    return knn_compact_regs<(kMaxP + 31) / 32>(pool, n, ksel, lane);
}

// knn_tc.cu: tensor-core (tcgen05) selection for symmetric L2, d <= 16.  Packs its own operand images,
// fills a.pool / a.fill / a.tau with the schedule already set in `a` (query blocks of kTcQueries) and
// writes mu (fp32 centre, kMaxDim floats) and stats[0..1] (max |x'|, max ||x' - mu||^2) for the
// certificate.  slots = CTAs of the persistent grid.
constexpr int kTcQueries = 256;  // queries per work item
constexpr int kTcBN = 128;       // data records per B tile
constexpr int kTcPoolExtra = 64; // pools of the tensor-core path hold ksel + 64 entries (knn_tc.cu: kTcSlack)
int knn_tc_slots(const Ctx& c);
int launch_knn_tc_select(const Ctx& c, const float* X, const float* Xq, KnnArgs& a, float* mu_dev,
                         uint32_t* stats);

}  // namespace lipfit
