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

// Warp-cooperative compaction of one pool of n entries: keeps the ksel smallest (key, index)
// in slots [0, ksel) in ascending order and returns the ksel-th smallest key (the new tau).
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


// knn_tc.cu: tensor-core (tcgen05) selection for symmetric L2, d <= 16.  Packs its own operand images,
// fills a.pool / a.fill / a.tau with the schedule already set in `a` (query blocks of kTcQueries) and
// writes mu (fp32 centre, kMaxDim floats) and stats[0..1] (max |x'|, max ||x' - mu||^2) for the
// certificate.  slots = CTAs of the persistent grid.
constexpr int kTcQueries = 256;  // queries per work item
constexpr int kTcBN = 128;       // data records per B tile
int knn_tc_slots(const Ctx& c);
int launch_knn_tc_select(const Ctx& c, const float* X, const float* Xq, KnnArgs& a, float* mu_dev,
                         uint32_t* stats);

}  // namespace lipfit
