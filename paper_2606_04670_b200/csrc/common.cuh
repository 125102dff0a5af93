// common.cuh -- shared device/host helpers of the sm_100a LipFit kernels.
// (Nothing here is shared with oracle/: the oracle is plain C and includes none of this.)
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include <nvtx3/nvToolsExt.h>  // header-only NVTX v3: a no-op unless a profiler injects itself

#include "../../include/lipfit.h"

namespace lipfit {

constexpr int kMaxDim = LIPFIT_MAX_DIM;

// Coordinate transform decided on the host from (mono_mask, weights): packed coordinate j is
//   x'_j = sw[j] * x[perm[j]],  sw = weight * (mask == -1 ? -1 : +1)          (readings R2, R3)
// with the dU unconstrained coordinates first and the dC constrained ones after them, so that
// every constrained coordinate looks "monotone increasing" to the kernels (PAPER.md:140
// "W.l.o.g. consider monotone increasing") and the mask never reaches the hot loop
// ("a suitable modification to distance calculation, which avoids branching").
struct Xform {
    int32_t perm[kMaxDim];
    float sw[kMaxDim];
    int32_t d, dU, dC;  // packed coordinates: d = dU + dC (zero-weight padding coordinates included)
    int32_t dsrc;       // floats per row of the caller's X / Xq (= d unless the transform was padded)
};

// Floats per packed record [x'_0 .. x'_{d-1}, y, pad]: a multiple of 4 so that a record is a
// whole number of 16-byte words (LDS.128 broadcast, cp.async.bulk granularity).
__host__ __device__ constexpr int record_floats(int d) { return (d + 1 + 3) & ~3; }

extern std::atomic<int64_t> g_launches;

// Optional per-kernel device timing of the three dominant kernels (lipfit_set_timing): when on,
// the launch is bracketed by CUDA events on its own stream and the call waits for it.
enum TimedKernel { TK_BOUNDS = 0, TK_KNN_SELECT = 1, TK_SMOOTH_PAIRS = 2, TK_LIPCONST_PAIRS = 3, TK_LOCAL_TABLE = 4, TK_LOCAL_EVAL = 5, TK_BOUNDS_PRUNED = 6, TK_SMOOTH_PRUNED = 7,
                   TK_KNN_RERANK = 8, TK_BOUNDS_TOPK = 9, TK_BOUNDS_REGION = 10, TK_COUNT = 11 };
struct KernelTimer {
    int which;
    cudaStream_t s;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    bool on = false;
    KernelTimer(int which_, cudaStream_t s_);
    void stop();  // call right after the launch
    ~KernelTimer();
};

// NVTX range around an entry point of the C ABI (visible in Nsight Systems / ncu --nvtx).
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
    NvtxRange(const NvtxRange&) = delete;
    NvtxRange& operator=(const NvtxRange&) = delete;
};

struct Ctx {
    cudaStream_t stream;
    int num_sms;
    int device;
};

int make_ctx(void* cuda_stream, Ctx* ctx);  // LIPFIT_OK or LIPFIT_E_CUDA

// cudaOccupancyMaxActiveBlocksPerMultiprocessor, cached per (kernel, block size, dynamic smem): the query costs
// microseconds, which is the whole budget of the latency-bound calls (config 1).
cudaError_t occupancy_cached(const void* func, int threads, size_t smem, int* occ);
template <class K>
inline cudaError_t occupancy_of(int* occ, K kern, int threads, size_t smem) {
    return occupancy_cached(reinterpret_cast<const void*>(kern), threads, smem, occ);
}

inline int cuda_rc(cudaError_t e) {
    if (e == cudaSuccess) return LIPFIT_OK;
    return (e == cudaErrorMemoryAllocation) ? LIPFIT_E_NOMEM : LIPFIT_E_CUDA;
}

#define LIPFIT_CUDA(expr)                                  \
    do {                                                   \
        cudaError_t _e = (expr);                           \
        if (_e != cudaSuccess) {                           \
            (void)cudaGetLastError();                      \
            return ::lipfit::cuda_rc(_e);                  \
        }                                                  \
    } while (0)

// The library's PRIVATE stream-ordered memory pool of the current device (created on first use, release
// threshold "keep": freed workspaces stay cached across synchronisations until lipfit_release_workspace()).
// The device's default pool, which the host application may use, is never touched.
cudaError_t workspace_pool(cudaMemPool_t* pool);

// Stream-ordered workspace that frees itself (stream-ordered) when it goes out of scope.
struct Workspace {
    void* p = nullptr;
    cudaStream_t s = nullptr;
    int alloc(size_t bytes, cudaStream_t stream) {
        s = stream;
        cudaMemPool_t pool;
        cudaError_t e = workspace_pool(&pool);
        if (e == cudaSuccess) e = cudaMallocFromPoolAsync(&p, bytes ? bytes : 16, pool, stream);
        if (e != cudaSuccess) {
            (void)cudaGetLastError();
            p = nullptr;
            return cuda_rc(e);
        }
        return LIPFIT_OK;
    }
    ~Workspace() {
        if (p) cudaFreeAsync(p, s);
    }
    template <class T>
    T* as() const { return reinterpret_cast<T*>(p); }
};

// ---------------------------------------------------------------------------------------------
// Device helpers
// ---------------------------------------------------------------------------------------------
#ifdef __CUDACC__

// One MUFU.SQRT (<= 2 ulp); sqrt(0) = 0.  DESIGN.md §6 shows the bound this leaves.
__device__ __forceinline__ float fast_sqrt(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// Order-preserving float <-> uint32 key (atomicMin/atomicMax on keys == min/max on floats).
__device__ __forceinline__ uint32_t f2key(float f) {
    uint32_t b = __float_as_uint(f);
    return b ^ ((b >> 31) ? 0xFFFFFFFFu : 0x80000000u);
}
__device__ __forceinline__ float key2f(uint32_t k) {
    uint32_t b = k ^ ((k >> 31) ? 0x80000000u : 0xFFFFFFFFu);
    return __uint_as_float(b);
}

// ---- mbarrier + 1-D bulk async copy (TMA engine; SASS UBLKCP) -------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// global -> shared::cta bulk copy of `bytes` (multiple of 16, both addresses 16-byte aligned),
// completion counted on `bar`.
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes,
                                         uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
            "r"(smem_u32(dst_smem)),
        "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

// Double-buffered stream of packed records through shared memory.
//   rec      : global records, `rf` floats each; records [begin, end) are streamed
//   buf      : 2 * TILE * rf floats of shared memory (16-byte aligned), bars: 2 mbarriers
// Usage (all threads of the CTA, uniformly):
//   RecordStream rs(...); for (int t = 0; t < rs.ntiles; ++t) { const float* s = rs.acquire(t);
//   int n = rs.count(t); ...consume s[0 .. n*rf)...; rs.release(t); }
// acquire() waits for tile t (issued one tile ahead); release() is a __syncthreads() after which
// thread 0 refills the buffer just freed.  Parities persist across streams via `phase`.
template <int TILE>
struct RecordStream {
    const float* rec;
    float* buf;
    uint64_t* bars;
    int rf, begin, end, ntiles;
    uint32_t* phase;  // per-thread copy of the two barrier parities (bit0: buf 0, bit1: buf 1)

    __device__ __forceinline__ RecordStream(const float* rec_, int rf_, int begin_, int end_,
                                            float* buf_, uint64_t* bars_, uint32_t* phase_)
        : rec(rec_), buf(buf_), bars(bars_), rf(rf_), begin(begin_), end(end_), phase(phase_) {
        ntiles = (end - begin + TILE - 1) / TILE;
        if (threadIdx.x == 0 && ntiles > 0) issue(0);
    }
    __device__ __forceinline__ int count(int t) const {
        int n = end - (begin + t * TILE);
        return n < TILE ? n : TILE;
    }
    __device__ __forceinline__ void issue(int t) {
        int b = t & 1;
        uint32_t bytes = static_cast<uint32_t>(count(t)) * rf * 4u;
        mbar_arrive_expect_tx(&bars[b], bytes);
        bulk_g2s(buf + static_cast<size_t>(b) * TILE * rf,
                 rec + static_cast<size_t>(begin + t * TILE) * rf, bytes, &bars[b]);
    }
    __device__ __forceinline__ const float* acquire(int t) {
        if (threadIdx.x == 0 && t + 1 < ntiles) issue(t + 1);
        int b = t & 1;
        mbar_wait(&bars[b], (*phase >> b) & 1u);
        *phase ^= (1u << b);
        return buf + static_cast<size_t>(b) * TILE * rf;
    }
    __device__ __forceinline__ void release(int) { __syncthreads(); }
};


// Decoupled multi-stage stream of packed records through shared memory (no CTA-wide barrier per tile).
//   buf: STAGES * TILE * rf floats (16-byte aligned), full: STAGES mbarriers (count 1),
//   done: STAGES ints in shared memory (zeroed once), NW = warps of the CTA (all of them consume).
// A warp that has finished tile t bumps done[t % STAGES]; the LAST warp to do so refills that stage
// with tile t + STAGES, so warps drift up to STAGES-1 tiles apart instead of meeting at a barrier
// every tile.  (Every LDS of the tile has completed before the bump: its values were consumed by
// arithmetic issued earlier in program order.)  Consecutive streams of one CTA are separated by the
// __syncthreads() in the constructor.
template <int TILE, int STAGES, int NW>
struct RecordPipe {
    const float* rec;
    float* buf;
    uint64_t* full;
    int* done;
    int rf, begin, end, ntiles;
    uint32_t* phase;  // per-thread parities of the STAGES full barriers

    __device__ __forceinline__ RecordPipe(const float* rec_, int rf_, int begin_, int end_, float* buf_,
                                          uint64_t* full_, int* done_, uint32_t* phase_)
        : rec(rec_), buf(buf_), full(full_), done(done_), rf(rf_), begin(begin_), end(end_),
          phase(phase_) {
        ntiles = (end - begin + TILE - 1) / TILE;
        __syncthreads();  // every warp has left the previous stream of this CTA
        if (threadIdx.x == 0)
            for (int t = 0; t < STAGES && t < ntiles; ++t) issue(t);
    }
    __device__ __forceinline__ int count(int t) const {
        int n = end - (begin + t * TILE);
        return n < TILE ? n : TILE;
    }
    __device__ __forceinline__ void issue(int t) {
        const int b = t % STAGES;
        const uint32_t bytes = static_cast<uint32_t>(count(t)) * rf * 4u;
        mbar_arrive_expect_tx(&full[b], bytes);
        bulk_g2s(buf + static_cast<size_t>(b) * TILE * rf,
                 rec + static_cast<size_t>(begin + t * TILE) * rf, bytes, &full[b]);
    }
    __device__ __forceinline__ const float* acquire(int t) {
        const int b = t % STAGES;
        mbar_wait(&full[b], (*phase >> b) & 1u);
        *phase ^= (1u << b);
        return buf + static_cast<size_t>(b) * TILE * rf;
    }
    __device__ __forceinline__ void release(int t) {
        __syncwarp();
        if ((threadIdx.x & 31) == 0) {
            const int b = t % STAGES;
            const int old = atomicAdd(&done[b], 1);
            if ((old % NW) == NW - 1 && t + STAGES < ntiles) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                issue(t + STAGES);
            }
        }
    }
};

#endif  // __CUDACC__

}  // namespace lipfit
