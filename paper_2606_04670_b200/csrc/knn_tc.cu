// knn_tc.cu -- step a3 on the 5th-generation tensor cores (north_star:
// "Tensor cores are used only if the L2 cross term is done as a GEMM, and then only with an
// fp32-accurate correction").  Symmetric L2, d <= 16.
//
// Selection key of (query q, datum x), both centred at mu (c = . - mu):
//     key = ||x_c||^2 - 2 q_c . x_c      ( = ||q - x||^2 - ||q_c||^2 : same order as the distance )
// as ONE bf16 GEMM with K = 64 and fp32 accumulation in tensor memory.  fp32 values are split
// v = hi + lo (two bf16, 16 significant bits) and the operand rows are
//     A (query) = [ hi(-2 q_c) | hi(-2 q_c) | lo(-2 q_c) | 1 1 1 0.. ]      d + d + d + 3 of the 64 bf16 of a row
//     B (datum) = [ hi(x_c)    | lo(x_c)    | hi(x_c)    | x2_h x2_m x2_l 0.. ]   (||x_c||^2 in 3 bf16)
// and only the ceil((3 d + 3) / 16) K steps that hold non-zero columns are multiplied (d = 16: 4, d <= 15: 3,
// d <= 9: 2, d <= 4: 1)
// so A.B = hi.hi + hi.lo + lo.hi + ||x_c||^2: the dropped lo.lo terms and the split residue are
// <= 3 * 2^-16 |q'_j x_j| per coordinate; the fp64 re-rank + certificate of knn.cu
// turn the selected pools into the exact answer, whatever the key arithmetic was.
//
// Kernel (one CTA per SM, 608 threads = 19 warps, warp-specialised):
//   warp 8   TMA producer : 1-D bulk copies of pre-swizzled operand tiles (the pack kernels write the
//                           global image in the canonical K-major SWIZZLE_128B shared-memory layout,
//                           so no tensor map is needed) into a 4-stage ring; A (2 x 128 queries) once
//                           per work item.
//   warps 9, 18 MMA issuers: one thread each, one per query half (so a held-up half does not block the
//                           other): per B tile up to 4 tcgen05.mma (M=128, N=128, K=16) into double-
//                           buffered TMEM accumulators (2 query halves x 2 stages x 128 columns).
//   warps 0-7 detectors   : tcgen05.ld 32 columns at a time (thread = query row), min-tree + one compare
//                           against the query's threshold; every row of a 32 x 32 block that holds a key
//                           below its threshold goes into a shared-memory ring as one 144-byte message.
//   warps 10-17 appenders : one per detector warp; own the thresholds and candidate pools of its 32
//                           queries, append the hits of the row messages (lane = column) / compact the
//                           pools exactly as in knn.cu, and publish lowered thresholds back through shared
//                           memory.
// Every work item starts with a seeding phase (tc_tiles_a() tiles) that gives each query a finite threshold
// before the sweep.
#include <cuda_bf16.h>

#include "knn_common.cuh"

// back-off of the ring-counter / mbarrier polls (shared-memory loads: keep them rare)
#define LIPFIT_TC_POLL_NS 100

namespace lipfit {

namespace {

constexpr int kTcThreads = 608;     // 8 detector warps, TMA warp, MMA warp (half 0), 8 appender warps, MMA warp (half 1)
// Detector -> appender ring: one message = one query row of a 32 x 32 key block that holds a key below the
// query's threshold: 32 keys + (first datum index, row) in 36 floats (16-byte aligned; the stride keeps
// the 128-bit row stores of different lanes on different banks).  Flow control: a head counter the
// detector publishes, a tail counter the appender publishes.
constexpr int kTcRowFloats = 36;
// A pool is compacted back to its ksel best entries once it holds ksel + kTcSlack: the sooner, the lower the
// thresholds the detectors test against (fewer messages) and the more compactions the appenders run.
constexpr int kTcSlack = 32;
static_assert(kTcSlack + 32 <= kTcPoolExtra, "a row message appends up to 32 entries");
constexpr int kTcRing = 96;         // row messages in flight between a detector warp and its appender warp
constexpr int kTcMinimaA = 96;      // seeding minima per query (phase A); they overlay the ring: 32 x 97 floats
constexpr int kTcRingFloats = kTcRing * kTcRowFloats;
static_assert(32 * (kTcMinimaA + 1) <= kTcRingFloats, "phase A minima overlay the ring");
constexpr int kTcStages = 4;
// Threshold seeding (phase A of a work item): the first tc_tiles_a() B tiles are multiplied once more up
// front; the detectors only take the minimum key of every group of 4 or 8 tiles per query, kTcMinimaA
// minima in all, and the appender sets the query's starting threshold to the ksel-th smallest of them
// (each minimum is the key of a different datum, so at least ksel data lie at or below it).  Without it
// the first ~1 % of the tiles of an item carry half of its appends and compactions (the thresholds
// start at +inf), a burst the appenders cannot absorb.  Groups of 8 tiles (a threshold of rank ~50 among
// the first 98 304 data instead of 49 152) pay for their extra tiles on long items only: measured on
// config 4 (7813 tiles per item) 76.0 ms with groups of 4, 74.5 with 8, 80.2 with 16.
constexpr int kTcGroupShort = 4, kTcGroupLong = 8;  // tiles per seeding minimum
constexpr int kTcLongItem = 4096;                   // tiles: items at least this long use kTcGroupLong
constexpr int kTcMaxKselA = 88;                     // of 96 minima (k <= 80)
__host__ __device__ __forceinline__ int tc_tiles_a(int tb, int te, int ksel) {
    if (ksel > kTcMaxKselA) return 0;
    if (te - tb >= kTcLongItem) return kTcMinimaA * kTcGroupLong;
    return te - tb >= 2 * kTcMinimaA * kTcGroupShort ? kTcMinimaA * kTcGroupShort : 0;  // shorter: not worth it
}
constexpr int kTcK = 64;                          // bf16 per operand row (= one 128-byte swizzle row)
constexpr int kTcTileBytes = kTcBN * kTcK * 2;    // 16 KB: 128 rows x 128 B
constexpr size_t kTcSmemBytes = 1024 /*alignment slack*/ + 2 * kTcTileBytes + kTcStages * kTcTileBytes +
                                8 * kTcRingFloats * sizeof(float);

// byte offset of 16-byte chunk c (0..7) of row r inside a K-major SWIZZLE_128B tile of 128-byte rows
__host__ __device__ __forceinline__ uint32_t sw128_offset(int r, int c) {
    return static_cast<uint32_t>((r >> 3) * 1024 + (r & 7) * 128 + ((c ^ (r & 7)) << 4));
}

// ---- PTX wrappers (tcgen05 / mbarrier) -------------------------------------------------------
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// Polling wait with a short sleep between polls: a dozen warps spinning on mbarrier.try_wait starve the
// working warps of issue slots and shared-memory bandwidth (measured); only the MMA warp spins tightly.
__device__ __forceinline__ void mbar_wait_sleep(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    for (;;) {
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}\n"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
        if (done) break;
        __nanosleep(LIPFIT_TC_POLL_NS);
    }
}
// release / acquire on a shared-memory word (CTA scope): the flags of the detector <-> appender ring
__device__ __forceinline__ void st_release_s(volatile void* p, uint32_t v) {
    asm volatile("st.release.cta.shared::cta.u32 [%0], %1;" ::"r"(smem_u32(const_cast<void*>(p))), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t ld_acquire_s(const volatile void* p) {
    uint32_t v;
    asm volatile("ld.acquire.cta.shared::cta.u32 %0, [%1];" : "=r"(v) : "r"(smem_u32(const_cast<void*>(p))) : "memory");
    return v;
}
__device__ __forceinline__ void tc_fence_before() {
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tc_fence_after() {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tc_commit(uint64_t* bar) {  // arrives when all prior MMAs of this thread are done
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(
                     smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                       uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}\n" ::"r"(d_tmem),
        "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// K-major, SWIZZLE_128B, 128-byte rows: LBO = 1 (unused), SBO = 1024 B between 8-row groups, version 1
__device__ __forceinline__ uint64_t tc_smem_desc(uint32_t saddr) {
    return static_cast<uint64_t>((saddr & 0x3FFFFu) >> 4) | (1ull << 16) | (64ull << 32) | (1ull << 46) |
           (2ull << 61);
}
// kind::f16: D fp32, A/B bf16, both K-major, N = 128, M = 128
constexpr uint32_t kTcIdesc = (1u << 4) | (1u << 7) | (1u << 10) | ((kTcBN >> 3) << 17) | ((128u >> 4) << 24);

__device__ __forceinline__ void tc_ld32(uint32_t taddr, float (&v)[32]) {
    uint32_t r[32];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];\n"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]),
          "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]),
          "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]),
          "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr));
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tc_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// ---------------------------------------------------------------------------------------------
// Operand images
// ---------------------------------------------------------------------------------------------
// Centre: the mean of the first min(N, 4096) records, one block, fixed summation order (so that the
// whole call is deterministic).  Any centre is valid; a good one shrinks the error bound.
__global__ void __launch_bounds__(256)
knn_tc_centre_kernel(const float* __restrict__ X, int N, Xform xf, float* __restrict__ mu) {
    __shared__ double red[256];
    const int n = N < 4096 ? N : 4096;
    for (int j = 0; j < kMaxDim; ++j) {
        double s = 0.0;
        if (j < xf.d)
            for (int k = threadIdx.x; k < n; k += 256)
                s += static_cast<double>(xf.sw[j] * X[static_cast<size_t>(k) * xf.d + xf.perm[j]]);
        red[threadIdx.x] = s;
        __syncthreads();
        for (int o = 128; o > 0; o >>= 1) {
            if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
            __syncthreads();
        }
        if (threadIdx.x == 0) mu[j] = j < xf.d ? static_cast<float>(red[0] / n) : 0.f;
        __syncthreads();
    }
}

__device__ __forceinline__ void split2(float v, __nv_bfloat16& hi, __nv_bfloat16& lo) {
    hi = __float2bfloat16_rn(v);
    lo = __float2bfloat16_rn(v - __bfloat162float(hi));
}

__device__ __forceinline__ void store_row(unsigned char* tile, int r, const __nv_bfloat16 (&row)[kTcK]) {
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        uint4 w;
        const uint16_t* p = reinterpret_cast<const uint16_t*>(&row[8 * c]);
        w.x = p[0] | (static_cast<uint32_t>(p[1]) << 16);
        w.y = p[2] | (static_cast<uint32_t>(p[3]) << 16);
        w.z = p[4] | (static_cast<uint32_t>(p[5]) << 16);
        w.w = p[6] | (static_cast<uint32_t>(p[7]) << 16);
        *reinterpret_cast<uint4*>(tile + sw128_offset(r, c)) = w;
    }
}

// B image: record k -> tile k / 128, row k % 128.  Rows past N carry key = +huge.
__global__ void __launch_bounds__(256)
knn_tc_pack_b_kernel(const float* __restrict__ X, int N, int Npad, Xform xf, const float* __restrict__ mu,
                     unsigned char* __restrict__ img, uint32_t* __restrict__ stats) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    float amax = 0.f, x2f = 0.f;
    if (k < Npad) {
        __nv_bfloat16 row[kTcK];
#pragma unroll
        for (int j = 0; j < kTcK; ++j) row[j] = __float2bfloat16_rn(0.f);
        if (k < N) {
            const float* src = X + static_cast<size_t>(k) * xf.d;
            double s2 = 0.0;
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                float xc = 0.f;
                if (j < xf.d) {
                    const float xw = xf.sw[j] * src[xf.perm[j]];
                    amax = fmaxf(amax, fabsf(xw));
                    xc = xw - mu[j];
                }
                s2 += static_cast<double>(xc) * static_cast<double>(xc);
                __nv_bfloat16 hi, lo;
                split2(xc, hi, lo);
                if (j < xf.d) {
                    row[j] = hi;
                    row[xf.d + j] = lo;
                    row[2 * xf.d + j] = hi;
                }
            }
            x2f = static_cast<float>(s2);
            const __nv_bfloat16 h = __float2bfloat16_rn(x2f);
            const float r1 = x2f - __bfloat162float(h);
            const __nv_bfloat16 m = __float2bfloat16_rn(r1);
            const __nv_bfloat16 l = __float2bfloat16_rn(r1 - __bfloat162float(m));
            row[3 * xf.d] = h;
            row[3 * xf.d + 1] = m;
            row[3 * xf.d + 2] = l;
        } else {
            row[3 * xf.d] = __float2bfloat16_rn(3.0e38f);
        }
        store_row(img + static_cast<size_t>(k / kTcBN) * kTcTileBytes, k % kTcBN, row);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
        x2f = fmaxf(x2f, __shfl_xor_sync(0xffffffffu, x2f, o));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMax(stats + 0, __float_as_uint(amax));
        atomicMax(stats + 1, __float_as_uint(x2f));
    }
}

// A image: query slot q -> tile q / 128, row q % 128.  Slots past Q are all-zero rows.
__global__ void __launch_bounds__(256)
knn_tc_pack_a_kernel(const float* __restrict__ Xq, int Q, int Qp, Xform xf, const float* __restrict__ mu,
                     unsigned char* __restrict__ img) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= Qp) return;
    __nv_bfloat16 row[kTcK];
#pragma unroll
    for (int j = 0; j < kTcK; ++j) row[j] = __float2bfloat16_rn(0.f);
    if (q < Q) {
        const float* src = Xq + static_cast<size_t>(q) * xf.d;
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            float qc = 0.f;
            if (j < xf.d) qc = xf.sw[j] * src[xf.perm[j]] - mu[j];
            __nv_bfloat16 hi, lo;
            split2(-2.f * qc, hi, lo);
            if (j < xf.d) {
                row[j] = hi;
                row[xf.d + j] = hi;
                row[2 * xf.d + j] = lo;
            }
        }
        row[3 * xf.d] = row[3 * xf.d + 1] = row[3 * xf.d + 2] = __float2bfloat16_rn(1.f);
    }
    store_row(img + static_cast<size_t>(q / 128) * kTcTileBytes, q % 128, row);
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// Selection kernel
// ---------------------------------------------------------------------------------------------
struct KnnTcArgs {
    const unsigned char* Aimg;  // [Qp/128] tiles of 128 query rows
    const unsigned char* Bimg;  // [ntilesB] tiles of 128 data rows
    int ntilesB;
    int ksteps;                 // K steps (16 bf16 each) that hold non-zero operand columns
    KnnArgs k;                  // pools, schedule (query blocks of kTcQueries), N, Q, ksel, P
};

// min of 32 values as a depth-4 tree of 3-input minima (FMNMX3)
__device__ __forceinline__ float tc_min32(const float (&v)[32]) {
    float t[11];
#pragma unroll
    for (int i = 0; i < 10; ++i) t[i] = fminf(fminf(v[3 * i], v[3 * i + 1]), v[3 * i + 2]);
    t[10] = fminf(v[30], v[31]);
    const float u0 = fminf(fminf(t[0], t[1]), t[2]), u1 = fminf(fminf(t[3], t[4]), t[5]);
    const float u2 = fminf(fminf(t[6], t[7]), t[8]), u3 = fminf(t[9], t[10]);
    return fminf(fminf(u0, u1), fminf(u2, u3));
}

__global__ void __launch_bounds__(kTcThreads, 1)
knn_tc_select_kernel(const KnnTcArgs g) {
    extern __shared__ unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t a_full, a_empty, b_full[kTcStages], b_empty[kTcStages], acc_full[2][2],
        acc_empty[2][2];
    __shared__ __align__(8) unsigned long long tau_s[8][32];  // (item << 32 | tau bits) published by the appenders
    __shared__ volatile uint32_t head_s[8], tail_s[8];  // ring counters (messages written / consumed)
    __shared__ volatile int seed_s[8];                  // item whose phase A minima are complete
    __shared__ uint32_t s_tmem;
    // 1024-byte aligned carve-up (SWIZZLE_128B atoms are 1024 B)
    const uint32_t raw = smem_u32(smem_raw);
    unsigned char* base = smem_raw + ((1024u - (raw & 1023u)) & 1023u);
    unsigned char* sA = base;                                // 2 tiles
    unsigned char* sB = sA + 2 * kTcTileBytes;               // kTcStages tiles
    float* sR = reinterpret_cast<float*>(sB + kTcStages * kTcTileBytes);  // 8 rings of kTcRing row messages

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const KnnArgs& a = g.k;
    if (threadIdx.x == 0) {
        mbar_init(&a_full, 1);
        mbar_init(&a_empty, 2);  // both MMA issuers
        for (int s = 0; s < kTcStages; ++s) {
            mbar_init(&b_full[s], 1);
            mbar_init(&b_empty[s], 2);
        }
        for (int h = 0; h < 2; ++h)
            for (int b = 0; b < 2; ++b) {
                mbar_init(&acc_full[h][b], 1);
                mbar_init(&acc_empty[h][b], 4);  // the 4 detector warps of the half
            }
        for (int w = 0; w < 8; ++w) {
            head_s[w] = 0;
            tail_s[w] = 0;
            seed_s[w] = -1;
        }
        mbar_fence_init();
    }
    if (warp == 8) {  // the whole warp allocates all 512 TMEM columns of this SM
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                         smem_u32(&s_tmem)),
                     "r"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    if (threadIdx.x < 256) tau_s[threadIdx.x >> 5][threadIdx.x & 31] = 0xFFFFFFFF00000000ull;  // no item yet
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = s_tmem;

    const int nitems = a.nfull + a.ntail * a.T;
    const int chunk_tiles = a.chunk / kTcBN;
    // item -> (query block, chunk, B tile range)
    auto decode = [&](int item, int& qb, int& ch, int& tb, int& te) {
        if (item < a.nfull) {
            qb = item;
            ch = 0;
            tb = 0;
            te = g.ntilesB;
        } else {
            const int t = item - a.nfull;
            qb = a.nfull + t / a.T;
            ch = t - (qb - a.nfull) * a.T;
            tb = ch * chunk_tiles;
            te = min(g.ntilesB, tb + chunk_tiles);
        }
    };

    if (warp == 8) {
        // ================= TMA producer =================
        if (lane == 0) {
            uint32_t gB = 0, it = 0;
            for (int item = blockIdx.x; item < nitems; item += gridDim.x, ++it) {
                int qb, ch, tb, te;
                decode(item, qb, ch, tb, te);
                mbar_wait_sleep(&a_empty, (it & 1u) ^ 1u);
                mbar_arrive_expect_tx(&a_full, 2 * kTcTileBytes);
                bulk_g2s(sA, g.Aimg + static_cast<size_t>(qb) * 2 * kTcTileBytes, 2 * kTcTileBytes, &a_full);
                const int nA = tc_tiles_a(tb, te, a.ksel);
                for (int vt = -nA; vt < te - tb; ++vt, ++gB) {  // seeding tiles first, then the sweep
                    const int t = tb + (vt < 0 ? vt + nA : vt);
                    const uint32_t s = gB % kTcStages, u = gB / kTcStages;
                    mbar_wait_sleep(&b_empty[s], (u & 1u) ^ 1u);
                    mbar_arrive_expect_tx(&b_full[s], kTcTileBytes);
                    bulk_g2s(sB + s * kTcTileBytes, g.Bimg + static_cast<size_t>(t) * kTcTileBytes,
                             kTcTileBytes, &b_full[s]);
                }
            }
        }
    } else if (warp == 9 || warp == 18) {
        // ================= MMA issuers: one thread per query half =================
        // Two issuers so that a half whose detectors are held up (pushes, a full ring) does not block the
        // other half's accumulator stages; they share the B ring and drift at most kTcStages tiles apart.
        if (lane == 0) {
            const int h = warp == 9 ? 0 : 1;
            uint32_t gB = 0, it = 0;
            const uint64_t ad = tc_smem_desc(smem_u32(sA + h * kTcTileBytes));
            for (int item = blockIdx.x; item < nitems; item += gridDim.x, ++it) {
                int qb, ch, tb, te;
                decode(item, qb, ch, tb, te);
                mbar_wait(&a_full, it & 1u);
                tc_fence_after();
                const int ntiles = te - tb + tc_tiles_a(tb, te, a.ksel);
                for (int t = 0; t < ntiles; ++t, ++gB) {
                    const uint32_t s = gB % kTcStages, u = gB / kTcStages;
                    const uint32_t b = gB & 1u, ua = gB >> 1;
                    mbar_wait(&b_full[s], u & 1u);
                    mbar_wait(&acc_empty[h][b], (ua & 1u) ^ 1u);
                    tc_fence_after();
                    const uint64_t bdesc = tc_smem_desc(smem_u32(sB + s * kTcTileBytes));
                    const uint32_t dcol = tmem + (h * 2 + b) * kTcBN;
#pragma unroll
                    for (int k = 0; k < kTcK / 16; ++k)  // 32 bytes (16 bf16) per K step: +2 in the address field
                        if (k < g.ksteps) tc_mma(dcol, ad + 2 * k, bdesc + 2 * k, kTcIdesc, k > 0 ? 1u : 0u);
                    tc_commit(&acc_full[h][b]);
                    tc_commit(&b_empty[s]);
                }
                tc_commit(&a_empty);
            }
        }
    } else if (warp < 8) {
        // ================= detector warps: h = query half, quad = TMEM lane quadrant =================
        // They only FIND blocks of 32 x 32 keys that contain a key below some query's threshold and hand
        // those blocks to their appender warp through a shared-memory ring, so the tensor pipe never waits
        // for an append or a compaction (both are latency-bound: ~800 and ~6000 cycles per event).
        const int h = warp >> 2, quad = warp & 3;
        float* ring = sR + warp * kTcRingFloats;
        uint32_t gB = 0, head = 0, hslot = 0, tail_seen = 0;
        // room for n more messages (the appender's tail counter only grows)
        auto reserve = [&](uint32_t n) {
            while (head + n - tail_seen > static_cast<uint32_t>(kTcRing)) {
                tail_seen = ld_acquire_s(&tail_s[warp]);
                if (head + n - tail_seen > static_cast<uint32_t>(kTcRing)) __nanosleep(LIPFIT_TC_POLL_NS);
            }
        };
        auto publish = [&](uint32_t n) {
            head += n;
            hslot += n;
            if (hslot >= static_cast<uint32_t>(kTcRing)) hslot -= kTcRing;
            __syncwarp();
            if (lane == 0) st_release_s(&head_s[warp], head);
        };
        // the rows `hm` of a 32 x 32 block (thread = row) go to the appender, one message each
        auto push = [&](const float (&v)[32], unsigned hm, int kbase) {
            const uint32_t n = __popc(hm);
            reserve(n);
            if ((hm >> lane) & 1u) {
                uint32_t sl = hslot + __popc(hm & ((1u << lane) - 1u));
                if (sl >= static_cast<uint32_t>(kTcRing)) sl -= kTcRing;
                float4* p = reinterpret_cast<float4*>(ring + sl * kTcRowFloats);
#pragma unroll
                for (int c = 0; c < 8; ++c) p[c] = make_float4(v[4 * c], v[4 * c + 1], v[4 * c + 2], v[4 * c + 3]);
                *reinterpret_cast<int2*>(p + 8) = make_int2(kbase, lane);
            }
            publish(n);
        };
        for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
            int qb, ch, tb, te;
            decode(item, qb, ch, tb, te);
            const int qslot = qb * kTcQueries + h * 128 + quad * 32 + lane;
            float tau = qslot < a.Q ? 1.0e38f : __int_as_float(0xff800000);  // real keys are far below 1e38
            const int nA = tc_tiles_a(tb, te, a.ksel);
            if (nA) {  // phase A: group minima of the first tiles, [row][kTcMinimaA + 1] over the drained ring
                while (ld_acquire_s(&tail_s[warp]) != head) __nanosleep(LIPFIT_TC_POLL_NS);
                tail_seen = head;
                float gm = __int_as_float(0x7f800000);
                const int grp = nA / kTcMinimaA;
                for (int vt = 0, ing = 0, ng = 0; vt < nA; ++vt, ++gB) {
                    const uint32_t b = gB & 1u, ua = gB >> 1;
                    mbar_wait_sleep(&acc_full[h][b], ua & 1u);
                    tc_fence_after();
                    const uint32_t trow = tmem + (static_cast<uint32_t>(quad * 32) << 16) + (h * 2 + b) * kTcBN;
                    float va[32];  // one buffer, rolled loop: ptxas spills a buffer in any unrolled form
#pragma unroll 1
                    for (int cb = 0; cb < 4; ++cb) {
                        tc_ld32(trow + 32 * cb, va);
                        tc_ld_wait();
                        gm = fminf(gm, tc_min32(va));
                    }
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&acc_empty[h][b]);
                    if (++ing == grp) {
                        ring[lane * (kTcMinimaA + 1) + ng++] = gm;
                        gm = __int_as_float(0x7f800000);
                        ing = 0;
                    }
                }
                __syncwarp();
                if (lane == 0) st_release_s(&seed_s[warp], static_cast<uint32_t>(item));
                // the sweep starts from the appender's seeded threshold (and the ring is free again)
                for (;;) {
                    const unsigned long long ts = *reinterpret_cast<volatile unsigned long long*>(&tau_s[warp][lane]);
                    if (static_cast<uint32_t>(ts >> 32) == static_cast<uint32_t>(item)) break;
                    __nanosleep(200);
                }
                __syncwarp();
            }
            for (int t = tb; t < te; ++t, ++gB) {
                const uint32_t b = gB & 1u, ua = gB >> 1;
                {  // adopt the appender's latest threshold for this item (stale values only cost extra pushes)
                    const unsigned long long ts = *reinterpret_cast<volatile unsigned long long*>(&tau_s[warp][lane]);
                    if (static_cast<uint32_t>(ts >> 32) == static_cast<uint32_t>(item))
                        tau = fminf(tau, __uint_as_float(static_cast<uint32_t>(ts)));
                }
                mbar_wait_sleep(&acc_full[h][b], ua & 1u);
                tc_fence_after();
                const uint32_t trow = tmem + (static_cast<uint32_t>(quad * 32) << 16) + (h * 2 + b) * kTcBN;
                // Software pipeline over the four 32-column blocks: the TMEM load of block cb+1 is in flight
                // while block cb is reduced / pushed (two register buffers).
                auto process = [&](const float (&v)[32], int cb) {
                    const float m = tc_min32(v);
                    const unsigned hm = __ballot_sync(0xffffffffu, m < tau);
                    if (hm) push(v, hm, t * kTcBN + cb * 32);
                };
                float va[32], vb[32];
                tc_ld32(trow, va);
                tc_ld_wait();
                tc_ld32(trow + 32, vb);
                process(va, 0);
                tc_ld_wait();
                tc_ld32(trow + 64, va);
                process(vb, 1);
                tc_ld_wait();
                tc_ld32(trow + 96, vb);
                process(va, 2);
                tc_ld_wait();
                tc_fence_before();  // all four blocks are in registers: hand the TMEM stage back
                __syncwarp();
                if (lane == 0) mbar_arrive(&acc_empty[h][b]);
                process(vb, 3);
            }
            // end of item: the appender writes fill / tau and moves on
            reserve(1);
            if (lane == 0) *reinterpret_cast<int2*>(ring + hslot * kTcRowFloats + 32) = make_int2(-1, 0);
            publish(1);
        }
    } else if (warp < 18) {
        // ================= appender warps: own the thresholds and pools of the paired detector's queries ====
        const int aw = warp - 10;  // paired detector warp
        const int h = aw >> 2, quad = aw & 3;
        const float* ring = sR + aw * kTcRingFloats;
        uint32_t tail = 0, tslot = 0, head_seen = 0;
        for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
            int qb, ch, tb, te;
            decode(item, qb, ch, tb, te);
            const int qslot = qb * kTcQueries + h * 128 + quad * 32 + lane;
            float tau = qslot < a.Q ? 1.0e38f : __int_as_float(0xff800000);
            int fill = 0;
            const size_t slot = knn_pool_slot(qslot, ch, a.Qp, a.Qtp, a.nfullq);
            int2* pool = a.pool + slot * a.P;
            if (tc_tiles_a(tb, te, a.ksel)) {
                // phase A: row L's kTcMinimaA group minima sit at ring[L][.], one per lane per 32.  tau = the
                // next float above the ksel-th smallest, so that at least ksel data pass the strict
                // `key < tau` test of the sweep.
                while (ld_acquire_s(&seed_s[aw]) != static_cast<uint32_t>(item)) __nanosleep(LIPFIT_TC_POLL_NS);
                uint32_t seed = 0;
#pragma unroll 2
                for (int L = 0; L < 32; ++L) {
                    uint32_t key[kTcMinimaA / 32];
#pragma unroll
                    for (int j = 0; j < kTcMinimaA / 32; ++j)
                        key[j] = f2key(ring[L * (kTcMinimaA + 1) + j * 32 + lane]);
                    int need;
                    const uint32_t kth = knn_rank_select<kTcMinimaA / 32>(key, a.ksel, need);
                    if (lane == L) seed = kth;
                }
                __syncwarp();
                tau = fminf(tau, key2f(seed + 1u));
                tau_s[aw][lane] = (static_cast<unsigned long long>(static_cast<uint32_t>(item)) << 32) |
                                  __float_as_uint(tau);
            }
            for (;;) {
                if (head_seen == tail) {
                    while ((head_seen = ld_acquire_s(&head_s[aw])) == tail) __nanosleep(LIPFIT_TC_POLL_NS);
                }
                const float* p = ring + tslot * kTcRowFloats;
                const int2 hd = *reinterpret_cast<const int2*>(p + 32);  // (first datum index, row)
                const float val = p[lane];                               // lane = column
                ++tail;
                if (++tslot == static_cast<uint32_t>(kTcRing)) tslot = 0;
                if (hd.x < 0) {
                    __syncwarp();
                    if (lane == 0) st_release_s(&tail_s[aw], tail);
                    break;
                }
                const int L = hd.y;
                float tauL = __shfl_sync(0xffffffffu, tau, L);
                int fillL = __shfl_sync(0xffffffffu, fill, L);
                int2* poolL = pool + static_cast<ptrdiff_t>(L - lane) * a.P;  // consecutive lanes = consecutive slots
                if (fillL >= a.ksel + kTcSlack) {  // compact (warp-cooperative radix select): lowers tau
                    __syncwarp();
                    tauL = knn_compact(poolL, fillL, a.ksel, nullptr, lane);
                    fillL = a.ksel;
                    if (lane == L) tau = tauL;
                    // publish the lowered threshold for the detector
                    tau_s[aw][lane] = (static_cast<unsigned long long>(static_cast<uint32_t>(item)) << 32) |
                                      __float_as_uint(tau);
                }
                const bool hit = val < tauL;
                const unsigned bm = __ballot_sync(0xffffffffu, hit);
                if (hit) poolL[fillL + __popc(bm & ((1u << lane) - 1u))] = make_int2(__float_as_int(val), hd.x + lane);
                if (lane == L) fill = fillL + __popc(bm);
                if (lane == 0) st_release_s(&tail_s[aw], tail);  // every lane's read of the message fed the ballot above
            }
            a.fill[slot] = fill;
            a.tau[slot] = tau;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 8)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512));
}

int knn_tc_slots(const Ctx& c) { return c.num_sms; }

int launch_knn_tc_select(const Ctx& c, const float* X, const float* Xq, KnnArgs& a, float* mu_dev,
                         uint32_t* stats) {
    const int ntilesB = (a.N + kTcBN - 1) / kTcBN;
    const int Npad = ntilesB * kTcBN;
    Workspace wa, wb;
    int rc;
    if ((rc = wa.alloc(static_cast<size_t>(a.Qp) * kTcK * 2, c.stream))) return rc;
    if ((rc = wb.alloc(static_cast<size_t>(Npad) * kTcK * 2, c.stream))) return rc;
    knn_tc_centre_kernel<<<1, 256, 0, c.stream>>>(X, a.N, a.xf, mu_dev);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    knn_tc_pack_b_kernel<<<(Npad + 255) / 256, 256, 0, c.stream>>>(X, a.N, Npad, a.xf, mu_dev,
                                                                   wb.as<unsigned char>(), stats);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    knn_tc_pack_a_kernel<<<(a.Qp + 255) / 256, 256, 0, c.stream>>>(Xq, a.Q, a.Qp, a.xf, mu_dev,
                                                                   wa.as<unsigned char>());
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    KnnTcArgs g{};
    g.Aimg = wa.as<unsigned char>();
    g.Bimg = wb.as<unsigned char>();
    g.ntilesB = ntilesB;
    g.ksteps = (3 * a.xf.d + 3 + 15) / 16;
    g.k = a;
    LIPFIT_CUDA(cudaFuncSetAttribute(knn_tc_select_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     static_cast<int>(kTcSmemBytes)));
    const long long nitems = static_cast<long long>(a.nfull) + static_cast<long long>(a.ntail) * a.T;
    const int grid = static_cast<int>(nitems < c.num_sms ? nitems : c.num_sms);
    KernelTimer kt(TK_KNN_SELECT, c.stream);
    knn_tc_select_kernel<<<grid, kTcThreads, kTcSmemBytes, c.stream>>>(g);
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

}  // namespace lipfit
