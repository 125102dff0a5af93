// bounds.cu -- step a2: fused distance + running min/max.
//   upper[q] = min_k (y^k + M D^u),  lower[q] = max_k (y^k - M D^l),  g = (upper+lower)/2
// Eq.(2),(3) PAPER.md:103-116 with the distance of Eq.(4) PAPER.md:142.  The Q x N distance matrix
// of the paper's cdist+topk composition is never formed.
//
// Shape of the kernel: every thread keeps R queries (R x D coordinates) and their 2R running
// extrema in registers; packed data records stream through shared memory in double-buffered tiles
// filled by the TMA engine (cp.async.bulk + mbarrier) and are read with broadcast LDS.128, so one
// 16-byte shared load feeds R pairs.  Work is cut into (query block, data chunk) tiles spread over a
// persistent grid; with more than one chunk the partial extrema meet through atomicMin/atomicMax on
// order-preserving integer keys (min/max are order independent, so the result is deterministic).
#include "kernels.h"

namespace lipfit {

struct BoundsArgs {
    const float* rec;
    const float* Xq;
    const float* centre;  // translation applied to the records (launch_prepack) or NULL
    float* upper;
    float* lower;
    float* g;
    uint32_t* keyU;
    uint32_t* keyL;
    int N, Q, d, rf, vslot;
    int nqb, nch, chunk;
    float M;
    Xform xf;
};

template <int THREADS, int R>
__device__ __forceinline__ int query_index(int qb, int r, int Q) {
    int qi = (qb * R + r) * THREADS + static_cast<int>(threadIdx.x);
    return qi;
}

// Core = compile-time description of the pair arithmetic:
//   Core::D      packed coordinates held per query
//   Core::RF     floats per record (0 = runtime a.rf), Core::VSLOT value slot (-1 = runtime)
//   Core::pair(q, rec_regs, ff, M, hi, lo)
template <int NORM, int DU, int DC>
struct SpecCore {
    static constexpr int D = DU + DC;
    static constexpr int RF = record_floats(D);
    static constexpr int VSLOT = D;
    static constexpr bool kGeneric = false;
    static constexpr bool kFold = false;
    static __device__ __forceinline__ float query_term(const float*) { return 0.f; }
    static __device__ __forceinline__ void pair(const float* q, const float* x, const FreeFlags&,
                                                float M, float& hi, float& lo) {
        float au, al;
        PairAcc<NORM, DU, DC>::run(q, x, au, al);
        float y = x[VSLOT];
        if (NORM == 2 && DC == 0) {
            float dist = fast_sqrt(au);
            hi = fmaf(M, dist, y);
            lo = fmaf(-M, dist, y);
        } else {
            hi = fmaf(M, PairAcc<NORM, DU, DC>::finish(au), y);
            lo = fmaf(-M, PairAcc<NORM, DU, DC>::finish(al), y);
        }
    }
};

// Weighted L1 with constrained coordinates, folded (the coordinates arrive PRE-MULTIPLIED BY M).  With
// delta = q - x per coordinate, sq / sx = sum of the constrained coordinates of the query / the datum:
//   (delta)_+ = max(q, x) - x   and   (-delta)_+ = max(q, x) - q        (exact identities)
//   T     = sum_free |delta_j| + sum_constr max(q_j, x_j)
//   M D^u = T - sx,   M D^l = T - sq
//   hi = y + M D^u = (y - sx) + T,      lo = y - M D^l = (2 y - sx) - hi + sq = c' - hi + sq
// The record carries y - sx in its value slot (it starts the accumulation chain) and c' = 2 y - sx; sq is constant
// per query and is added AFTER the running maximum.  Per pair: unconstrained coordinate = sub + add(|.|) on the
// FMA pipe, constrained coordinate = ONE max on the ALU pipe + one add (instead of sub + relu + add), + one sub
// for lo: 7 FMA-pipe + 2 ALU-pipe operations for config 2's shape, plus the min / max of the running extrema
// (the plain form of SURVEY.md: 12 + 6).  (Valid for L1 only: no square root stands between the sums.  Rounding:
// max(q, x) - x and c' - hi cancel terms of magnitude M |x|, so both bounds carry a few 2^-24 M |x| -- inside the
// budget of DESIGN.md §6, measured in the tests; api.cu translates the data to the first datum to keep |x| small.)
template <int DU, int DC>
struct FoldL1Core {
    static constexpr int D = DU + DC;
    static constexpr int RF = record_floats(D + 1);
    static constexpr int VSLOT = D;
    static constexpr int CSLOT = D + 1;
    static constexpr bool kGeneric = false;
    static constexpr bool kFold = true;
    static __device__ __forceinline__ void pair(const float* q, const float* x, const FreeFlags&, float,
                                                float& hi, float& lo) {
        float a = x[VSLOT];  // y - sx
#pragma unroll
        for (int j = 0; j < DU; ++j) a += fabsf(q[j] - x[j]);
#pragma unroll
        for (int j = DU; j < D; ++j) a += fmaxf(q[j], x[j]);
        hi = a;
        lo = x[CSLOT] - a;
    }
    static __device__ __forceinline__ float query_term(const float* q) {
        float sq = 0.f;
#pragma unroll
        for (int j = DU; j < D; ++j) sq += q[j];
        return sq;
    }
};

template <int NORM, int DP>
struct GenCore {
    static constexpr int D = DP;
    static constexpr int RF = DP + 4;
    static constexpr int VSLOT = DP;
    static constexpr bool kGeneric = true;
    static constexpr bool kFold = false;
    static __device__ __forceinline__ float query_term(const float*) { return 0.f; }
    static __device__ __forceinline__ void pair(const float* q, const float* x, const FreeFlags& ff,
                                                float M, float& hi, float& lo) {
        float au, al;
        if (DP >= 16) PairAccChunked<NORM, DP>::run(q, x, ff, au, al);  // d > 8: chunks under uniform conditions
        else PairAccGeneric<NORM, DP>::run(q, x, ff, au, al);
        float y = x[VSLOT];
        hi = fmaf(M, PairAccGeneric<NORM, DP>::finish(au), y);
        lo = fmaf(-M, PairAccGeneric<NORM, DP>::finish(al), y);
    }
};

template <int RF>
__device__ __forceinline__ void load_record(const float* s, float* x) {
#pragma unroll
    for (int c = 0; c < RF / 4; ++c) {
        float4 v = reinterpret_cast<const float4*>(s)[c];
        x[4 * c + 0] = v.x;
        x[4 * c + 1] = v.y;
        x[4 * c + 2] = v.z;
        x[4 * c + 3] = v.w;
    }
}

template <int RF>
__host__ __device__ constexpr int tile_records() {
    return RF <= 8 ? 512 : (RF <= 16 ? 256 : (RF <= 24 ? 128 : 96));
}

template <class Core, int R, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
bounds_kernel(const BoundsArgs a, const FreeFlags ff) {
    constexpr int D = Core::D;
    constexpr int RF = Core::RF;
    constexpr int TILE = tile_records<RF>();
    __shared__ __align__(128) float sbuf[2 * TILE * RF];
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

        // ---- queries of this block -> registers, transformed on the fly (Xform) ----
        float q[R][D];
        float U[R], L[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            int qi = (qb * R + r) * THREADS + static_cast<int>(threadIdx.x);
            qi = qi < a.Q ? qi : a.Q - 1;
            const float* src = a.Xq + static_cast<size_t>(qi) * a.d;
#pragma unroll
            for (int j = 0; j < D; ++j) {
                if (Core::kGeneric) {
                    q[r][j] = (j < a.d) ? a.xf.sw[j] * __ldg(src + a.xf.perm[j]) : 0.f;
                } else {
                    const int o = a.xf.perm[j];
                    q[r][j] = a.xf.sw[j] * (a.centre ? __ldg(src + o) - __ldg(a.centre + o) : __ldg(src + o));
                }
            }
            U[r] = __int_as_float(0x7f800000);
            L[r] = __int_as_float(0xff800000);
        }

        const int begin = ch * a.chunk;
        const int end = min(a.N, begin + a.chunk);
        RecordStream<TILE> rs(a.rec, RF, begin, end, sbuf, bars, &phase);
        for (int t = 0; t < rs.ntiles; ++t) {
            const float* s = rs.acquire(t);
            const int n = rs.count(t);
            int j = 0;
            for (; j + 2 <= n; j += 2) {
                float xa[RF], xb[RF];
                load_record<RF>(s + j * RF, xa);
                load_record<RF>(s + (j + 1) * RF, xb);
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    float hia, loa, hib, lob;
                    Core::pair(q[r], xa, ff, a.M, hia, loa);
                    Core::pair(q[r], xb, ff, a.M, hib, lob);
                    U[r] = fminf(fminf(U[r], hia), hib);  // FMNMX3
                    L[r] = fmaxf(fmaxf(L[r], loa), lob);
                }
            }
            if (j < n) {
                float xa[RF];
                load_record<RF>(s + j * RF, xa);
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    float hia, loa;
                    Core::pair(q[r], xa, ff, a.M, hia, loa);
                    U[r] = fminf(U[r], hia);
                    L[r] = fmaxf(L[r], loa);
                }
            }
            rs.release(t);
        }

        // ---- results ----
#pragma unroll
        for (int r = 0; r < R; ++r) {
            int qi = (qb * R + r) * THREADS + static_cast<int>(threadIdx.x);
            if (Core::kFold) L[r] += Core::query_term(q[r]);  // the per-query constant of the folded lower bound
            if (qi < a.Q) {
                if (a.nch == 1) {
                    if (a.upper) a.upper[qi] = U[r];
                    if (a.lower) a.lower[qi] = L[r];
                    if (a.g) a.g[qi] = 0.5f * (U[r] + L[r]);
                } else {
                    atomicMin(a.keyU + qi, f2key(U[r]));
                    atomicMax(a.keyL + qi, f2key(L[r]));
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Packed-f32x2 version of the folded L1 bounds (sm_100 FADD2): a thread keeps RP PAIRS of queries as
// (q_r, q_r+1) register pairs; records arrive duplicated (x, x) so that one FADD2 forms the difference of
// both queries (free coordinates), one FADD2 accumulates both max(q, x) (constrained coordinates), one FADD2
// forms both lower candidates.  |.| has no packed form: the free coordinates are accumulated with two scalar
// FADD (|.| modifier).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 sub2(float2 a, float2 b) {  // a - b, one FADD2
    return __fadd2_rn(a, make_float2(-b.x, -b.y));
}

// Packed policies: D coordinates, RFL logical floats per record, pair2() -> both candidates of both queries,
// query_term2() -> per-query constants added to the lower bounds after the running maximum.
template <int DU, int DC>
struct PackedFoldL1 {
    static constexpr int D = DU + DC;
    static constexpr int RFL = record_floats(D + 1);
    static __device__ __forceinline__ void pair2(const float2* qq, const float2* x, float2& hi, float2& lo) {
        float2 acc = x[D];  // (y - sx, y - sx), see FoldL1Core
#pragma unroll
        for (int j = 0; j < DU; ++j) {
            const float2 dlt = sub2(qq[j], x[j]);
            acc.x += fabsf(dlt.x);
            acc.y += fabsf(dlt.y);
        }
#pragma unroll
        for (int j = DU; j < D; ++j)  // (delta)_+ = max(q, x) - x: the subtraction rides in the record
            acc = __fadd2_rn(acc, make_float2(fmaxf(qq[j].x, x[j].x), fmaxf(qq[j].y, x[j].y)));
        hi = acc;
        lo = sub2(x[D + 1], acc);  // c' - hi
    }
    static __device__ __forceinline__ float2 query_term2(const float2* qq) {
        float2 sq = make_float2(0.f, 0.f);
#pragma unroll
        for (int j = DU; j < D; ++j) {
            sq.x += qq[j].x;
            sq.y += qq[j].y;
        }
        return sq;
    }
};

// Weighted Linf with the coordinates pre-multiplied by M: the subtractions and the two final additions are
// FADD2, the maxima stay scalar (|.| and negation are free modifiers of FMNMX / FMNMX3):
//   s = max_free |delta_j|,  hi = y + max(s, delta_c..),  lo = y - max(s, -delta_c..).
template <int DU, int DC>
struct PackedLinf {
    static constexpr int D = DU + DC;
    static constexpr int RFL = record_floats(D);
    static __device__ __forceinline__ void pair2(const float2* qq, const float2* x, float2& hi, float2& lo) {
        // s = max_free |delta_j| as a chain of 3-input maxima that STARTS from |delta_0| (not from 0): n values
        // cost (n - 1) / 2 FMNMX3 -- 3 for config 3's 7 free coordinates instead of 4; an odd one out is folded
        // into the first constrained coordinate's pair of maxima (or a last 2-input maximum).
        float2 dl[D];
#pragma unroll
        for (int j = 0; j < D; ++j) dl[j] = sub2(qq[j], x[j]);
        float2 sm = make_float2(0.f, 0.f);  // (DU == 0: the constrained maxima start from 0, which is their relu)
        constexpr int NCH = DU >= 1 ? (DU - 1) / 2 : 0;     // full (a, b) pairs after the first value
        constexpr bool LEFT = DU >= 1 && ((DU - 1) % 2 == 1);  // one free value left over
        if (DU >= 1) sm = make_float2(fabsf(dl[0].x), fabsf(dl[0].y));
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
            const float2 a = dl[1 + 2 * c], b = dl[2 + 2 * c];
            sm.x = fmaxf(fmaxf(sm.x, fabsf(a.x)), fabsf(b.x));  // FMNMX3
            sm.y = fmaxf(fmaxf(sm.y, fabsf(a.y)), fabsf(b.y));
        }
        float2 pu = sm, pl = sm;
        if (LEFT) {
            const float2 e = dl[DU - 1];
            if (DC >= 1) {  // s >= 0 already: max(s, relu(d)) == max(s, d)
                pu.x = fmaxf(fmaxf(pu.x, fabsf(e.x)), dl[DU].x);
                pu.y = fmaxf(fmaxf(pu.y, fabsf(e.y)), dl[DU].y);
                pl.x = fmaxf(fmaxf(pl.x, fabsf(e.x)), -dl[DU].x);
                pl.y = fmaxf(fmaxf(pl.y, fabsf(e.y)), -dl[DU].y);
            } else {
                pu.x = pl.x = fmaxf(pu.x, fabsf(e.x));
                pu.y = pl.y = fmaxf(pu.y, fabsf(e.y));
            }
        }
#pragma unroll
        for (int j = DU + ((LEFT && DC >= 1) ? 1 : 0); j < D; ++j) {
            pu.x = fmaxf(pu.x, dl[j].x);
            pu.y = fmaxf(pu.y, dl[j].y);
            pl.x = fmaxf(pl.x, -dl[j].x);
            pl.y = fmaxf(pl.y, -dl[j].y);
        }
        hi = __fadd2_rn(x[D], pu);
        lo = sub2(x[D], pl);
    }
    static __device__ __forceinline__ float2 query_term2(const float2*) { return make_float2(0.f, 0.f); }
};

// Weighted L2 with the coordinates pre-multiplied by M: subtractions and squared accumulations are
// FADD2 / FFMA2, the positive / negative parts stay scalar FMNMX, one MUFU.SQRT per bound and query.
template <int DU, int DC>
struct PackedL2 {
    static constexpr int D = DU + DC;
    static constexpr int RFL = record_floats(D);
    static __device__ __forceinline__ void pair2(const float2* qq, const float2* x, float2& hi, float2& lo) {
        float2 sm = make_float2(0.f, 0.f);
#pragma unroll
        for (int j = 0; j < DU; ++j) {
            const float2 dlt = sub2(qq[j], x[j]);
            sm = __ffma2_rn(dlt, dlt, sm);
        }
        if (DC == 0) {  // symmetric: both bounds share the distance
            const float2 dist = make_float2(fast_sqrt(sm.x), fast_sqrt(sm.y));
            hi = __fadd2_rn(x[D], dist);
            lo = sub2(x[D], dist);
            return;
        }
        float2 pu = sm, pl = sm;
#pragma unroll
        for (int j = DU; j < D; ++j) {
            const float2 dlt = sub2(qq[j], x[j]);
            const float2 r = make_float2(fmaxf(dlt.x, 0.f), fmaxf(dlt.y, 0.f));
            const float2 m = make_float2(fminf(dlt.x, 0.f), fminf(dlt.y, 0.f));
            pu = __ffma2_rn(r, r, pu);
            pl = __ffma2_rn(m, m, pl);
        }
        hi = __fadd2_rn(x[D], make_float2(fast_sqrt(pu.x), fast_sqrt(pu.y)));
        lo = sub2(x[D], make_float2(fast_sqrt(pl.x), fast_sqrt(pl.y)));
    }
    static __device__ __forceinline__ float2 query_term2(const float2*) { return make_float2(0.f, 0.f); }
};

template <class P2, int RP, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
bounds_packed_kernel(const BoundsArgs a) {
    constexpr int D = P2::D;
    constexpr int RFL = P2::RFL;               // logical floats per record
    constexpr int RF = 2 * RFL;                // physical (duplicated)
    constexpr int TILE = tile_records<RF>();
    constexpr int R = 2 * RP;
    __shared__ __align__(128) float sbuf[2 * TILE * RF];
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
        float2 q[RP][D], U[RP], L[RP];
#pragma unroll
        for (int rp = 0; rp < RP; ++rp) {
            int q0 = (qb * R + 2 * rp) * THREADS + static_cast<int>(threadIdx.x);
            int q1 = q0 + THREADS;
            q0 = q0 < a.Q ? q0 : a.Q - 1;
            q1 = q1 < a.Q ? q1 : a.Q - 1;
            const float* s0 = a.Xq + static_cast<size_t>(q0) * a.d;
            const float* s1 = a.Xq + static_cast<size_t>(q1) * a.d;
#pragma unroll
            for (int j = 0; j < D; ++j) {
                const int o = a.xf.perm[j];
                const float cj = a.centre ? __ldg(a.centre + o) : 0.f;  // x - 0 is exact
                q[rp][j] = make_float2(a.xf.sw[j] * (__ldg(s0 + o) - cj), a.xf.sw[j] * (__ldg(s1 + o) - cj));
            }
            U[rp] = make_float2(__int_as_float(0x7f800000), __int_as_float(0x7f800000));
            L[rp] = make_float2(__int_as_float(0xff800000), __int_as_float(0xff800000));
        }
        const int begin = ch * a.chunk;
        const int end = min(a.N, begin + a.chunk);
        RecordStream<TILE> rs(a.rec, RF, begin, end, sbuf, bars, &phase);
        for (int t = 0; t < rs.ntiles; ++t) {
            const float* s = rs.acquire(t);
            const int n = rs.count(t);
            int j = 0;
            for (; j + 2 <= n; j += 2) {
                float2 xa[RFL], xb[RFL];
#pragma unroll
                for (int c = 0; c < RF / 4; ++c) {
                    const float4 va = reinterpret_cast<const float4*>(s + j * RF)[c];
                    const float4 vb = reinterpret_cast<const float4*>(s + (j + 1) * RF)[c];
                    xa[2 * c] = make_float2(va.x, va.y);
                    xa[2 * c + 1] = make_float2(va.z, va.w);
                    xb[2 * c] = make_float2(vb.x, vb.y);
                    xb[2 * c + 1] = make_float2(vb.z, vb.w);
                }
#pragma unroll
                for (int rp = 0; rp < RP; ++rp) {
                    float2 hia, loa, hib, lob;
                    P2::pair2(q[rp], xa, hia, loa);
                    P2::pair2(q[rp], xb, hib, lob);
                    U[rp].x = fminf(fminf(U[rp].x, hia.x), hib.x);  // FMNMX3
                    U[rp].y = fminf(fminf(U[rp].y, hia.y), hib.y);
                    L[rp].x = fmaxf(fmaxf(L[rp].x, loa.x), lob.x);
                    L[rp].y = fmaxf(fmaxf(L[rp].y, loa.y), lob.y);
                }
            }
            if (j < n) {
                float2 xa[RFL];
#pragma unroll
                for (int c = 0; c < RF / 4; ++c) {
                    const float4 va = reinterpret_cast<const float4*>(s + j * RF)[c];
                    xa[2 * c] = make_float2(va.x, va.y);
                    xa[2 * c + 1] = make_float2(va.z, va.w);
                }
#pragma unroll
                for (int rp = 0; rp < RP; ++rp) {
                    float2 hia, loa;
                    P2::pair2(q[rp], xa, hia, loa);
                    U[rp].x = fminf(U[rp].x, hia.x);
                    U[rp].y = fminf(U[rp].y, hia.y);
                    L[rp].x = fmaxf(L[rp].x, loa.x);
                    L[rp].y = fmaxf(L[rp].y, loa.y);
                }
            }
            rs.release(t);
        }
#pragma unroll
        for (int rp = 0; rp < RP; ++rp) {
            const float2 sq = P2::query_term2(q[rp]);  // the per-query constant of the folded lower bound
            const float Uv[2] = {U[rp].x, U[rp].y}, Lv[2] = {L[rp].x + sq.x, L[rp].y + sq.y};
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int qi = (qb * R + 2 * rp + e) * THREADS + static_cast<int>(threadIdx.x);
                if (qi < a.Q) {
                    if (a.nch == 1) {
                        if (a.upper) a.upper[qi] = Uv[e];
                        if (a.lower) a.lower[qi] = Lv[e];
                        if (a.g) a.g[qi] = 0.5f * (Uv[e] + Lv[e]);
                    } else {
                        atomicMin(a.keyU + qi, f2key(Uv[e]));
                        atomicMax(a.keyL + qi, f2key(Lv[e]));
                    }
                }
            }
        }
    }
}

__global__ void __launch_bounds__(256)
bounds_finalize_kernel(const uint32_t* __restrict__ keyU, const uint32_t* __restrict__ keyL, int Q,
                       float* __restrict__ upper, float* __restrict__ lower, float* __restrict__ g) {
    int qi = blockIdx.x * blockDim.x + threadIdx.x;
    if (qi >= Q) return;
    float U = key2f(keyU[qi]);
    float L = key2f(keyL[qi]);
    if (upper) upper[qi] = U;
    if (lower) lower[qi] = L;
    if (g) g[qi] = 0.5f * (U + L);
}

int launch_bounds_finalize(const Ctx& c, const uint32_t* keyU, const uint32_t* keyL, int Q, float* upper,
                           float* lower, float* g) {
    bounds_finalize_kernel<<<(Q + 255) / 256, 256, 0, c.stream>>>(keyU, keyL, Q, upper, lower, g);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

// ---------------------------------------------------------------------------------------------
// Host dispatch
// ---------------------------------------------------------------------------------------------
namespace {

struct Variant {
    int norm, dU, dC;  // generic: dU = DP, dC = -1
    const char* name;
    RecLayout lay;
    // launches with the given R flavour (0 = big-R throughput kernel, 1 = small-R latency kernel)
    int (*launch)(const Ctx&, BoundsArgs&, const FreeFlags&, int flavour);
    bool padded_list = false;  // reached through bounds_xform() only (see kVariants)
};

template <class Core, int R, int THREADS, int MINB>
int launch_one(const Ctx& c, BoundsArgs& a, const FreeFlags& ff) {
    auto kern = bounds_kernel<Core, R, THREADS, MINB>;
    int occ = 0;
    LIPFIT_CUDA(occupancy_of(&occ, kern, THREADS, 0));
    if (occ < 1) occ = 1;
    const int slots = c.num_sms * occ;
    constexpr int TILE = tile_records<Core::RF>();
    a.nqb = (a.Q + THREADS * R - 1) / (THREADS * R);
    // Cut the data into chunks until there are >= 16 tiles per resident CTA (tail effect <= ~6 %),
    // but keep a chunk at least 4 smem tiles long.
    int want = (16 * slots + a.nqb - 1) / a.nqb;
    int max_ch = (a.N + 4 * TILE - 1) / (4 * TILE);
    int nch = want < 1 ? 1 : want;
    if (nch > max_ch) nch = max_ch;
    if (nch < 1) nch = 1;
    int chunk = (a.N + nch - 1) / nch;
    chunk = ((chunk + TILE - 1) / TILE) * TILE;
    nch = (a.N + chunk - 1) / chunk;
    a.nch = nch;
    a.chunk = chunk;

    Workspace keys;
    if (nch > 1) {
        int rc = keys.alloc(sizeof(uint32_t) * 2 * static_cast<size_t>(a.Q), c.stream);
        if (rc) return rc;
        a.keyU = keys.as<uint32_t>();
        a.keyL = a.keyU + a.Q;
        LIPFIT_CUDA(cudaMemsetAsync(a.keyU, 0xFF, sizeof(uint32_t) * a.Q, c.stream));
        LIPFIT_CUDA(cudaMemsetAsync(a.keyL, 0x00, sizeof(uint32_t) * a.Q, c.stream));
    }
    long long ntiles = static_cast<long long>(a.nqb) * nch;
    int grid = static_cast<int>(ntiles < slots ? ntiles : slots);
    KernelTimer kt(TK_BOUNDS, c.stream);
    kern<<<grid, THREADS, 0, c.stream>>>(a, ff);
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    if (nch > 1) {
        bounds_finalize_kernel<<<(a.Q + 255) / 256, 256, 0, c.stream>>>(a.keyU, a.keyL, a.Q, a.upper,
                                                                      a.lower, a.g);
        ++g_launches;
        LIPFIT_CUDA(cudaGetLastError());
    }
    return LIPFIT_OK;
}

template <int NORM, int DU, int DC>
int launch_spec(const Ctx& c, BoundsArgs& a, const FreeFlags& ff, int flavour) {
    using Core = SpecCore<NORM, DU, DC>;
    constexpr int D = DU + DC;
    constexpr int RBIG = (D <= 5) ? 8 : 4;
    if (flavour == 0) return launch_one<Core, RBIG, 128, 2>(c, a, ff);
    return launch_one<Core, 1, 128, 4>(c, a, ff);
}

// throughput flavour of the packed f32x2 kernels: duplicated records (the layout says so)
// (Measured alternatives on config 2, profiles/r2_profiles.md: 2 or 3 query pairs per thread at 3-4 CTAs per
// SM, 256-thread CTAs, separate running extrema for even / odd records (2-input FMNMX only): all >= this one.)
template <class P2, int RP>
int launch_packed(const Ctx& c, BoundsArgs& a) {
    constexpr int THREADS = 128, R = 2 * RP;
    auto kern = bounds_packed_kernel<P2, RP, THREADS, 2>;
    int occ = 0;
    LIPFIT_CUDA(occupancy_of(&occ, kern, THREADS, 0));
    if (occ < 1) occ = 1;
    const int slots = c.num_sms * occ;
    constexpr int TILE = tile_records<2 * P2::RFL>();
    a.nqb = (a.Q + THREADS * R - 1) / (THREADS * R);
    int want = (16 * slots + a.nqb - 1) / a.nqb;
    int max_ch = (a.N + 4 * TILE - 1) / (4 * TILE);
    int nch = want < 1 ? 1 : want;
    if (nch > max_ch) nch = max_ch;
    if (nch < 1) nch = 1;
    int chunk = (a.N + nch - 1) / nch;
    chunk = ((chunk + TILE - 1) / TILE) * TILE;
    nch = (a.N + chunk - 1) / chunk;
    a.nch = nch;
    a.chunk = chunk;
    Workspace keys;
    if (nch > 1) {
        int rc = keys.alloc(sizeof(uint32_t) * 2 * static_cast<size_t>(a.Q), c.stream);
        if (rc) return rc;
        a.keyU = keys.as<uint32_t>();
        a.keyL = a.keyU + a.Q;
        LIPFIT_CUDA(cudaMemsetAsync(a.keyU, 0xFF, sizeof(uint32_t) * a.Q, c.stream));
        LIPFIT_CUDA(cudaMemsetAsync(a.keyL, 0x00, sizeof(uint32_t) * a.Q, c.stream));
    }
    const long long ntiles = static_cast<long long>(a.nqb) * nch;
    KernelTimer kt(TK_BOUNDS, c.stream);
    kern<<<static_cast<int>(ntiles < slots ? ntiles : slots), THREADS, 0, c.stream>>>(a);
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    if (nch > 1) {
        bounds_finalize_kernel<<<(a.Q + 255) / 256, 256, 0, c.stream>>>(a.keyU, a.keyL, a.Q, a.upper, a.lower, a.g);
        ++g_launches;
        LIPFIT_CUDA(cudaGetLastError());
    }
    return LIPFIT_OK;
}

template <int DU, int DC>
int launch_fold(const Ctx& c, BoundsArgs& a, const FreeFlags& ff, int flavour) {
    if (flavour != 0) return launch_one<FoldL1Core<DU, DC>, 1, 128, 4>(c, a, ff);  // small Q: plain records
    return launch_packed<PackedFoldL1<DU, DC>, 4>(c, a);
}

// L2 with M folded into the coordinates: SpecCore<2,..> with M = 1 for small Q
template <int DU, int DC>
int launch_l2p(const Ctx& c, BoundsArgs& a, const FreeFlags& ff, int flavour) {
    if (flavour != 0) {
        a.M = 1.f;
        return launch_one<SpecCore<2, DU, DC>, 1, 128, 4>(c, a, ff);
    }
    return launch_packed<PackedL2<DU, DC>, 4>(c, a);
}

// Linf with M folded into the coordinates (records [M x', y]): SpecCore<3,..> with M = 1 for small Q
template <int DU, int DC>
int launch_linf(const Ctx& c, BoundsArgs& a, const FreeFlags& ff, int flavour) {
    if (flavour != 0) {
        a.M = 1.f;
        return launch_one<SpecCore<3, DU, DC>, 1, 128, 4>(c, a, ff);
    }
    return launch_packed<PackedLinf<DU, DC>, 4>(c, a);
}

template <int NORM, int DP>
int launch_gen(const Ctx& c, BoundsArgs& a, const FreeFlags& ff, int flavour) {
    using Core = GenCore<NORM, DP>;
    constexpr int RBIG = (DP <= 8) ? 4 : (DP <= 16 ? 2 : 1);
    if (flavour == 0 || RBIG == 1) return launch_one<Core, RBIG, 128, 2>(c, a, ff);
    return launch_one<Core, 1, 128, 2>(c, a, ff);
}

#define SPEC(NORM, DU, DC, NAME) \
    { NORM, DU, DC, NAME, {record_floats(DU + DC), DU + DC}, &launch_spec<NORM, DU, DC> }
#define FOLD(DU, DC, NAME) \
    { 1, DU, DC, NAME, {record_floats(DU + DC + 1), DU + DC, DU + DC + 1, true, false, true}, &launch_fold<DU, DC> }
#define LINF2(DU, DC, NAME) \
    { 3, DU, DC, NAME, {record_floats(DU + DC), DU + DC, -1, true, false, true}, &launch_linf<DU, DC> }
#define L2P(DU, DC, NAME) \
    { 2, DU, DC, NAME, {record_floats(DU + DC), DU + DC, -1, true, false, true}, &launch_l2p<DU, DC> }
#define GEN(NORM, DP, NAME) \
    { NORM, DP, -1, NAME, {DP + 4, DP}, &launch_gen<NORM, DP> }
// Off-table shapes with d <= 8: the counts of unconstrained / constrained coordinates are rounded up to even
// numbers with zero-weight padding coordinates (bounds_xform), which contribute |0 - 0| = relu(0 - 0) = 0 to every
// norm, so any (d, mask) with roundup2(dU) + roundup2(dC) <= 8 runs compile-time pair arithmetic (2 lane-ops per
// unconstrained and 5 (Linf: 3) per constrained coordinate) instead of the generic kernel's flag arithmetic
// (6 per padded coordinate of DP = 4 / 8).
#define PAD(NORM, DU, DC, NAME) \
    { NORM, DU, DC, NAME, {record_floats(DU + DC), DU + DC}, &launch_spec<NORM, DU, DC>, true }
#define PAD3(DU, DC, TAG) \
    PAD(1, DU, DC, "bounds<L1," TAG ",padded>"), PAD(2, DU, DC, "bounds<L2," TAG ",padded>"), \
        PAD(3, DU, DC, "bounds<Linf," TAG ",padded>")

const Variant kVariants[] = {
    // shapes of BASELINE.json configs 1, 2, 3, 5 (+ the symmetric versions of the same dims)
    SPEC(2, 2, 0, "bounds<L2,U2,C0>"),
    FOLD(2, 2, "bounds<L1,U2,C2,folded>"),
    LINF2(7, 1, "bounds<Linf,U7,C1,packed>"),
    L2P(0, 5, "bounds<L2,U0,C5,packed>"),
    SPEC(2, 3, 0, "bounds<L2,U3,C0>"),
    SPEC(2, 0, 3, "bounds<L2,U0,C3>"),
    SPEC(1, 4, 0, "bounds<L1,U4,C0>"),
    SPEC(2, 4, 0, "bounds<L2,U4,C0>"),
    SPEC(3, 8, 0, "bounds<Linf,U8,C0>"),
    SPEC(2, 5, 0, "bounds<L2,U5,C0>"),
    // even-rounded shapes for everything else with d <= 8 (bounds_xform pads the transform to one of these)
    PAD3(2, 0, "U2,C0"), PAD3(4, 0, "U4,C0"), PAD3(6, 0, "U6,C0"), PAD3(8, 0, "U8,C0"),
    PAD3(0, 2, "U0,C2"), PAD3(2, 2, "U2,C2"), PAD3(4, 2, "U4,C2"), PAD3(6, 2, "U6,C2"),
    PAD3(0, 4, "U0,C4"), PAD3(2, 4, "U2,C4"), PAD3(4, 4, "U4,C4"),
    PAD3(0, 6, "U0,C6"), PAD3(2, 6, "U2,C6"),
    PAD3(0, 8, "U0,C8"),
    // generic fall-back (any mask / d up to 32): still a GPU kernel, never a CPU path
    GEN(1, 4, "bounds_generic<L1,DP4>"), GEN(2, 4, "bounds_generic<L2,DP4>"),
    GEN(3, 4, "bounds_generic<Linf,DP4>"),
    GEN(1, 8, "bounds_generic<L1,DP8>"), GEN(2, 8, "bounds_generic<L2,DP8>"),
    GEN(3, 8, "bounds_generic<Linf,DP8>"),
    GEN(1, 16, "bounds_generic<L1,DP16>"), GEN(2, 16, "bounds_generic<L2,DP16>"),
    GEN(3, 16, "bounds_generic<Linf,DP16>"),
    GEN(1, 32, "bounds_generic<L1,DP32>"), GEN(2, 32, "bounds_generic<L2,DP32>"),
    GEN(3, 32, "bounds_generic<Linf,DP32>"),
};

// exact table shapes first (in table order: the tuned config kernels come before the even-rounded list), then
// the generic kernels.  with_padded_list = false (top-k pass: it has no kernels for that list) skips the list.
const Variant* pick(const Xform& xf, int norm, bool with_padded_list = true) {
    for (const Variant& v : kVariants)
        if (v.dC >= 0 && v.norm == norm && v.dU == xf.dU && v.dC == xf.dC && (with_padded_list || !v.padded_list))
            return &v;
    for (const Variant& v : kVariants)
        if (v.dC < 0 && v.norm == norm && v.dU >= xf.d) return &v;
    return nullptr;
}

}  // namespace

namespace {
// Small problems (cannot fill the chip with 8-query threads): one query per thread.
int bounds_flavour(const Ctx& c, int64_t Q) { return ((Q + 7) / 8 < 2LL * c.num_sms * 128) ? 1 : 0; }
}  // namespace

// The transform lipfit_bounds_ex really uses: shapes without a tuned kernel and with d <= 8 get zero-weight
// padding coordinates so that both counts are even (see PAD above); everything else is returned unchanged.
Xform bounds_xform(const Xform& xf, int norm) {
    for (const Variant& v : kVariants)
        if (v.dC >= 0 && !v.padded_list && v.norm == norm && v.dU == xf.dU && v.dC == xf.dC) return xf;
    const int du = (xf.dU + 1) & ~1, dc = (xf.dC + 1) & ~1;
    if (xf.d > 8 || du + dc > 8 || (du == xf.dU && dc == xf.dC)) return xf;
    Xform o = xf;
    o.dU = du;
    o.dC = dc;
    o.d = du + dc;
    for (int j = 0; j < kMaxDim; ++j) {
        o.perm[j] = 0;
        o.sw[j] = 0.f;
    }
    for (int j = 0; j < xf.dU; ++j) {
        o.perm[j] = xf.perm[j];
        o.sw[j] = xf.sw[j];
    }
    for (int j = 0; j < xf.dC; ++j) {
        o.perm[du + j] = xf.perm[xf.dU + j];
        o.sw[du + j] = xf.sw[xf.dU + j];
    }
    return o;
}

RecLayout bounds_layout(const Ctx& c, const Xform& xf, int norm, int64_t Q) {
    const Variant* v = pick(xf, norm);
    if (!v) return RecLayout{0, 0};
    RecLayout lay = v->lay;
    if (lay.packed && bounds_flavour(c, Q) == 0) {  // throughput flavour of a packed variant: duplicated records
        lay.rf *= 2;
        lay.dup = true;
    }
    return lay;
}

const char* bounds_variant_name(const Xform& xf, int norm) {
    const Variant* v = pick(xf, norm);
    return v ? v->name : "none";
}

int launch_bounds(const Ctx& c, const float* rec, int64_t N, const float* Xq, int64_t Q,
                  const Xform& xf, int norm, float M, float* upper, float* lower, float* g,
                  const float* centre) {
    const Variant* v = pick(xf, norm);
    if (!v) return LIPFIT_E_PARAM;
    if (centre && v->dC < 0) return LIPFIT_E_PARAM;  // the generic kernels take untranslated records
    BoundsArgs a{};
    a.rec = rec;
    a.Xq = Xq;
    a.centre = centre;
    a.upper = upper;
    a.lower = lower;
    a.g = g;
    a.N = static_cast<int>(N);
    a.Q = static_cast<int>(Q);
    a.d = xf.dsrc;
    a.rf = v->lay.rf;
    a.vslot = v->lay.vslot;
    a.M = M;
    a.xf = xf;
    FreeFlags ff = make_free_flags(xf);
    return v->launch(c, a, ff, bounds_flavour(c, Q));
}

// ---------------------------------------------------------------------------------------------
// NEXT-2: approximation with k > 1 neighbours:
//   upper = sum_j wk[j] * (j-th smallest of y^k + M D^u),  lower = sum_j wk[j] * (j-th largest of y^k - M D^l).
// The same fused pass with the SAME pair arithmetic as lipfit_bounds (the specialised / folded cores of the
// variant table, the generic core elsewhere); every query keeps its K best upper and lower candidates sorted
// in registers (K = 4 for k <= 4, else 8).  The hot loop is the pair arithmetic plus one compare per side
// against the worst kept value and ONE branch; the rare candidates that pass (rate ~ K ln(N) / N) are inserted
// by an unrolled compare-exchange chain.  Small Q: the data are cut into chunks (as in bounds_kernel), every
// (query block, chunk) tile writes its two K-lists to a workspace and a merge kernel forms the weighted sums.
// ---------------------------------------------------------------------------------------------
constexpr int kTopK = LIPFIT_MAX_TOPK;

struct TopkWeights {
    float w[kTopK];
};

template <int K>
__device__ __forceinline__ void topk_insert_min(float (&U)[K], float v) {  // U ascending, U[K-1] = worst kept
    U[K - 1] = v;
#pragma unroll
    for (int i = K - 1; i > 0; --i) {
        const float lo_ = fminf(U[i - 1], U[i]), hi_ = fmaxf(U[i - 1], U[i]);
        U[i - 1] = lo_;
        U[i] = hi_;
    }
}
template <int K>
__device__ __forceinline__ void topk_insert_max(float (&L)[K], float v) {  // L descending
    L[K - 1] = v;
#pragma unroll
    for (int i = K - 1; i > 0; --i) {
        const float hi_ = fmaxf(L[i - 1], L[i]), lo_ = fminf(L[i - 1], L[i]);
        L[i - 1] = hi_;
        L[i] = lo_;
    }
}

template <class Core, int R, int K>
__global__ void __launch_bounds__(128, 2)
bounds_topk_kernel(const BoundsArgs a, const FreeFlags ff, const TopkWeights wk, float* __restrict__ part) {
    constexpr int THREADS = 128;
    constexpr int D = Core::D;
    constexpr int RF = Core::RF;
    constexpr int TILE = tile_records<RF>();
    __shared__ __align__(128) float sbuf[2 * TILE * RF];
    __shared__ __align__(8) uint64_t bars[2];
    if (threadIdx.x == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    uint32_t phase = 0;
    const float inf = __int_as_float(0x7f800000);
    const int ntiles = a.nqb * a.nch;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int qb = tile / a.nch;
        const int ch = tile - qb * a.nch;
        float q[R][D];
        float U[R][K], L[R][K];  // U ascending (U[K-1] = worst kept), L descending
#pragma unroll
        for (int r = 0; r < R; ++r) {
            int qi = (qb * R + r) * THREADS + static_cast<int>(threadIdx.x);
            qi = qi < a.Q ? qi : a.Q - 1;
            const float* src = a.Xq + static_cast<size_t>(qi) * a.d;
#pragma unroll
            for (int j = 0; j < D; ++j) {
                if (Core::kGeneric) {
                    q[r][j] = (j < a.d) ? a.xf.sw[j] * __ldg(src + a.xf.perm[j]) : 0.f;
                } else {
                    const int o = a.xf.perm[j];
                    q[r][j] = a.xf.sw[j] * (a.centre ? __ldg(src + o) - __ldg(a.centre + o) : __ldg(src + o));
                }
            }
#pragma unroll
            for (int j = 0; j < K; ++j) {
                U[r][j] = inf;
                L[r][j] = -inf;
            }
        }
        const int begin = ch * a.chunk;
        const int end = min(a.N, begin + a.chunk);
        RecordStream<TILE> rs(a.rec, RF, begin, end, sbuf, bars, &phase);
        for (int t = 0; t < rs.ntiles; ++t) {
            const float* s = rs.acquire(t);
            const int n = rs.count(t);
            for (int j = 0; j < n; ++j) {
                float x[RF];
                load_record<RF>(s + j * RF, x);
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    float hi, lo;
                    Core::pair(q[r], x, ff, a.M, hi, lo);
                    const bool pu = hi < U[r][K - 1], pl = lo > L[r][K - 1];
                    if (pu | pl) {  // rare: insert into the sorted lists
                        if (pu) topk_insert_min<K>(U[r], hi);
                        if (pl) topk_insert_max<K>(L[r], lo);
                    }
                }
            }
            rs.release(t);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int qi = (qb * R + r) * THREADS + static_cast<int>(threadIdx.x);
            if (qi >= a.Q) continue;
            if (Core::kFold) {  // the per-query constant of the folded lower values (finite entries only)
                const float sq = Core::query_term(q[r]);
#pragma unroll
                for (int j = 0; j < K; ++j) L[r][j] += sq;
            }
            if (a.nch == 1) {
                float su = 0.f, sl = 0.f;
#pragma unroll
                for (int j = 0; j < K; ++j) {  // slots past k have weight 0 (and may hold +-inf: skip them)
                    if (wk.w[j] != 0.f) {
                        su = fmaf(wk.w[j], U[r][j], su);
                        sl = fmaf(wk.w[j], L[r][j], sl);
                    }
                }
                if (a.upper) a.upper[qi] = su;
                if (a.lower) a.lower[qi] = sl;
                if (a.g) a.g[qi] = 0.5f * (su + sl);
            } else {
                float* dst = part + (static_cast<size_t>(ch) * a.Q + qi) * (2 * K);
#pragma unroll
                for (int j = 0; j < K; ++j) {
                    dst[j] = U[r][j];
                    dst[K + j] = L[r][j];
                }
            }
        }
    }
}

// merges the K-lists of the data chunks of one query and forms the weighted sums
template <int K>
__global__ void __launch_bounds__(128)
bounds_topk_merge_kernel(const float* __restrict__ part, int Q, int nch, const TopkWeights wk,
                         float* __restrict__ upper, float* __restrict__ lower, float* __restrict__ g) {
    const int qi = blockIdx.x * blockDim.x + threadIdx.x;
    if (qi >= Q) return;
    float U[K], L[K];
#pragma unroll
    for (int j = 0; j < K; ++j) {
        U[j] = __int_as_float(0x7f800000);
        L[j] = __int_as_float(0xff800000);
    }
    for (int ch = 0; ch < nch; ++ch) {
        const float* src = part + (static_cast<size_t>(ch) * Q + qi) * (2 * K);
#pragma unroll
        for (int j = 0; j < K; ++j) {
            const float u = src[j], l = src[K + j];
            if (u < U[K - 1]) topk_insert_min<K>(U, u);
            if (l > L[K - 1]) topk_insert_max<K>(L, l);
        }
    }
    float su = 0.f, sl = 0.f;
#pragma unroll
    for (int j = 0; j < K; ++j) {
        if (wk.w[j] != 0.f) {
            su = fmaf(wk.w[j], U[j], su);
            sl = fmaf(wk.w[j], L[j], sl);
        }
    }
    if (upper) upper[qi] = su;
    if (lower) lower[qi] = sl;
    if (g) g[qi] = 0.5f * (su + sl);
}

// Packed-f32x2 flavour of the same pass for the variants that have a packed pair policy (throughput flavour,
// duplicated records): RP pairs of queries per thread, pair2() as in bounds_packed_kernel, four sorted lists
// per query pair.  One branch per (record, query pair).
template <class P2, int RP, int K>
__global__ void __launch_bounds__(128, 2)
bounds_topk_packed_kernel(const BoundsArgs a, const TopkWeights wk, float* __restrict__ part) {
    constexpr int THREADS = 128;
    constexpr int D = P2::D;
    constexpr int RFL = P2::RFL;
    constexpr int RF = 2 * RFL;
    constexpr int TILE = tile_records<RF>();
    constexpr int R = 2 * RP;
    __shared__ __align__(128) float sbuf[2 * TILE * RF];
    __shared__ __align__(8) uint64_t bars[2];
    if (threadIdx.x == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    uint32_t phase = 0;
    const float inf = __int_as_float(0x7f800000);
    const int ntiles = a.nqb * a.nch;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int qb = tile / a.nch;
        const int ch = tile - qb * a.nch;
        float2 q[RP][D];
        float U[R][K], L[R][K];
#pragma unroll
        for (int rp = 0; rp < RP; ++rp) {
            int q0 = (qb * R + 2 * rp) * THREADS + static_cast<int>(threadIdx.x);
            int q1 = q0 + THREADS;
            q0 = q0 < a.Q ? q0 : a.Q - 1;
            q1 = q1 < a.Q ? q1 : a.Q - 1;
            const float* s0 = a.Xq + static_cast<size_t>(q0) * a.d;
            const float* s1 = a.Xq + static_cast<size_t>(q1) * a.d;
#pragma unroll
            for (int j = 0; j < D; ++j) {
                const int o = a.xf.perm[j];
                const float cj = a.centre ? __ldg(a.centre + o) : 0.f;
                q[rp][j] = make_float2(a.xf.sw[j] * (__ldg(s0 + o) - cj), a.xf.sw[j] * (__ldg(s1 + o) - cj));
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r)
#pragma unroll
            for (int j = 0; j < K; ++j) {
                U[r][j] = inf;
                L[r][j] = -inf;
            }
        const int begin = ch * a.chunk;
        const int end = min(a.N, begin + a.chunk);
        RecordStream<TILE> rs(a.rec, RF, begin, end, sbuf, bars, &phase);
        for (int t = 0; t < rs.ntiles; ++t) {
            const float* s = rs.acquire(t);
            const int n = rs.count(t);
            for (int j = 0; j < n; ++j) {
                float2 x[RFL];
#pragma unroll
                for (int c = 0; c < RF / 4; ++c) {
                    const float4 v = reinterpret_cast<const float4*>(s + j * RF)[c];
                    x[2 * c] = make_float2(v.x, v.y);
                    x[2 * c + 1] = make_float2(v.z, v.w);
                }
#pragma unroll
                for (int rp = 0; rp < RP; ++rp) {
                    float2 hi, lo;
                    P2::pair2(q[rp], x, hi, lo);
                    const bool p0 = hi.x < U[2 * rp][K - 1], p1 = hi.y < U[2 * rp + 1][K - 1];
                    const bool p2 = lo.x > L[2 * rp][K - 1], p3 = lo.y > L[2 * rp + 1][K - 1];
                    if (p0 | p1 | p2 | p3) {  // rare
                        if (p0) topk_insert_min<K>(U[2 * rp], hi.x);
                        if (p1) topk_insert_min<K>(U[2 * rp + 1], hi.y);
                        if (p2) topk_insert_max<K>(L[2 * rp], lo.x);
                        if (p3) topk_insert_max<K>(L[2 * rp + 1], lo.y);
                    }
                }
            }
            rs.release(t);
        }
#pragma unroll
        for (int rp = 0; rp < RP; ++rp) {
            const float2 sq2 = P2::query_term2(q[rp]);  // per-query constant of the folded lower values
            const float sqv[2] = {sq2.x, sq2.y};
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int r = 2 * rp + e;
                const int qi = (qb * R + r) * THREADS + static_cast<int>(threadIdx.x);
                if (qi >= a.Q) continue;
#pragma unroll
                for (int j = 0; j < K; ++j) L[r][j] += sqv[e];
                if (a.nch == 1) {
                    float su = 0.f, sl = 0.f;
#pragma unroll
                    for (int j = 0; j < K; ++j) {
                        if (wk.w[j] != 0.f) {
                            su = fmaf(wk.w[j], U[r][j], su);
                            sl = fmaf(wk.w[j], L[r][j], sl);
                        }
                    }
                    if (a.upper) a.upper[qi] = su;
                    if (a.lower) a.lower[qi] = sl;
                    if (a.g) a.g[qi] = 0.5f * (su + sl);
                } else {
                    float* dst = part + (static_cast<size_t>(ch) * a.Q + qi) * (2 * K);
#pragma unroll
                    for (int j = 0; j < K; ++j) {
                        dst[j] = U[r][j];
                        dst[K + j] = L[r][j];
                    }
                }
            }
        }
    }
}

namespace {

// schedule + launch shared by the two flavours: KERN(args, part) over (query block, chunk) tiles
template <int K, int TILE, class Launch>
int launch_topk_sched(const Ctx& c, BoundsArgs& a, const TopkWeights& wk, const void* kern, int R, const Launch& go) {
    constexpr int THREADS = 128;
    int occ = 0;
    LIPFIT_CUDA(occupancy_cached(kern, THREADS, 0, &occ));
    if (occ < 1) occ = 1;
    const int slots = c.num_sms * occ;
    a.nqb = (a.Q + THREADS * R - 1) / (THREADS * R);
    // enough (query block, chunk) tiles to fill the chip twice; a chunk at least 8 smem tiles long and at
    // most 64 chunks (the merge reads nch lists per query)
    int want = (2 * slots + a.nqb - 1) / a.nqb;
    int max_ch = (a.N + 8 * TILE - 1) / (8 * TILE);
    if (max_ch > 64) max_ch = 64;
    int nch = want < 1 ? 1 : want;
    if (nch > max_ch) nch = max_ch;
    if (nch < 1) nch = 1;
    int chunk = (a.N + nch - 1) / nch;
    chunk = ((chunk + TILE - 1) / TILE) * TILE;
    nch = (a.N + chunk - 1) / chunk;
    a.nch = nch;
    a.chunk = chunk;
    Workspace part;
    if (nch > 1) {
        int rc = part.alloc(sizeof(float) * 2 * K * static_cast<size_t>(nch) * a.Q, c.stream);
        if (rc) return rc;
    }
    const long long ntiles = static_cast<long long>(a.nqb) * nch;
    KernelTimer kt(TK_BOUNDS_TOPK, c.stream);
    go(static_cast<int>(ntiles < slots ? ntiles : slots), part.as<float>());
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    if (nch > 1) {
        bounds_topk_merge_kernel<K><<<(a.Q + 127) / 128, 128, 0, c.stream>>>(part.as<float>(), a.Q, nch, wk, a.upper,
                                                                              a.lower, a.g);
        ++g_launches;
        LIPFIT_CUDA(cudaGetLastError());
    }
    return LIPFIT_OK;
}

template <class Core, int R, int K>
int launch_topk_t(const Ctx& c, BoundsArgs& a, const FreeFlags& ff, const TopkWeights& wk) {
    auto kern = bounds_topk_kernel<Core, R, K>;
    return launch_topk_sched<K, tile_records<Core::RF>()>(
        c, a, wk, reinterpret_cast<const void*>(kern), R,
        [&](int grid, float* part) { kern<<<grid, 128, 0, c.stream>>>(a, ff, wk, part); });
}

template <class P2, int K>
int launch_topk_packed_t(const Ctx& c, BoundsArgs& a, const TopkWeights& wk) {
    constexpr int RP = 2;
    auto kern = bounds_topk_packed_kernel<P2, RP, K>;
    return launch_topk_sched<K, tile_records<2 * P2::RFL>()>(
        c, a, wk, reinterpret_cast<const void*>(kern), 2 * RP,
        [&](int grid, float* part) { kern<<<grid, 128, 0, c.stream>>>(a, wk, part); });
}

template <class Core, int RBIG>
int launch_topk_core(const Ctx& c, BoundsArgs& a, const FreeFlags& ff, const TopkWeights& wk, int k) {
    // small Q: one query per thread (more tiles to spread); k <= 4: lists of 4
    const bool small = (static_cast<long long>(a.Q) + RBIG - 1) / RBIG < 2LL * c.num_sms * 128;
    if (k <= 4) {
        if (small || RBIG == 1) return launch_topk_t<Core, 1, 4>(c, a, ff, wk);
        return launch_topk_t<Core, RBIG, 4>(c, a, ff, wk);
    }
    if (small || RBIG == 1) return launch_topk_t<Core, 1, 8>(c, a, ff, wk);
    return launch_topk_t<Core, RBIG, 8>(c, a, ff, wk);
}

// dup: the records are in the duplicated layout of the packed-f32x2 kernels (bounds_layout chose the
// throughput flavour of a packed variant)
template <int NORM, int DU, int DC>
int topk_spec(const Ctx& c, BoundsArgs& a, const FreeFlags& ff, const TopkWeights& wk, int k, bool) {
    return launch_topk_core<SpecCore<NORM, DU, DC>, 4>(c, a, ff, wk, k);
}
template <class P2>
int topk_packed(const Ctx& c, BoundsArgs& a, const TopkWeights& wk, int k) {
    return k <= 4 ? launch_topk_packed_t<P2, 4>(c, a, wk) : launch_topk_packed_t<P2, 8>(c, a, wk);
}
template <int DU, int DC>
int topk_fold(const Ctx& c, BoundsArgs& a, const FreeFlags& ff, const TopkWeights& wk, int k, bool dup) {
    if (dup) return topk_packed<PackedFoldL1<DU, DC>>(c, a, wk, k);
    return launch_topk_core<FoldL1Core<DU, DC>, 4>(c, a, ff, wk, k);
}
template <int NORM, int DU, int DC>
int topk_mfold(const Ctx& c, BoundsArgs& a, const FreeFlags& ff, const TopkWeights& wk, int k, bool dup) {
    if (dup) {
        if (NORM == 2) return topk_packed<PackedL2<DU, DC>>(c, a, wk, k);
        return topk_packed<PackedLinf<DU, DC>>(c, a, wk, k);
    }
    a.M = 1.f;  // M rides in the coordinates (layouts with mscale)
    return launch_topk_core<SpecCore<NORM, DU, DC>, 4>(c, a, ff, wk, k);
}
template <int NORM, int DP>
int topk_gen(const Ctx& c, BoundsArgs& a, const FreeFlags& ff, const TopkWeights& wk, int k, bool) {
    return launch_topk_core<GenCore<NORM, DP>, (DP <= 8 ? 2 : 1)>(c, a, ff, wk, k);
}

using TopkLaunch = int (*)(const Ctx&, BoundsArgs&, const FreeFlags&, const TopkWeights&, int, bool);

// same order as kVariants
const TopkLaunch kTopkLaunch[] = {
    &topk_spec<2, 2, 0>, &topk_fold<2, 2>, &topk_mfold<3, 7, 1>, &topk_mfold<2, 0, 5>, &topk_spec<2, 3, 0>,
    &topk_spec<2, 0, 3>, &topk_spec<1, 4, 0>, &topk_spec<2, 4, 0>, &topk_spec<3, 8, 0>, &topk_spec<2, 5, 0>,
    // the even-rounded list of kVariants has no top-k kernels: pick(..., false) never returns those entries
    nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr,
    nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr,
    nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr,
    nullptr, nullptr, nullptr, nullptr, nullptr, nullptr,
    &topk_gen<1, 4>, &topk_gen<2, 4>, &topk_gen<3, 4>, &topk_gen<1, 8>, &topk_gen<2, 8>, &topk_gen<3, 8>,
    &topk_gen<1, 16>, &topk_gen<2, 16>, &topk_gen<3, 16>, &topk_gen<1, 32>, &topk_gen<2, 32>, &topk_gen<3, 32>,
};
static_assert(sizeof(kTopkLaunch) / sizeof(kTopkLaunch[0]) == sizeof(kVariants) / sizeof(kVariants[0]),
              "one top-k launcher per bounds variant");

}  // namespace

// records of the top-k pass: the same layout lipfit_bounds would use (duplicated for the packed flavour)
RecLayout bounds_topk_layout(const Ctx& c, const Xform& xf, int norm, int64_t Q) {
    const Variant* v = pick(xf, norm, false);
    if (!v) return RecLayout{0, 0};
    RecLayout lay = v->lay;
    if (lay.packed && bounds_flavour(c, Q) == 0) {  // throughput flavour of a packed variant: duplicated records
        lay.rf *= 2;
        lay.dup = true;
    }
    return lay;
}

int launch_bounds_topk(const Ctx& c, const float* rec, int64_t N, const float* Xq, int64_t Q, const Xform& xf,
                       int norm, float M, int k, const float* wk_host, float* upper, float* lower, float* g,
                       const float* centre, bool dup) {
    const Variant* v = pick(xf, norm, false);
    if (!v) return LIPFIT_E_PARAM;
    if (centre && v->dC < 0) return LIPFIT_E_PARAM;
    BoundsArgs a{};
    a.rec = rec;
    a.Xq = Xq;
    a.centre = centre;
    a.upper = upper;
    a.lower = lower;
    a.g = g;
    a.N = static_cast<int>(N);
    a.Q = static_cast<int>(Q);
    a.d = xf.dsrc;
    a.rf = v->lay.rf;
    a.vslot = v->lay.vslot;
    a.M = M;
    a.xf = xf;
    TopkWeights wk;
    for (int j = 0; j < kTopK; ++j) wk.w[j] = j < k ? wk_host[j] : 0.f;
    FreeFlags ff = make_free_flags(xf);
    return kTopkLaunch[v - kVariants](c, a, ff, wk, k, dup);
}

}  // namespace lipfit
