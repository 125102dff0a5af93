// local.cu -- NEXT-1: local Lipschitz interpolation, PAPER.md:169-183 (section 4.3).
//   (1) knots t_1..t_J: nearest-rank quantiles of a sample of inter-point distances;
//   (2) per-datum non-decreasing step functions M_k: table[k][j] = max(|y_k - y_(1)|/d_(1),
//       max_{i != k, D(x^k,x^i) <= t_j} |y_k - y_i| / D), last knot = +inf -- an all-pairs pass, J running
//       maxima per row in registers, nothing of size N x N stored;
//   (3) evaluation: Eq.(2),(3) with M replaced by M_k(D(x, x^k)): the fused bounds pass
//       with the table row riding in the packed record and a two-level knot lookup (3 + 3 compares, the
//       paper's torch.searchsorted) that indexes the row in shared memory.
// Radial, symmetric weighted distance D(a,b) = ||w (a - b)||_p; J is fixed at LIPFIT_LOCAL_KNOTS = 16.
#include <cub/device/device_radix_sort.cuh>

#include <cmath>
#include <cstring>

#include "kernels.h"

namespace lipfit {

constexpr int kJ = LIPFIT_LOCAL_KNOTS;
constexpr int kLocThreads = 128;

struct Knots {
    float t[kJ];
    // cell table of the knot lookup (local_knot_lut): cell = clamp(bits(D) >> shift, lo, hi) - lo
    int lut_shift;
    uint32_t lut_lo, lut_hi;
};
constexpr int kLutCells = 1024;  // 8 KB of shared memory

// exact-ish distance from the accumulated quantity: IEEE square root (bin decisions compare D with knots)
template <int NORM>
__device__ __forceinline__ float local_finish(float acc) {
    return NORM == 2 ? __fsqrt_rn(acc) : acc;
}

template <int RF>
__device__ __forceinline__ void local_load_record(const float* s, float* x) {
#pragma unroll
    for (int c = 0; c < RF / 4; ++c) {
        float4 v = reinterpret_cast<const float4*>(s)[c];
        x[4 * c + 0] = v.x;
        x[4 * c + 1] = v.y;
        x[4 * c + 2] = v.z;
        x[4 * c + 3] = v.w;
    }
}

// Knot lookup (the paper's searchsorted): index of the first knot t_j >= D among t_0..t_{J-2}, J-1 if none
// = number of those knots below D (they are sorted).  Two levels of 3 compares instead of a chain of 15
// compare/selects: which quarter (knots 3, 7, 11 from the constant bank), then the quarter's three knots as
// one 16-byte shared-memory word.
static_assert(kJ == 16, "two levels of four");
__device__ __forceinline__ void local_knot_groups(const Knots& kn, float4* sk4) {
    if (threadIdx.x < 4) {
        const int q = threadIdx.x;
        sk4[q] = make_float4(kn.t[4 * q], kn.t[4 * q + 1], kn.t[4 * q + 2], 0.f);
    }
}
__device__ __forceinline__ int local_knot_index(float D, const Knots& kn, const float4* sk4) {
    const int q = (D > kn.t[3] ? 1 : 0) + (D > kn.t[7] ? 1 : 0) + (D > kn.t[11] ? 1 : 0);
    const float4 g = sk4[q];
    return 4 * q + (D > g.x ? 1 : 0) + (D > g.y ? 1 : 0) + (D > g.z ? 1 : 0);
}

// The same lookup for knot sets that allow it (template parameter LUT of the kernels; local_lut_params decides):
// the bit pattern of a non-negative float is monotone in its value, so bits(D) >> shift cuts the axis into
// cells; when no cell holds more than one of the knots t_0..t_{J-2}, a table of (the knot inside the cell or
// +inf, the number of knots below the cell) per cell answers with one 8-byte shared-memory load and ONE
// compare: 9 instructions per pair instead of 22.  Values outside [t_0, t_{J-2}] clamp to the end cells,
// which hold those two knots, so the count stays exact.
__device__ __forceinline__ void local_knot_lut_build(const Knots& kn, float2* lut) {
    const uint32_t ncell = kn.lut_hi - kn.lut_lo + 1u;
    for (uint32_t c = threadIdx.x; c < ncell; c += blockDim.x) {
        const uint32_t lo = (kn.lut_lo + c) << kn.lut_shift, width = 1u << kn.lut_shift;
        int below = 0;
        float inside = __int_as_float(0x7f800000);
        for (int j = 0; j < kJ - 1; ++j) {
            const uint32_t b = __float_as_uint(kn.t[j]);
            if (b < lo) ++below;
            else if (b - lo < width) inside = kn.t[j];
        }
        lut[c] = make_float2(inside, __int_as_float(below));
    }
}
__device__ __forceinline__ int local_knot_lut(float D, const Knots& kn, const float2* lut) {
    const uint32_t c = min(max(__float_as_uint(D) >> kn.lut_shift, kn.lut_lo), kn.lut_hi) - kn.lut_lo;
    const float2 e = lut[c];
    return __float_as_int(e.y) + (D > e.x ? 1 : 0);
}

template <int RF>
__host__ __device__ constexpr int local_tile_records() {
    return RF <= 8 ? 512 : (RF <= 20 ? 256 : (RF <= 40 ? 128 : 64));
}

// ---------------------------------------------------------------------------------------------
// (1) knots
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
local_pair_dist_kernel(const float* __restrict__ X, int N, Xform xf, int norm, const int32_t* __restrict__ pi,
                       const int32_t* __restrict__ pk, int S, float* __restrict__ out, int* __restrict__ bad) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= S) return;
    const int i = pi[s], k = pk[s];
    if (i < 0 || i >= N || k < 0 || k >= N) {
        *bad = 1;
        out[s] = 0.f;
        return;
    }
    const float* a = X + static_cast<size_t>(i) * xf.d;
    const float* b = X + static_cast<size_t>(k) * xf.d;
    float acc = 0.f;
    for (int j = 0; j < xf.d; ++j) {
        const int o = xf.perm[j];
        const float c = fabsf(xf.sw[j] * a[o] - xf.sw[j] * b[o]);
        if (norm == 1) acc += c;
        else if (norm == 2) acc = fmaf(c, c, acc);
        else acc = fmaxf(acc, c);
    }
    out[s] = norm == 2 ? __fsqrt_rn(acc) : acc;
}

__global__ void local_pick_kernel(const float* __restrict__ sorted, long long S, int J, float* __restrict__ knots) {
    int j = threadIdx.x + 1;
    if (j > J) return;
    const long long idx = (static_cast<long long>(j) * S + J - 1) / J - 1;  // ceil(j S / J) - 1
    knots[j - 1] = sorted[idx];
}

// ---------------------------------------------------------------------------------------------
// (2) step tables
// ---------------------------------------------------------------------------------------------
struct TableArgs {
    const float* rec;          // [N][RF]: x' (DP), y at slot DP
    uint32_t* tab;             // [N][kJ] bits of the running maxima (non-negative floats)
    unsigned long long* nn;    // [N] (bits of d_(1)) << 32 | ~(bits of its ratio): atomicMin = nearest, then largest ratio
    int N, nrb, nch, chunk;
};

// records per shared-memory tile of the table kernel: its per-thread bins take R * kJ * 512 B of the 48 KB
template <int RF, bool LUT>
__host__ __device__ constexpr int local_table_tile() {
    return (RF <= 8 ? 128 : local_tile_records<RF>() / 2) / (LUT && RF <= 12 ? 2 : 1);  // room for the cell table
}

// DP: padded coordinates of a record (layout); DA <= DP: the coordinates that exist (d), the only ones the
// distance arithmetic visits (for d <= 8 a compile-time constant: no work on padding)
template <int NORM, int DP, int DA, int R, bool LUT>
__global__ void __launch_bounds__(kLocThreads, 2)
local_table_kernel(const TableArgs a, const Knots kn) {
    constexpr int RF = DP + 4;
    constexpr int TILE = local_table_tile<RF, LUT>();
    __shared__ __align__(128) float sbuf[2 * TILE * RF];
    __shared__ __align__(8) uint64_t bars[2];
    // running maxima per (row, bin) in thread-private shared memory ([r][j][thread]: conflict-free): a pair
    // raises ONE bin (the first knot >= its distance); the cumulative table is a prefix maximum at the end
    __shared__ float sM[R * kJ * kLocThreads];
    __shared__ float4 sk4[4];
    __shared__ float2 slut[LUT ? kLutCells : 1];
    local_knot_groups(kn, sk4);
    if (LUT) local_knot_lut_build(kn, slut);
    if (threadIdx.x == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    uint32_t phase = 0;
    const float inf = __int_as_float(0x7f800000);
    const int ntiles = a.nrb * a.nch;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int rb = tile / a.nch, ch = tile - rb * a.nch;
        float xi[R][DA], yi[R], dmin[R], dmin2[R], rnn[R];
        float* myM = sM + threadIdx.x;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            int i = (rb * R + r) * kLocThreads + static_cast<int>(threadIdx.x);
            i = i < a.N ? i : a.N - 1;
            const float* src = a.rec + static_cast<size_t>(i) * RF;
#pragma unroll
            for (int j = 0; j < DA; ++j) xi[r][j] = __ldg(src + j);
            yi[r] = __ldg(src + DP);
#pragma unroll
            for (int j = 0; j < kJ; ++j) myM[(r * kJ + j) * kLocThreads] = 0.f;
            dmin[r] = inf;
            dmin2[r] = inf;
            rnn[r] = 0.f;
        }
        const int begin = ch * a.chunk;
        const int end = min(a.N, begin + a.chunk);
        RecordStream<TILE> rs(a.rec, RF, begin, end, sbuf, bars, &phase);
        for (int t = 0; t < rs.ntiles; ++t) {
            const float* s = rs.acquire(t);
            const int n = rs.count(t);
            for (int jrec = 0; jrec < n; ++jrec) {
                float x[DP + 4];
                local_load_record<DP + 4>(s + jrec * RF, x);
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    // L2: the knots of this kernel are squared (launch_local_lipschitz): bins from the squared
                    // distance.  The IEEE square root and quotient of the ratio are only taken by the pairs that
                    // can raise their bin (ratio > M  <=>  dy > M D, tested with the 2-ulp MUFU root and a
                    // 2^-20 margin so that no raise is missed) or that are a nearest neighbour so far: a few
                    // hundred of the N pairs of a row.
                    const float acc = PairAccU<NORM, DA, 0>::run(xi[r], x);
                    const float dy = fabsf(yi[r] - x[DP]);
                    const int bin = LUT ? local_knot_lut(acc, kn, slut) : local_knot_index(acc, kn, sk4);
                    float* pb = myM + (r * kJ + bin) * kLocThreads;
                    const float Mb = *pb;
                    const float Da = NORM == 2 ? fast_sqrt(acc) : acc;
                    const bool valid = (acc > 0.f) || (dy > 0.f);  // not the row itself / an exact duplicate
                    if (dy > Mb * Da * (1.f - 0x1p-20f) || (valid && acc <= dmin2[r])) {
                        const float D = local_finish<NORM>(acc);
                        // duplicate position with a different value: +inf
                        const float ratio = D > 0.f ? __fdiv_rn(dy, D) : (dy > 0.f ? inf : 0.f);
                        *pb = fmaxf(Mb, ratio);
                        if (valid && acc < dmin2[r]) {
                            dmin2[r] = acc;
                            dmin[r] = D;
                            rnn[r] = ratio;
                        } else if (valid && acc == dmin2[r]) {
                            rnn[r] = fmaxf(rnn[r], ratio);
                        }
                    }
                }
            }
            rs.release(t);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int i = (rb * R + r) * kLocThreads + static_cast<int>(threadIdx.x);
            if (i < a.N) {
                float m = 0.f;
#pragma unroll
                for (int j = 0; j < kJ; ++j) {
                    m = fmaxf(m, myM[(r * kJ + j) * kLocThreads]);
                    if (m > 0.f) atomicMax(a.tab + static_cast<size_t>(i) * kJ + j, __float_as_uint(m));
                }
                const unsigned long long key = (static_cast<unsigned long long>(__float_as_uint(dmin[r])) << 32) |
                                               static_cast<unsigned long long>(~__float_as_uint(rnn[r]));
                atomicMin(a.nn + i, key);
            }
        }
    }
}

__global__ void __launch_bounds__(256)
local_table_final_kernel(const uint32_t* __restrict__ tab, const unsigned long long* __restrict__ nn, int N,
                         float* __restrict__ table) {
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= N * kJ) return;
    const int i = e / kJ;
    const unsigned long long key = nn[i];
    const float dmin = __uint_as_float(static_cast<uint32_t>(key >> 32));
    const float rnn = (dmin < __int_as_float(0x7f800000)) ? __uint_as_float(~static_cast<uint32_t>(key)) : 0.f;
    table[e] = fmaxf(__uint_as_float(tab[e]), rnn);
}

// ---------------------------------------------------------------------------------------------
// (3) evaluation
// ---------------------------------------------------------------------------------------------
// records for the evaluation: [x' (DP), y, 0, 0, 0, M_k[0..15]]
__global__ void __launch_bounds__(256)
local_eval_pack_kernel(const float* __restrict__ X, const float* __restrict__ y, const float* __restrict__ table,
                       int N, Xform xf, int dp, float* __restrict__ rec) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const int rf = dp + 4 + kJ;
    float* dst = rec + static_cast<size_t>(k) * rf;
    const float* src = X + static_cast<size_t>(k) * xf.d;
    for (int j = 0; j < dp + 4; ++j) dst[j] = j < xf.d ? xf.sw[j] * src[xf.perm[j]] : (j == dp ? y[k] : 0.f);
    for (int j = 0; j < kJ; ++j) dst[dp + 4 + j] = table[static_cast<size_t>(k) * kJ + j];
}

struct EvalArgs {
    const float* rec;
    const float* Xq;
    uint32_t* keyU;
    uint32_t* keyL;
    int N, Q, d, nqb, nch, chunk;
    Xform xf;
};

template <int NORM, int DP, int DA, int R, bool LUT>
__global__ void __launch_bounds__(kLocThreads, 2)
local_eval_kernel(const EvalArgs a, const Knots kn) {
    constexpr int RF = DP + 4 + kJ;
    constexpr int TILE = local_tile_records<RF>();
    __shared__ __align__(128) float sbuf[2 * TILE * RF];
    __shared__ __align__(8) uint64_t bars[2];
    __shared__ float4 sk4[4];
    __shared__ float2 slut[LUT ? kLutCells : 1];
    local_knot_groups(kn, sk4);
    if (LUT) local_knot_lut_build(kn, slut);
    if (threadIdx.x == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    uint32_t phase = 0;
    const int ntiles = a.nqb * a.nch;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int qb = tile / a.nch, ch = tile - qb * a.nch;
        float q[R][DA], U[R], L[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            int qi = (qb * R + r) * kLocThreads + static_cast<int>(threadIdx.x);
            qi = qi < a.Q ? qi : a.Q - 1;
            const float* src = a.Xq + static_cast<size_t>(qi) * a.d;
#pragma unroll
            for (int j = 0; j < DA; ++j) q[r][j] = (j < a.d) ? a.xf.sw[j] * __ldg(src + a.xf.perm[j]) : 0.f;
            U[r] = __int_as_float(0x7f800000);
            L[r] = __int_as_float(0xff800000);
        }
        const int begin = ch * a.chunk;
        const int end = min(a.N, begin + a.chunk);
        RecordStream<TILE> rs(a.rec, RF, begin, end, sbuf, bars, &phase);
        for (int t = 0; t < rs.ntiles; ++t) {
            const float* s = rs.acquire(t);
            const int n = rs.count(t);
            for (int jrec = 0; jrec < n; ++jrec) {
                float x[DP + 4];
                local_load_record<DP + 4>(s + jrec * RF, x);
                const float yk = x[DP];
                const float* mk = s + jrec * RF + DP + 4;  // the datum's step table stays in shared memory
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    // L2: the knots of this kernel are squared (launch_values_local), so the bin is decided on
                    // the squared distance and the square root (one MUFU, <= 2 ulp) only scales M_k
                    const float acc = PairAccU<NORM, DA, 0>::run(q[r], x);
                    const float Mk = mk[LUT ? local_knot_lut(acc, kn, slut) : local_knot_index(acc, kn, sk4)];
                    const float D = NORM == 2 ? fast_sqrt(acc) : acc;
                    const float MD = D > 0.f ? Mk * D : 0.f;  // M_k may be +inf at a duplicate: inf * 0 := 0
                    U[r] = fminf(U[r], yk + MD);
                    L[r] = fmaxf(L[r], yk - MD);
                }
            }
            rs.release(t);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int qi = (qb * R + r) * kLocThreads + static_cast<int>(threadIdx.x);
            if (qi < a.Q) {
                atomicMin(a.keyU + qi, f2key(U[r]));
                atomicMax(a.keyL + qi, f2key(L[r]));
            }
        }
    }
}

// ---- packed f32x2 evaluation (L2, d <= 8) ----------------------------------------------------
// A thread keeps its 8 queries as 4 register pairs (q_r, q_r+1); the records carry every coordinate twice,
//     [x'_0, x'_0, x'_1, x'_1, .. (2 * DE floats, DE = d rounded up to even), y, 0, 0, 0, M_k[0..15]],
// so that an LDS.128 yields two operands of FADD2 / FFMA2: the 2 d distance instructions of a pair become d,
// and y +- M_k D one FADD2 each per two pairs.  Same operations in the same order as local_eval_kernel:
// bit-identical outputs.
__global__ void __launch_bounds__(256)
local_eval_pack2_kernel(const float* __restrict__ X, const float* __restrict__ y, const float* __restrict__ table,
                        int N, Xform xf, int de, float* __restrict__ rec) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const int rf = 2 * de + 4 + kJ;
    float* dst = rec + static_cast<size_t>(k) * rf;
    const float* src = X + static_cast<size_t>(k) * xf.d;
    for (int j = 0; j < de; ++j) {
        const float v = j < xf.d ? xf.sw[j] * src[xf.perm[j]] : 0.f;
        dst[2 * j] = v;
        dst[2 * j + 1] = v;
    }
    dst[2 * de] = y[k];
    dst[2 * de + 1] = dst[2 * de + 2] = dst[2 * de + 3] = 0.f;
    for (int j = 0; j < kJ; ++j) dst[2 * de + 4 + j] = table[static_cast<size_t>(k) * kJ + j];
}

constexpr int kLocPairs = 4;  // query pairs per thread (measured on config 6: 2 / 3 / 4 pairs 191 / 184 / 181 ms)
__device__ __forceinline__ float2 local_sub2(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }

template <int DA, bool LUT>
__global__ void __launch_bounds__(kLocThreads, 2)
local_eval_packed_kernel(const EvalArgs a, const Knots kn) {
    constexpr int DE = (DA + 1) & ~1;
    constexpr int RF = 2 * DE + 4 + kJ;
    constexpr int TILE = local_tile_records<RF>();
    constexpr int RP = kLocPairs;
    __shared__ __align__(128) float sbuf[2 * TILE * RF];
    __shared__ __align__(8) uint64_t bars[2];
    __shared__ float4 sk4[4];
    __shared__ float2 slut[LUT ? kLutCells : 1];
    local_knot_groups(kn, sk4);
    if (LUT) local_knot_lut_build(kn, slut);
    if (threadIdx.x == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    uint32_t phase = 0;
    const int ntiles = a.nqb * a.nch;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int qb = tile / a.nch, ch = tile - qb * a.nch;
        float2 q[RP][DA], U[RP], L[RP];
#pragma unroll
        for (int rp = 0; rp < RP; ++rp) {
            int q0 = (qb * 2 * RP + 2 * rp) * kLocThreads + static_cast<int>(threadIdx.x);
            int q1 = q0 + kLocThreads;
            q0 = q0 < a.Q ? q0 : a.Q - 1;
            q1 = q1 < a.Q ? q1 : a.Q - 1;
            const float* s0 = a.Xq + static_cast<size_t>(q0) * a.d;
            const float* s1 = a.Xq + static_cast<size_t>(q1) * a.d;
#pragma unroll
            for (int j = 0; j < DA; ++j)
                q[rp][j] = make_float2(a.xf.sw[j] * __ldg(s0 + a.xf.perm[j]), a.xf.sw[j] * __ldg(s1 + a.xf.perm[j]));
            U[rp] = make_float2(__int_as_float(0x7f800000), __int_as_float(0x7f800000));
            L[rp] = make_float2(__int_as_float(0xff800000), __int_as_float(0xff800000));
        }
        const int begin = ch * a.chunk;
        const int end = min(a.N, begin + a.chunk);
        RecordStream<TILE> rs(a.rec, RF, begin, end, sbuf, bars, &phase);
        for (int t = 0; t < rs.ntiles; ++t) {
            const float* s = rs.acquire(t);
            const int n = rs.count(t);
            for (int jrec = 0; jrec < n; ++jrec) {
                float xr[2 * DE];
                local_load_record<2 * DE>(s + jrec * RF, xr);
                const float yk = s[jrec * RF + 2 * DE];
                const float2 y2 = make_float2(yk, yk);
                const float* mk = s + jrec * RF + 2 * DE + 4;  // the datum's step table stays in shared memory
#pragma unroll
                for (int rp = 0; rp < RP; ++rp) {
                    float2 acc = make_float2(0.f, 0.f);
#pragma unroll
                    for (int j = 0; j < DA; ++j) {
                        const float2 dl = local_sub2(q[rp][j], make_float2(xr[2 * j], xr[2 * j + 1]));
                        acc = __ffma2_rn(dl, dl, acc);
                    }
                    const float M0 = mk[LUT ? local_knot_lut(acc.x, kn, slut) : local_knot_index(acc.x, kn, sk4)];
                    const float M1 = mk[LUT ? local_knot_lut(acc.y, kn, slut) : local_knot_index(acc.y, kn, sk4)];
                    const float D0 = fast_sqrt(acc.x), D1 = fast_sqrt(acc.y);
                    // M_k may be +inf at a duplicate: inf * 0 := 0
                    const float2 MD = make_float2(D0 > 0.f ? M0 * D0 : 0.f, D1 > 0.f ? M1 * D1 : 0.f);
                    const float2 hi = __fadd2_rn(y2, MD), lo = local_sub2(y2, MD);
                    U[rp] = make_float2(fminf(U[rp].x, hi.x), fminf(U[rp].y, hi.y));
                    L[rp] = make_float2(fmaxf(L[rp].x, lo.x), fmaxf(L[rp].y, lo.y));
                }
            }
            rs.release(t);
        }
#pragma unroll
        for (int rp = 0; rp < RP; ++rp) {
            const int q0 = (qb * 2 * RP + 2 * rp) * kLocThreads + static_cast<int>(threadIdx.x);
            const int q1 = q0 + kLocThreads;
            if (q0 < a.Q) {
                atomicMin(a.keyU + q0, f2key(U[rp].x));
                atomicMax(a.keyL + q0, f2key(L[rp].x));
            }
            if (q1 < a.Q) {
                atomicMin(a.keyU + q1, f2key(U[rp].y));
                atomicMax(a.keyL + q1, f2key(L[rp].y));
            }
        }
    }
}

__global__ void __launch_bounds__(256)
local_eval_final_kernel(const uint32_t* __restrict__ keyU, const uint32_t* __restrict__ keyL, int Q,
                        float* __restrict__ upper, float* __restrict__ lower, float* __restrict__ g) {
    int qi = blockIdx.x * blockDim.x + threadIdx.x;
    if (qi >= Q) return;
    const float U = key2f(keyU[qi]), L = key2f(keyL[qi]);
    if (upper) upper[qi] = U;
    if (lower) lower[qi] = L;
    if (g) g[qi] = 0.5f * (U + L);
}

namespace {

int local_dp(int d) { return d <= 4 ? 4 : (d <= 8 ? 8 : (d <= 16 ? 16 : 32)); }
constexpr int local_r(int dp) { return dp <= 8 ? 4 : (dp <= 16 ? 2 : 1); }

// (row/query blocks) x (data chunks): enough work items for ~8 per resident CTA
void local_schedule(int units, int per_block, int N, int tile, int slots, int* nb, int* nch, int* chunk) {
    *nb = (units + per_block - 1) / per_block;
    int want = (8 * slots + *nb - 1) / *nb;
    int max_ch = (N + 2 * tile - 1) / (2 * tile);
    int c = want < 1 ? 1 : want;
    if (c > max_ch) c = max_ch;
    if (c < 1) c = 1;
    int ck = (N + c - 1) / c;
    ck = ((ck + tile - 1) / tile) * tile;
    *nch = (N + ck - 1) / ck;
    *chunk = ck;
}

template <int NORM, int DP, int DA, bool LUT>
int launch_table_l(const Ctx& c, TableArgs& a, const Knots& kn) {
    constexpr int R = local_r(DP);
    auto kern = local_table_kernel<NORM, DP, DA, R, LUT>;
    int occ = 0;
    LIPFIT_CUDA(occupancy_of(&occ, kern, kLocThreads, 0));
    if (occ < 1) occ = 1;
    const int slots = c.num_sms * occ;
    local_schedule(a.N, kLocThreads * R, a.N, local_table_tile<DP + 4, LUT>(), slots, &a.nrb, &a.nch, &a.chunk);
    const long long nt = static_cast<long long>(a.nrb) * a.nch;
    KernelTimer kt(TK_LOCAL_TABLE, c.stream);
    kern<<<static_cast<int>(nt < slots ? nt : slots), kLocThreads, 0, c.stream>>>(a, kn);
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

template <int NORM, int DP, int DA>
int launch_table(const Ctx& c, TableArgs& a, const Knots& kn) {
    return kn.lut_shift >= 0 ? launch_table_l<NORM, DP, DA, true>(c, a, kn) : launch_table_l<NORM, DP, DA, false>(c, a, kn);
}

template <int NORM, int DP, int DA, bool LUT>
int launch_eval_l(const Ctx& c, EvalArgs& a, const Knots& kn) {
    constexpr int R = local_r(DP);
    auto kern = local_eval_kernel<NORM, DP, DA, R, LUT>;
    int occ = 0;
    LIPFIT_CUDA(occupancy_of(&occ, kern, kLocThreads, 0));
    if (occ < 1) occ = 1;
    const int slots = c.num_sms * occ;
    local_schedule(a.Q, kLocThreads * R, a.N, local_tile_records<DP + 4 + kJ>(), slots, &a.nqb, &a.nch, &a.chunk);
    const long long nt = static_cast<long long>(a.nqb) * a.nch;
    KernelTimer kt(TK_LOCAL_EVAL, c.stream);
    kern<<<static_cast<int>(nt < slots ? nt : slots), kLocThreads, 0, c.stream>>>(a, kn);
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

template <int NORM, int DP, int DA>
int launch_eval(const Ctx& c, EvalArgs& a, const Knots& kn) {
    return kn.lut_shift >= 0 ? launch_eval_l<NORM, DP, DA, true>(c, a, kn) : launch_eval_l<NORM, DP, DA, false>(c, a, kn);
}

template <int DA, bool LUT>
int launch_eval_packed_l(const Ctx& c, EvalArgs& a, const Knots& kn) {
    constexpr int RF = 2 * ((DA + 1) & ~1) + 4 + kJ;
    auto kern = local_eval_packed_kernel<DA, LUT>;
    int occ = 0;
    LIPFIT_CUDA(occupancy_of(&occ, kern, kLocThreads, 0));
    if (occ < 1) occ = 1;
    const int slots = c.num_sms * occ;
    local_schedule(a.Q, kLocThreads * 2 * kLocPairs, a.N, local_tile_records<RF>(), slots, &a.nqb, &a.nch, &a.chunk);
    const long long nt = static_cast<long long>(a.nqb) * a.nch;
    KernelTimer kt(TK_LOCAL_EVAL, c.stream);
    kern<<<static_cast<int>(nt < slots ? nt : slots), kLocThreads, 0, c.stream>>>(a, kn);
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}
template <int DA>
int launch_eval_packed(const Ctx& c, EvalArgs& a, const Knots& kn) {
    return kn.lut_shift >= 0 ? launch_eval_packed_l<DA, true>(c, a, kn) : launch_eval_packed_l<DA, false>(c, a, kn);
}
int dispatch_eval_packed(const Ctx& c, EvalArgs& a, const Knots& kn, int d) {
    switch (d) {
        case 1: return launch_eval_packed<1>(c, a, kn);
        case 2: return launch_eval_packed<2>(c, a, kn);
        case 3: return launch_eval_packed<3>(c, a, kn);
        case 4: return launch_eval_packed<4>(c, a, kn);
        case 5: return launch_eval_packed<5>(c, a, kn);
        case 6: return launch_eval_packed<6>(c, a, kn);
        case 7: return launch_eval_packed<7>(c, a, kn);
        default: return launch_eval_packed<8>(c, a, kn);
    }
}

// Kernel knots (squared for L2) -> cell table parameters; lut_shift = -1 when the knot set does not allow a
// table of kLutCells cells with at most one knot per cell (a zero or repeated knot, knots closer than a cell).
void local_lut_params(Knots& kn) {
    kn.lut_shift = -1;
    kn.lut_lo = kn.lut_hi = 0;
    uint32_t b[kJ - 1];
    for (int j = 0; j < kJ - 1; ++j) {
        if (!(kn.t[j] > 0.f) || !std::isfinite(kn.t[j])) return;
        std::memcpy(&b[j], &kn.t[j], 4);
        if (j > 0 && b[j] <= b[j - 1]) return;
    }
    for (int sh = 0; sh <= 23; ++sh) {
        if ((b[kJ - 2] >> sh) - (b[0] >> sh) + 1u > static_cast<uint32_t>(kLutCells)) continue;
        for (int j = 1; j < kJ - 1; ++j)
            if ((b[j] >> sh) == (b[j - 1] >> sh)) return;  // two knots in one cell at the finest table that fits
        kn.lut_shift = sh;
        kn.lut_lo = b[0] >> sh;
        kn.lut_hi = b[kJ - 2] >> sh;
        return;
    }
}

// d <= 8: the number of coordinates is a template parameter (DA = d inside records padded to DP = 4 / 8);
// d > 8: padded arithmetic (DA = DP = 16 / 32)
#define LOCAL_DISPATCH_N(FN, ARGS, NORM)                 \
    switch (d) {                                         \
        case 1: return FN<NORM, 4, 1> ARGS;              \
        case 2: return FN<NORM, 4, 2> ARGS;              \
        case 3: return FN<NORM, 4, 3> ARGS;              \
        case 4: return FN<NORM, 4, 4> ARGS;              \
        case 5: return FN<NORM, 8, 5> ARGS;              \
        case 6: return FN<NORM, 8, 6> ARGS;              \
        case 7: return FN<NORM, 8, 7> ARGS;              \
        case 8: return FN<NORM, 8, 8> ARGS;              \
        default: break;                                  \
    }                                                    \
    if (d <= 16) return FN<NORM, 16, 16> ARGS;           \
    return FN<NORM, 32, 32> ARGS;
#define LOCAL_DISPATCH(FN, ARGS)                         \
    do {                                                 \
        if (norm == 1) {                                 \
            LOCAL_DISPATCH_N(FN, ARGS, 1)                \
        } else if (norm == 2) {                          \
            LOCAL_DISPATCH_N(FN, ARGS, 2)                \
        } else {                                         \
            LOCAL_DISPATCH_N(FN, ARGS, 3)                \
        }                                                \
    } while (0)

int dispatch_table(const Ctx& c, TableArgs& a, const Knots& kn, int norm, int d) {
    LOCAL_DISPATCH(launch_table, (c, a, kn));
}
int dispatch_eval(const Ctx& c, EvalArgs& a, const Knots& kn, int norm, int d) {
    LOCAL_DISPATCH(launch_eval, (c, a, kn));
}

}  // namespace

int launch_distance_quantiles(const Ctx& c, const float* X, int64_t N, const Xform& xf, int norm,
                              const int32_t* pair_i, const int32_t* pair_k, int64_t S, int J, float* knots,
                              int* bad_dev) {
    const int s = static_cast<int>(S);
    Workspace wd, ws, wt;
    int rc;
    if ((rc = wd.alloc(sizeof(float) * static_cast<size_t>(S), c.stream))) return rc;
    if ((rc = ws.alloc(sizeof(float) * static_cast<size_t>(S), c.stream))) return rc;
    size_t bytes = 0;
    LIPFIT_CUDA(cub::DeviceRadixSort::SortKeys(nullptr, bytes, static_cast<const float*>(nullptr),
                                               static_cast<float*>(nullptr), s, 0, 32, c.stream));
    if ((rc = wt.alloc(bytes, c.stream))) return rc;
    local_pair_dist_kernel<<<(s + 255) / 256, 256, 0, c.stream>>>(X, static_cast<int>(N), xf, norm, pair_i, pair_k,
                                                                 s, wd.as<float>(), bad_dev);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    LIPFIT_CUDA(cub::DeviceRadixSort::SortKeys(wt.p, bytes, wd.as<float>(), ws.as<float>(), s, 0, 32, c.stream));
    local_pick_kernel<<<1, 32 * ((J + 31) / 32), 0, c.stream>>>(ws.as<float>(), S, J, knots);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

int launch_local_lipschitz(const Ctx& c, const float* X, const float* y, int64_t N64, const Xform& xf, int norm,
                           const float* knots_host, float* table) {
    const int N = static_cast<int>(N64);
    const int dp = local_dp(xf.d);
    RecLayout lay{dp + 4, dp};
    Workspace wrec, wtab, wnn;
    int rc;
    if ((rc = wrec.alloc(sizeof(float) * static_cast<size_t>(N) * lay.rf, c.stream))) return rc;
    if ((rc = wtab.alloc(sizeof(uint32_t) * static_cast<size_t>(N) * kJ, c.stream))) return rc;
    if ((rc = wnn.alloc(sizeof(unsigned long long) * static_cast<size_t>(N), c.stream))) return rc;
    if ((rc = launch_prepack(c, X, y, nullptr, N, xf, lay, wrec.as<float>()))) return rc;
    LIPFIT_CUDA(cudaMemsetAsync(wtab.p, 0, sizeof(uint32_t) * static_cast<size_t>(N) * kJ, c.stream));
    LIPFIT_CUDA(cudaMemsetAsync(wnn.p, 0xFF, sizeof(unsigned long long) * static_cast<size_t>(N), c.stream));
    Knots kn;  // L2: squared knots, correctly rounded (the kernel bins squared distances)
    for (int j = 0; j < kJ; ++j)
        kn.t[j] = norm == 2 ? static_cast<float>(static_cast<double>(knots_host[j]) * knots_host[j]) : knots_host[j];
    local_lut_params(kn);
    TableArgs a{};
    a.rec = wrec.as<float>();
    a.tab = wtab.as<uint32_t>();
    a.nn = wnn.as<unsigned long long>();
    a.N = N;
    if ((rc = dispatch_table(c, a, kn, norm, xf.d))) return rc;
    const int ne = N * kJ;
    local_table_final_kernel<<<(ne + 255) / 256, 256, 0, c.stream>>>(a.tab, a.nn, N, table);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

int launch_values_local(const Ctx& c, const float* X, const float* y, int64_t N64, const float* Xq, int64_t Q64,
                        const Xform& xf, int norm, const float* knots_host, const float* table, float* upper,
                        float* lower, float* g) {
    const int N = static_cast<int>(N64), Q = static_cast<int>(Q64);
    const int dp = local_dp(xf.d);
    const bool packed = norm == 2 && xf.d <= 8;  // packed f32x2 kernel: duplicated coordinates
    const int de = (xf.d + 1) & ~1;
    const int rf = packed ? 2 * de + 4 + kJ : dp + 4 + kJ;
    Workspace wrec, wkeys;
    int rc;
    if ((rc = wrec.alloc(sizeof(float) * static_cast<size_t>(N) * rf, c.stream))) return rc;
    if ((rc = wkeys.alloc(sizeof(uint32_t) * 2 * static_cast<size_t>(Q), c.stream))) return rc;
    if (packed)
        local_eval_pack2_kernel<<<(N + 255) / 256, 256, 0, c.stream>>>(X, y, table, N, xf, de, wrec.as<float>());
    else
        local_eval_pack_kernel<<<(N + 255) / 256, 256, 0, c.stream>>>(X, y, table, N, xf, dp, wrec.as<float>());
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    Knots kn;  // L2: squared knots, correctly rounded (the kernel compares squared distances with them)
    for (int j = 0; j < kJ; ++j)
        kn.t[j] = norm == 2 ? static_cast<float>(static_cast<double>(knots_host[j]) * knots_host[j]) : knots_host[j];
    local_lut_params(kn);
    EvalArgs a{};
    a.rec = wrec.as<float>();
    a.Xq = Xq;
    a.keyU = wkeys.as<uint32_t>();
    a.keyL = a.keyU + Q;
    a.N = N;
    a.Q = Q;
    a.d = xf.d;
    a.xf = xf;
    LIPFIT_CUDA(cudaMemsetAsync(a.keyU, 0xFF, sizeof(uint32_t) * Q, c.stream));
    LIPFIT_CUDA(cudaMemsetAsync(a.keyL, 0x00, sizeof(uint32_t) * Q, c.stream));
    if ((rc = packed ? dispatch_eval_packed(c, a, kn, xf.d) : dispatch_eval(c, a, kn, norm, xf.d))) return rc;
    local_eval_final_kernel<<<(Q + 255) / 256, 256, 0, c.stream>>>(a.keyU, a.keyL, Q, upper, lower, g);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

}  // namespace lipfit
