// smooth.cu -- step a4: all-pairs objective and gradient of Eq.(7) PAPER.md:197,
// distances recomputed on the fly: nothing of size N x N is ever stored (the paper's precomputed
// d_ik / y_k - y_i matrices are its memory wall).
//
// With z = y + eps, D_ik = d_s(x^k, x^i) and V_ik = (z_i - z_k - M D_ik)_+ (reading R12):
//   F = ||eps||^2 / p + 2 sum_{i != k} V_ik^2,      dF/deps_i = 2 eps_i / p + 4 sum_k (V_ik - V_ki).
// V_ik > 0 needs z_i > z_k, so of the two ordered pairs (i,k), (k,i) at most one contributes.  Every
// evaluation therefore
//   (1) sorts the data by z (cub radix sort of N keys: microseconds) and gathers the packed records
//       [M x'_0 .. M x'_{d-1}, z] in that order (coordinates are pre-multiplied by M once per call);
//   (2) visits every UNORDERED pair once -- row i against the data k < i of the sorted order, where
//       only V_ik can be non-zero: one one-sided distance per pair, no sign select;
//   (3) pre-filters on the squared quantity (L2: sum (M u_j)^2 < (z_i - z_k)^2, no square root); the
//       rare surviving pairs (~1e-5 of all) take a slow path that forms V, adds V^2 to F, +V to row i
//       and -V to row k.  Gradient sums are kept in fixed point (64-bit integer atomics): exact, hence
//       independent of the order of the atomics -- an evaluation is bit-reproducible.  The scale is
//       2^e, e = min(40, 62 - ceil(log2(N (z_max - z_min)))), chosen per evaluation from the sorted z:
//       every V is <= z_max - z_min, so no row sum can reach 2^62 whatever the magnitude of the data.
// Kernel shape as in bounds.cu: R rows per thread in registers, data tiles through shared memory via
// the TMA engine (decoupled 4-stage pipe); work items (row block, data chunk) of the lower triangle
// are handed out by an atomic counter.
#include <cub/device/device_radix_sort.cuh>

#include <type_traits>

#include "kernels.h"

#pragma nv_diag_suppress 128  // MODE 1 leaves the item loop before the smoothing-only reductions

namespace lipfit {

constexpr int kSmThreads = 128;
constexpr int kSmWarps = kSmThreads / 32;
constexpr int kSmStages = 4;
constexpr int kSmChunk = 4096;  // data records per work item (multiple of every tile size)
constexpr int kFixMaxExp = 40;  // finest fixed-point scale of the gradient sums (2^-40)

struct SmoothArgs {
    const float* rec;         // sorted records [N][RF]
    unsigned long long* gfix; // [N] sum_k (V_ik - V_ki) of sorted position i, fixed point with scale fix[0]
    const double* fix;        // [2] fixed-point scale 2^e and its inverse (written by the gather kernel)
    double* fpart;            // [nitems] sum of V^2 over the item
    float* vpart;             // [nitems] max V over the item
    int* counter;             // work counter
    int N, nrb, maxc, nitems;
    // MODE 1 only
    unsigned long long* lmax;  // bits of the running maximum ratio (a non-negative double)
    const uint32_t* amax;      // bits of max |x'| over the packed coordinates (written by the gather)
    const float* X;            // original coordinates and
    const int32_t* perm;       // sorted position -> original index, for the exact fp64 ratio
    int norm;
    Xform xf;
};

// MODE 0: smoothing objective / gradient (records carry M-scaled coordinates and z).
// MODE 1: smallest consistent Lipschitz constant max (y_i - y_k) / d_s(x^k, x^i): same
//         sorted lower-triangle sweep (records carry the plain coordinates and y); the pre-filter is
//         "this pair beats the running maximum", which becomes rarer and rarer.
constexpr int kModeSmooth = 0, kModeLipConst = 1;

template <int RF>
__host__ __device__ constexpr int smooth_tile_records() {
    return RF <= 8 ? 256 : (RF <= 20 ? 128 : 64);
}

template <int RF>
__device__ __forceinline__ void smooth_load_record(const float* s, float* x) {
#pragma unroll
    for (int c = 0; c < RF / 4; ++c) {
        float4 v = reinterpret_cast<const float4*>(s)[c];
        x[4 * c + 0] = v.x;
        x[4 * c + 1] = v.y;
        x[4 * c + 2] = v.z;
        x[4 * c + 3] = v.w;
    }
}

// Slow path for one datum k (sorted position kpos): rows whose pre-filter passed form V.
template <class Acc, int R>
__device__ __forceinline__ void smooth_hit(const SmoothArgs& a, const float (&acc)[R], const float (&dz)[R],
                                           const bool (&pass)[R], int kpos, long long (&grow)[R],
                                           double& fd, float& vmax) {
    long long col = 0;
    const double kFix = __ldg(a.fix);
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if (pass[r]) {
            const float D = Acc::NORM == 2 ? __fsqrt_rn(acc[r]) : acc[r];  // M * distance
            const float V = dz[r] - D;
            if (V > 0.f) {
                fd += static_cast<double>(V) * static_cast<double>(V);
                const long long vf = __double2ll_rn(static_cast<double>(V) * kFix);
                grow[r] += vf;
                col += vf;
                vmax = fmaxf(vmax, V);
            }
        }
    }
    if (col != 0) atomicAdd(a.gfix + kpos, static_cast<unsigned long long>(-col));
}

// MODE 1 slow path: EXACT ratio (fp64, from the original fp32 inputs) of the pairs that passed the
// conservative fp32 filter.  lcur (fp32, rounded down) only feeds the filter; lbest is the result.
__device__ __forceinline__ double lipconst_exact_distance(const float* xi, const float* xk, const Xform& xf,
                                                          int norm) {
    double acc = 0.0;
    for (int j = 0; j < xf.d; ++j) {
        const int o = xf.perm[j];
        const double dlt = static_cast<double>(xf.sw[j]) *
                           (static_cast<double>(xi[o]) - static_cast<double>(xk[o]));
        const double comp = (j < xf.dU) ? fabs(dlt) : fmax(dlt, 0.0);
        if (norm == 1) acc += comp;
        else if (norm == 2) acc += comp * comp;
        else acc = fmax(acc, comp);
    }
    return norm == 2 ? sqrt(acc) : acc;
}

template <int R>
__device__ __forceinline__ void lipconst_hit(const SmoothArgs& a, const float (&zi)[R], float zk,
                                             const int (&ipos)[R], int kpos, const bool (&pass)[R],
                                             float& lcur, double& lbest) {
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if (pass[r]) {
            const double dzd = static_cast<double>(zi[r]) - static_cast<double>(zk);
            if (dzd > 0.0) {
                const float* xi = a.X + static_cast<size_t>(a.perm[ipos[r]]) * a.xf.d;
                const float* xk = a.X + static_cast<size_t>(a.perm[kpos]) * a.xf.d;
                const double D = lipconst_exact_distance(xi, xk, a.xf, a.norm);
                const double ratio = D > 0.0 ? dzd / D : __longlong_as_double(0x7ff0000000000000LL);
                lbest = fmax(lbest, ratio);
                lcur = fmaxf(lcur, __double2float_rd(ratio));
            }
        }
    }
}

template <class Acc, int R, int MODE>
__global__ void __launch_bounds__(kSmThreads, 4)
smooth_pairs_kernel(const SmoothArgs a, const FreeFlags ff) {
    constexpr int THREADS = kSmThreads;
    constexpr int D = Acc::D;
    constexpr int RF = Acc::RF;
    constexpr int TILE = smooth_tile_records<RF>();
    constexpr int ST = kSmStages;
    constexpr int RB = THREADS * R;
    __shared__ __align__(128) float sbuf[ST * TILE * RF];
    __shared__ __align__(8) uint64_t bars[ST];
    __shared__ int done[ST];
    __shared__ int s_item;
    __shared__ double redf[kSmWarps];
    __shared__ float redv[kSmWarps];
    if (threadIdx.x == 0) {
#pragma unroll
        for (int b = 0; b < ST; ++b) {
            mbar_init(&bars[b], 1);
            done[b] = 0;
        }
        mbar_fence_init();
    }
    uint32_t phase = 0;
    for (;;) {
        __syncthreads();  // s_item and the reduction scratch of the previous item are free
        if (threadIdx.x == 0) s_item = atomicAdd(a.counter, 1);
        __syncthreads();
        const int item = s_item;
        if (item >= a.nitems) break;
        const int rb = a.nrb - 1 - item / a.maxc;
        const int ch = item - (item / a.maxc) * a.maxc;
        const int row0 = rb * RB;
        const int rowend = min(a.N, row0 + RB);
        const int begin = ch * kSmChunk;
        const int end = min(begin + kSmChunk, rowend - 1);  // k < i <= rowend - 1
        if (begin >= end) {
            if (threadIdx.x == 0) {
                a.fpart[item] = 0.0;
                a.vpart[item] = 0.f;
            }
            continue;
        }
        // ---- rows of this block -> registers ----
        float xi[R][D], zi[R];
        int ipos[R];
        long long grow[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int i = row0 + r * THREADS + static_cast<int>(threadIdx.x);
            ipos[r] = i;
            grow[r] = 0;
            if (i < a.N) {
                const float* src = a.rec + static_cast<size_t>(i) * RF;
#pragma unroll
                for (int j = 0; j < D; ++j) xi[r][j] = __ldg(src + j);
                zi[r] = __ldg(src + Acc::VSLOT);
            } else {  // padding row: an infinite distance to everything, never passes the filter
#pragma unroll
                for (int j = 0; j < D; ++j) xi[r][j] = 1e30f;
                zi[r] = __int_as_float(0xff800000);  // -inf: z_i - z_k is never positive
            }
        }
        double fd = 0.0;
        float vmax = 0.f;
        float lcur = 0.f;    // MODE 1: running maximum ratio known to this thread, rounded down (filter)
        double lbest = 0.0;  //         and exactly (result)
        RecordPipe<TILE, ST, kSmWarps> rs(a.rec, RF, begin, end, sbuf, bars, done, &phase);
        for (int t = 0; t < rs.ntiles; ++t) {
            const float* s = rs.acquire(t);
            const int n = rs.count(t);
            const int base = begin + t * TILE;
            const bool below = (base + n <= row0);  // every k of the tile precedes every row of the block
            // MODE 1 filter: the pair can beat the running maximum L only if  L * D < dz.  With the fp32
            // distance D' (|D' - D| <= eta from the rounding of the weighted coordinates, plus a relative
            // (D+6) 2^-24 from the accumulation) the conservative form is  L (1-rel) D' < dz + L eta.
            float lthr = 0.f, leta = 0.f;
            auto refresh = [&]() {
                const float rel = 1.f - static_cast<float>(D + 6) * 1.1920929e-7f;
                const float cn = Acc::NORM == 1 ? static_cast<float>(a.xf.d)
                                                : (Acc::NORM == 2 ? sqrtf(static_cast<float>(a.xf.d)) : 1.f);
                const float eta = cn * 1.1920929e-7f * __uint_as_float(*a.amax);
                const float l = lcur * rel;
                lthr = Acc::NORM == 2 ? l * l : l;
                leta = lcur * eta;
            };
            if (MODE == kModeLipConst) {  // share the maximum between threads once per tile
                const double g = __longlong_as_double(
                    static_cast<long long>(*reinterpret_cast<volatile unsigned long long*>(a.lmax)));
                lcur = fmaxf(lcur, __double2float_rd(g));
                if (isinf(lcur)) lcur = 3.0e38f;  // keeps the filter arithmetic finite; the result stays +inf
                refresh();
            }
            // Two copies of the loop: tiles strictly below the diagonal (the vast majority) need neither
            // the index test nor the sign test -- sorted order guarantees k < i and z_k <= z_i there.
            auto sweep = [&](auto below_c) {
            constexpr bool BELOW = decltype(below_c)::value;
            for (int j = 0; j < n; ++j) {
                float x[RF];
                smooth_load_record<RF>(s + j * RF, x);
                const float zk = x[Acc::VSLOT];
                float acc[R], dz[R];
                bool pass[R];
                bool hit = false;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    acc[r] = Acc::run_u(xi[r], x, ff);
                    dz[r] = zi[r] - zk;
                    const float lhs = MODE == kModeLipConst ? acc[r] * lthr : acc[r];
                    if (MODE == kModeLipConst) dz[r] += leta;
                    pass[r] = Acc::NORM == 2 ? (lhs < dz[r] * dz[r]) : (lhs < dz[r]);
                    if (!BELOW) pass[r] = pass[r] && (base + j < ipos[r]) && (dz[r] > 0.f);
                    hit |= pass[r];
                }
                if (__any_sync(0xffffffffu, hit)) {  // warp-uniform, rare
                    if (MODE == kModeSmooth) {
                        smooth_hit<Acc, R>(a, acc, dz, pass, base + j, grow, fd, vmax);
                    } else {
                        lipconst_hit<R>(a, zi, zk, ipos, base + j, pass, lcur, lbest);
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1)
                            lcur = fmaxf(lcur, __shfl_xor_sync(0xffffffffu, lcur, o));
                        if (isinf(lcur)) lcur = 3.0e38f;
                        refresh();
                    }
                }
            }
            };
            if (below) sweep(std::true_type{});
            else sweep(std::false_type{});
            if (MODE == kModeLipConst) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) lbest = fmax(lbest, __shfl_xor_sync(0xffffffffu, lbest, o));
                if ((threadIdx.x & 31) == 0)
                    atomicMax(a.lmax, static_cast<unsigned long long>(__double_as_longlong(lbest)));
            }
            rs.release(t);
        }
        if (MODE == kModeLipConst) continue;  // nothing else to reduce
        // ---- row sums -> fixed-point atomics; per-item objective partial (fixed order) ----
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (grow[r] != 0) atomicAdd(a.gfix + ipos[r], static_cast<unsigned long long>(grow[r]));
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            fd += __shfl_xor_sync(0xffffffffu, fd, o);
            vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
        }
        if ((threadIdx.x & 31) == 0) {
            redf[threadIdx.x >> 5] = fd;
            redv[threadIdx.x >> 5] = vmax;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            double f = 0.0;
            float v = 0.f;
            for (int w = 0; w < kSmWarps; ++w) {
                f += redf[w];
                v = fmaxf(v, redv[w]);
            }
            a.fpart[item] = f;
            a.vpart[item] = v;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Packed-f32x2 smoothing sweep (L2, all DC coordinates constrained; config 5's shape): a thread keeps
// 4 PAIRS of rows as (x_i, x_i') register pairs, the sorted records are stored duplicated (x, x), so the
// subtractions, squared accumulations and the (z_i - z_k)^2 side of the filter are FADD2 / FFMA2 / FMUL2;
// the positive parts stay scalar FMNMX.  12 issue slots per visited pair instead of 20.5.
// Same work items, slow path, reductions and results as smooth_pairs_kernel<SpecAcc<2,0,DC>, 8, 0>.
// ---------------------------------------------------------------------------------------------
template <int DC>
__global__ void __launch_bounds__(kSmThreads, 3)
smooth_pairs_packed_kernel(const SmoothArgs a) {
    using Acc = SpecAcc<2, 0, DC>;
    constexpr int THREADS = kSmThreads;
    constexpr int RP = 4, R = 2 * RP;
    constexpr int RFL = record_floats(DC);  // logical floats per record: x'_0.., z, pad
    constexpr int RF = 2 * RFL;             // physical (duplicated)
    constexpr int TILE = smooth_tile_records<RF>();
    constexpr int ST = kSmStages;
    constexpr int RB = THREADS * R;
    __shared__ __align__(128) float sbuf[ST * TILE * RF];
    __shared__ __align__(8) uint64_t bars[ST];
    __shared__ int done[ST];
    __shared__ int s_item;
    __shared__ double redf[kSmWarps];
    __shared__ float redv[kSmWarps];
    if (threadIdx.x == 0) {
#pragma unroll
        for (int b = 0; b < ST; ++b) {
            mbar_init(&bars[b], 1);
            done[b] = 0;
        }
        mbar_fence_init();
    }
    uint32_t phase = 0;
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_item = atomicAdd(a.counter, 1);
        __syncthreads();
        const int item = s_item;
        if (item >= a.nitems) break;
        const int rb = a.nrb - 1 - item / a.maxc;
        const int ch = item - (item / a.maxc) * a.maxc;
        const int row0 = rb * RB;
        const int rowend = min(a.N, row0 + RB);
        const int begin = ch * kSmChunk;
        const int end = min(begin + kSmChunk, rowend - 1);  // k < i <= rowend - 1
        if (begin >= end) {
            if (threadIdx.x == 0) {
                a.fpart[item] = 0.0;
                a.vpart[item] = 0.f;
            }
            continue;
        }
        // ---- row pairs of this block -> registers: pair rp = rows (2 rp, 2 rp + 1) of the thread ----
        float2 xi[RP][DC], zi[RP];
        int ipos[R];
        long long grow[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int i = row0 + r * THREADS + static_cast<int>(threadIdx.x);
            ipos[r] = i;
            grow[r] = 0;
            float v[DC], z;
            if (i < a.N) {
                const float* src = a.rec + static_cast<size_t>(i) * RF;
#pragma unroll
                for (int j = 0; j < DC; ++j) v[j] = __ldg(src + 2 * j);
                z = __ldg(src + 2 * DC);
            } else {  // padding row: an infinite distance to everything, never passes the filter
#pragma unroll
                for (int j = 0; j < DC; ++j) v[j] = 1e30f;
                z = __int_as_float(0xff800000);
            }
#pragma unroll
            for (int j = 0; j < DC; ++j) {
                if (r & 1) xi[r >> 1][j].y = v[j];
                else xi[r >> 1][j].x = v[j];
            }
            if (r & 1) zi[r >> 1].y = z;
            else zi[r >> 1].x = z;
        }
        double fd = 0.0;
        float vmax = 0.f;
        RecordPipe<TILE, ST, kSmWarps> rs(a.rec, RF, begin, end, sbuf, bars, done, &phase);
        for (int t = 0; t < rs.ntiles; ++t) {
            const float* s = rs.acquire(t);
            const int n = rs.count(t);
            const int base = begin + t * TILE;
            const bool below = (base + n <= row0);
            auto sweep = [&](auto below_c) {
                constexpr bool BELOW = decltype(below_c)::value;
                for (int j = 0; j < n; ++j) {
                    float2 x[RFL];
#pragma unroll
                    for (int c = 0; c < RF / 4; ++c) {
                        const float4 v = reinterpret_cast<const float4*>(s + j * RF)[c];
                        x[2 * c] = make_float2(v.x, v.y);
                        x[2 * c + 1] = make_float2(v.z, v.w);
                    }
                    float2 acc[RP], dz[RP];
                    bool hit = false;
                    bool pass[R];
#pragma unroll
                    for (int rp = 0; rp < RP; ++rp) {
                        float2 s2 = make_float2(0.f, 0.f);
#pragma unroll
                        for (int c = 0; c < DC; ++c) {
                            const float2 dlt = __fadd2_rn(xi[rp][c], make_float2(-x[c].x, -x[c].y));
                            const float2 rl = make_float2(fmaxf(dlt.x, 0.f), fmaxf(dlt.y, 0.f));
                            s2 = __ffma2_rn(rl, rl, s2);
                        }
                        acc[rp] = s2;
                        dz[rp] = __fadd2_rn(zi[rp], make_float2(-x[DC].x, -x[DC].y));
                        const float2 dzz = __fmul2_rn(dz[rp], dz[rp]);
                        pass[2 * rp] = s2.x < dzz.x;
                        pass[2 * rp + 1] = s2.y < dzz.y;
                        if (!BELOW) {
                            pass[2 * rp] = pass[2 * rp] && (base + j < ipos[2 * rp]) && (dz[rp].x > 0.f);
                            pass[2 * rp + 1] = pass[2 * rp + 1] && (base + j < ipos[2 * rp + 1]) && (dz[rp].y > 0.f);
                        }
                        hit |= pass[2 * rp] | pass[2 * rp + 1];
                    }
                    if (__any_sync(0xffffffffu, hit)) {  // warp-uniform, rare
                        float accs[R], dzs[R];
#pragma unroll
                        for (int rp = 0; rp < RP; ++rp) {
                            accs[2 * rp] = acc[rp].x;
                            accs[2 * rp + 1] = acc[rp].y;
                            dzs[2 * rp] = dz[rp].x;
                            dzs[2 * rp + 1] = dz[rp].y;
                        }
                        smooth_hit<Acc, R>(a, accs, dzs, pass, base + j, grow, fd, vmax);
                    }
                }
            };
            if (below) sweep(std::true_type{});
            else sweep(std::false_type{});
            rs.release(t);
        }
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (grow[r] != 0) atomicAdd(a.gfix + ipos[r], static_cast<unsigned long long>(grow[r]));
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            fd += __shfl_xor_sync(0xffffffffu, fd, o);
            vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
        }
        if ((threadIdx.x & 31) == 0) {
            redf[threadIdx.x >> 5] = fd;
            redv[threadIdx.x >> 5] = vmax;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            double f = 0.0;
            float v = 0.f;
            for (int w = 0; w < kSmWarps; ++w) {
                f += redf[w];
                v = fmaxf(v, redv[w]);
            }
            a.fpart[item] = f;
            a.vpart[item] = v;
        }
    }
}

// z = y + eps and the identity permutation (sort input)
__global__ void __launch_bounds__(256)
smooth_z_kernel(const float* __restrict__ y, const float* __restrict__ eps, int N, float* __restrict__ z,
                int32_t* __restrict__ idx) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    z[k] = y[k] + (eps ? eps[k] : 0.f);
    idx[k] = k;
}

// sorted records: coordinates of datum perm[j] (already M-scaled, from the unsorted base records),
// value slot = z_sorted[j]; also clears the gradient accumulator of position j.
__global__ void __launch_bounds__(256)
smooth_gather_kernel(const float* __restrict__ base, const int32_t* __restrict__ perm,
                     const float* __restrict__ zs, int N, int rf, int vslot, float* __restrict__ rec,
                     unsigned long long* __restrict__ gfix, uint32_t* __restrict__ amax, int dup,
                     double* __restrict__ fix) {
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    if (j == 0 && fix) {
        // fixed-point scale of this evaluation's gradient sums: |sum_k V| <= (N-1) (z_max - z_min) < 2^ex
        const double r = static_cast<double>(N) * (static_cast<double>(zs[N - 1]) - static_cast<double>(zs[0]));
        int ex = 0;
        if (r > 0.0 && r < 1.0e300) (void)frexp(r, &ex);
        int e = 62 - ex;
        if (e > kFixMaxExp) e = kFixMaxExp;
        fix[0] = ldexp(1.0, e);
        fix[1] = ldexp(1.0, -e);
    }
    if (dup) {  // duplicated layout (x, x) for the packed kernel: 2 rf floats per record
        const float* src = base + static_cast<size_t>(perm[j]) * rf;
        float4* dst = reinterpret_cast<float4*>(rec + static_cast<size_t>(j) * 2 * rf);
        for (int c = 0; c < rf / 2; ++c) {
            const float v0 = (2 * c == vslot) ? zs[j] : src[2 * c];
            const float v1 = (2 * c + 1 == vslot) ? zs[j] : src[2 * c + 1];
            dst[c] = make_float4(v0, v0, v1, v1);
        }
        gfix[j] = 0ull;
        return;
    }
    float am = 0.f;
    const float4* src = reinterpret_cast<const float4*>(base + static_cast<size_t>(perm[j]) * rf);
    float4* dst = reinterpret_cast<float4*>(rec + static_cast<size_t>(j) * rf);
    for (int c = 0; c < rf / 4; ++c) {
        float4 v = src[c];
        if (amax) am = fmaxf(am, fmaxf(fmaxf(fabsf(v.x), fabsf(v.y)), fmaxf(fabsf(v.z), fabsf(v.w))));
        const int o = vslot - 4 * c;
        if (o == 0) v.x = zs[j];
        if (o == 1) v.y = zs[j];
        if (o == 2) v.z = zs[j];
        if (o == 3) v.w = zs[j];
        dst[c] = v;
    }
    gfix[j] = 0ull;
    if (amax) atomicMax(amax, __float_as_uint(am));  // MODE 1 only (base value slots are zero there)
}

__global__ void lipconst_final_kernel(const unsigned long long* __restrict__ lmax, float* __restrict__ L) {
    *L = static_cast<float>(__longlong_as_double(static_cast<long long>(*lmax)));
}

// grad[perm[j]] = 2 eps / p + 4 * gfix[j] / scale; per-block partial of sum eps^2.
__global__ void __launch_bounds__(256)
smooth_grad_kernel(const unsigned long long* __restrict__ gfix, const double* __restrict__ fix,
                   const int32_t* __restrict__ perm, int N,
                   const float* __restrict__ eps, float p, float* __restrict__ grad,
                   double* __restrict__ e2part) {
    __shared__ double red[8];
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    double e = 0.0;
    if (j < N) {
        const int i = perm[j];
        const double s = static_cast<double>(static_cast<long long>(gfix[j])) * fix[1];
        e = eps ? static_cast<double>(eps[i]) : 0.0;
        if (grad) grad[i] = static_cast<float>(2.0 * e / static_cast<double>(p) + 4.0 * s);
    }
    double e2 = e * e;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e2 += __shfl_xor_sync(0xffffffffu, e2, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = e2;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += red[w];
        e2part[blockIdx.x] = t;
    }
}

// Single block, fixed order: F = sum(e2part)/p + 2 sum(fpart); maxviol = max(vpart).
__global__ void __launch_bounds__(256)
smooth_final_kernel(const double* __restrict__ fpart, const float* __restrict__ vpart, int nitems,
                    const double* __restrict__ e2part, int nblk, float p, double* __restrict__ F,
                    double* __restrict__ maxviol) {
    __shared__ double rf_[256], re_[256], rv_[256];
    double f = 0.0, e = 0.0, v = 0.0;
    for (int t = threadIdx.x; t < nitems; t += 256) {
        f += fpart[t];
        v = fmax(v, static_cast<double>(vpart[t]));
    }
    for (int b = threadIdx.x; b < nblk; b += 256) e += e2part[b];
    rf_[threadIdx.x] = f;
    re_[threadIdx.x] = e;
    rv_[threadIdx.x] = v;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) {
            rf_[threadIdx.x] += rf_[threadIdx.x + o];
            re_[threadIdx.x] += re_[threadIdx.x + o];
            rv_[threadIdx.x] = fmax(rv_[threadIdx.x], rv_[threadIdx.x + o]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        if (F) *F = re_[0] / static_cast<double>(p) + 2.0 * rf_[0];
        if (maxviol) *maxviol = rv_[0];
    }
}

namespace {

template <class Acc, int R, int MODE>
int launch_pairs(const Ctx& c, SmoothArgs& a, const FreeFlags& ff) {
    auto kern = smooth_pairs_kernel<Acc, R, MODE>;
    int occ = 0;
    LIPFIT_CUDA(occupancy_of(&occ, kern, kSmThreads, 0));
    if (occ < 1) occ = 1;
    const int slots = c.num_sms * occ;
    const int grid = a.nitems < slots ? a.nitems : slots;
    KernelTimer kt(MODE == kModeSmooth ? TK_SMOOTH_PAIRS : TK_LIPCONST_PAIRS, c.stream);
    kern<<<grid, kSmThreads, 0, c.stream>>>(a, ff);
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

int smooth_dp(int d) { return d <= 4 ? 4 : (d <= 8 ? 8 : (d <= 16 ? 16 : 32)); }
bool is_spec(const Xform& xf, int norm) {
    return (norm == 2 && xf.dU == 0 && xf.dC == 5) || (norm == 2 && xf.dU == 2 && xf.dC == 0);
}
int smooth_rows(const Xform& xf, int norm) {  // R of the kernel that will run
    if (is_spec(xf, norm)) return 8;
    const int dp = smooth_dp(xf.d);
    return dp <= 8 ? 4 : (dp <= 16 ? 2 : 1);
}

template <int MODE>
int dispatch_pairs(const Ctx& c, SmoothArgs& a, const FreeFlags& ff, const Xform& xf, int norm) {
    int rc = LIPFIT_OK;
#define GO(ACC, RR) rc = launch_pairs<ACC, RR, MODE>(c, a, ff)
    using S205 = SpecAcc<2, 0, 5>;
    using S220 = SpecAcc<2, 2, 0>;
    using G14 = GenAcc<1, 4>;
    using G18 = GenAcc<1, 8>;
    using G116 = GenAcc<1, 16>;
    using G132 = GenAcc<1, 32>;
    using G24 = GenAcc<2, 4>;
    using G28 = GenAcc<2, 8>;
    using G216 = GenAcc<2, 16>;
    using G232 = GenAcc<2, 32>;
    using G34 = GenAcc<3, 4>;
    using G38 = GenAcc<3, 8>;
    using G316 = GenAcc<3, 16>;
    using G332 = GenAcc<3, 32>;
    const int dp = smooth_dp(xf.d);
    if (norm == 2 && xf.dU == 0 && xf.dC == 5) GO(S205, 8);
    else if (norm == 2 && xf.dU == 2 && xf.dC == 0) GO(S220, 8);
    else if (norm == 1) {
        if (dp == 4) GO(G14, 4);
        else if (dp == 8) GO(G18, 4);
        else if (dp == 16) GO(G116, 2);
        else GO(G132, 1);
    } else if (norm == 2) {
        if (dp == 4) GO(G24, 4);
        else if (dp == 8) GO(G28, 4);
        else if (dp == 16) GO(G216, 2);
        else GO(G232, 1);
    } else {
        if (dp == 4) GO(G34, 4);
        else if (dp == 8) GO(G38, 4);
        else if (dp == 16) GO(G316, 2);
        else GO(G332, 1);
    }
#undef GO
    return rc;
}

// NEXT-3 with the symmetric distance (no constrained coordinate: the paper's lipschitz_constant())
// and d <= 8: compile-time pair arithmetic over exactly the d coordinates (2 lane-ops per coordinate) instead of
// the flag arithmetic over DP padded ones (4 per padded coordinate).
bool lipconst_spec(const Xform& xf) { return xf.dC == 0 && xf.d <= 8; }

template <int NORM>
int dispatch_lipconst_spec(const Ctx& c, SmoothArgs& a, const FreeFlags& ff, int d) {
    switch (d) {
        case 1: return launch_pairs<SpecAcc<NORM, 1, 0>, 8, kModeLipConst>(c, a, ff);
        case 2: return launch_pairs<SpecAcc<NORM, 2, 0>, 8, kModeLipConst>(c, a, ff);
        case 3: return launch_pairs<SpecAcc<NORM, 3, 0>, 8, kModeLipConst>(c, a, ff);
        case 4: return launch_pairs<SpecAcc<NORM, 4, 0>, 8, kModeLipConst>(c, a, ff);
        case 5: return launch_pairs<SpecAcc<NORM, 5, 0>, 8, kModeLipConst>(c, a, ff);
        case 6: return launch_pairs<SpecAcc<NORM, 6, 0>, 4, kModeLipConst>(c, a, ff);
        case 7: return launch_pairs<SpecAcc<NORM, 7, 0>, 4, kModeLipConst>(c, a, ff);
        default: return launch_pairs<SpecAcc<NORM, 8, 0>, 4, kModeLipConst>(c, a, ff);
    }
}

}  // namespace

RecLayout lipconst_layout(const Xform& xf, int norm) {
    if (lipconst_spec(xf)) return RecLayout{record_floats(xf.d), xf.d};
    return smooth_layout(xf, norm);
}

RecLayout smooth_layout(const Xform& xf, int norm) {
    if (is_spec(xf, norm)) return RecLayout{record_floats(xf.d), xf.d};
    int dp = smooth_dp(xf.d);
    return RecLayout{dp + 4, dp};
}

int launch_smooth_objective(const Ctx& c, const float* base, const float* y, const float* eps, int64_t N64,
                            const Xform& xf, int norm, float p, double* F_dev, float* grad,
                            double* maxviol_dev) {
    const int N = static_cast<int>(N64);
    const RecLayout lay = smooth_layout(xf, norm);
    const int R = smooth_rows(xf, norm);
    const bool packed = (norm == 2 && xf.dU == 0 && xf.dC == 5);  // packed-f32x2 kernel, duplicated records
    SmoothArgs a{};
    a.N = N;
    a.nrb = (N + kSmThreads * R - 1) / (kSmThreads * R);
    a.maxc = (N + kSmChunk - 1) / kSmChunk;
    a.nitems = a.nrb * a.maxc;
    const int nblk = (N + 255) / 256;
    const size_t n = static_cast<size_t>(N);

    // ---- workspace ----
    size_t sort_bytes = 0;
    LIPFIT_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, sort_bytes, static_cast<const float*>(nullptr),
                                                static_cast<float*>(nullptr),
                                                static_cast<const int32_t*>(nullptr),
                                                static_cast<int32_t*>(nullptr), N, 0, 32, c.stream));
    Workspace wz, wzs, wi, wperm, wsort, wrec, wg, wf, wv, we, wc, wfix;
    int rc;
    if ((rc = wfix.alloc(sizeof(double) * 2, c.stream))) return rc;
    if ((rc = wz.alloc(sizeof(float) * n, c.stream))) return rc;
    if ((rc = wzs.alloc(sizeof(float) * n, c.stream))) return rc;
    if ((rc = wi.alloc(sizeof(int32_t) * n, c.stream))) return rc;
    if ((rc = wperm.alloc(sizeof(int32_t) * n, c.stream))) return rc;
    if ((rc = wsort.alloc(sort_bytes, c.stream))) return rc;
    if ((rc = wrec.alloc(sizeof(float) * n * lay.rf * (packed ? 2 : 1), c.stream))) return rc;
    if ((rc = wg.alloc(sizeof(unsigned long long) * n, c.stream))) return rc;
    if ((rc = wf.alloc(sizeof(double) * a.nitems, c.stream))) return rc;
    if ((rc = wv.alloc(sizeof(float) * a.nitems, c.stream))) return rc;
    if ((rc = we.alloc(sizeof(double) * nblk, c.stream))) return rc;
    if ((rc = wc.alloc(sizeof(int), c.stream))) return rc;

    // ---- (1) sort by z, gather ----
    smooth_z_kernel<<<nblk, 256, 0, c.stream>>>(y, eps, N, wz.as<float>(), wi.as<int32_t>());
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    LIPFIT_CUDA(cub::DeviceRadixSort::SortPairs(wsort.p, sort_bytes, wz.as<float>(), wzs.as<float>(),
                                                wi.as<int32_t>(), wperm.as<int32_t>(), N, 0, 32,
                                                c.stream));
    smooth_gather_kernel<<<nblk, 256, 0, c.stream>>>(base, wperm.as<int32_t>(), wzs.as<float>(), N, lay.rf,
                                                     lay.vslot, wrec.as<float>(),
                                                     wg.as<unsigned long long>(), nullptr, packed ? 1 : 0,
                                                     wfix.as<double>());
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    LIPFIT_CUDA(cudaMemsetAsync(wc.p, 0, sizeof(int), c.stream));

    // ---- (2),(3) lower-triangle pairs ----
    a.rec = wrec.as<float>();
    a.gfix = wg.as<unsigned long long>();
    a.fix = wfix.as<double>();
    a.fpart = wf.as<double>();
    a.vpart = wv.as<float>();
    a.counter = wc.as<int>();
    FreeFlags ff = make_free_flags(xf);
    if (packed) {
        auto kern = smooth_pairs_packed_kernel<5>;
        int occ = 0;
        LIPFIT_CUDA(occupancy_of(&occ, kern, kSmThreads, 0));
        if (occ < 1) occ = 1;
        const int slots = c.num_sms * occ;
        KernelTimer kt(TK_SMOOTH_PAIRS, c.stream);
        kern<<<a.nitems < slots ? a.nitems : slots, kSmThreads, 0, c.stream>>>(a);
        kt.stop();
        ++g_launches;
        LIPFIT_CUDA(cudaGetLastError());
        rc = LIPFIT_OK;
    } else {
        rc = dispatch_pairs<kModeSmooth>(c, a, ff, xf, norm);
    }
    if (rc) return rc;

    smooth_grad_kernel<<<nblk, 256, 0, c.stream>>>(a.gfix, a.fix, wperm.as<int32_t>(), N, eps, p, grad,
                                                   we.as<double>());
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    if (F_dev || maxviol_dev) {
        smooth_final_kernel<<<1, 256, 0, c.stream>>>(a.fpart, a.vpart, a.nitems, we.as<double>(), nblk, p,
                                                     F_dev, maxviol_dev);
        ++g_launches;
        LIPFIT_CUDA(cudaGetLastError());
    }
    return LIPFIT_OK;
}

// NEXT-3: L = max_{i != k, y_i > y_k} (y_i - y_k) / d_s(x^k, x^i).
// base: packed records with the PLAIN (weighted / mirrored, not M-scaled) coordinates.  L_dev: device
// float, the maximum ratio (+inf if a pair with y_i > y_k has zero distance, 0 if no pair qualifies).
int launch_lipschitz_constant(const Ctx& c, const float* X, const float* base, const float* y, int64_t N64,
                              const Xform& xf, int norm, float* L_dev) {
    const int N = static_cast<int>(N64);
    const bool spec = lipconst_spec(xf);
    const RecLayout lay = lipconst_layout(xf, norm);
    const int R = spec ? (xf.d <= 5 ? 8 : 4) : smooth_rows(xf, norm);
    SmoothArgs a{};
    a.N = N;
    a.nrb = (N + kSmThreads * R - 1) / (kSmThreads * R);
    a.maxc = (N + kSmChunk - 1) / kSmChunk;
    a.nitems = a.nrb * a.maxc;
    const int nblk = (N + 255) / 256;
    const size_t n = static_cast<size_t>(N);
    size_t sort_bytes = 0;
    LIPFIT_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, sort_bytes, static_cast<const float*>(nullptr),
                                                static_cast<float*>(nullptr),
                                                static_cast<const int32_t*>(nullptr),
                                                static_cast<int32_t*>(nullptr), N, 0, 32, c.stream));
    Workspace wz, wzs, wi, wperm, wsort, wrec, wg, wf, wv, wc, wl;
    int rc;
    if ((rc = wz.alloc(sizeof(float) * n, c.stream))) return rc;
    if ((rc = wzs.alloc(sizeof(float) * n, c.stream))) return rc;
    if ((rc = wi.alloc(sizeof(int32_t) * n, c.stream))) return rc;
    if ((rc = wperm.alloc(sizeof(int32_t) * n, c.stream))) return rc;
    if ((rc = wsort.alloc(sort_bytes, c.stream))) return rc;
    if ((rc = wrec.alloc(sizeof(float) * n * lay.rf, c.stream))) return rc;
    if ((rc = wg.alloc(sizeof(unsigned long long) * n, c.stream))) return rc;
    if ((rc = wf.alloc(sizeof(double) * a.nitems, c.stream))) return rc;
    if ((rc = wv.alloc(sizeof(float) * a.nitems, c.stream))) return rc;
    if ((rc = wc.alloc(sizeof(int), c.stream))) return rc;
    if ((rc = wl.alloc(sizeof(unsigned long long) * 2, c.stream))) return rc;  // [0] max ratio, [1] amax
    LIPFIT_CUDA(cudaMemsetAsync(wl.p, 0, sizeof(unsigned long long) * 2, c.stream));
    smooth_z_kernel<<<nblk, 256, 0, c.stream>>>(y, nullptr, N, wz.as<float>(), wi.as<int32_t>());
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    LIPFIT_CUDA(cub::DeviceRadixSort::SortPairs(wsort.p, sort_bytes, wz.as<float>(), wzs.as<float>(),
                                                wi.as<int32_t>(), wperm.as<int32_t>(), N, 0, 32,
                                                c.stream));
    smooth_gather_kernel<<<nblk, 256, 0, c.stream>>>(base, wperm.as<int32_t>(), wzs.as<float>(), N, lay.rf,
                                                     lay.vslot, wrec.as<float>(),
                                                     wg.as<unsigned long long>(),
                                                     reinterpret_cast<uint32_t*>(wl.as<unsigned long long>() + 1), 0,
                                                     nullptr);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    LIPFIT_CUDA(cudaMemsetAsync(wc.p, 0, sizeof(int), c.stream));
    a.rec = wrec.as<float>();
    a.gfix = wg.as<unsigned long long>();
    a.fpart = wf.as<double>();
    a.vpart = wv.as<float>();
    a.counter = wc.as<int>();
    a.lmax = wl.as<unsigned long long>();
    a.amax = reinterpret_cast<const uint32_t*>(wl.as<unsigned long long>() + 1);
    a.X = X;
    a.perm = wperm.as<int32_t>();
    a.norm = norm;
    a.xf = xf;
    FreeFlags ff = make_free_flags(xf);
    if (spec)
        rc = norm == 1 ? dispatch_lipconst_spec<1>(c, a, ff, xf.d)
                       : (norm == 2 ? dispatch_lipconst_spec<2>(c, a, ff, xf.d) : dispatch_lipconst_spec<3>(c, a, ff, xf.d));
    else
        rc = dispatch_pairs<kModeLipConst>(c, a, ff, xf, norm);
    if (rc) return rc;
    lipconst_final_kernel<<<1, 1, 0, c.stream>>>(a.lmax, L_dev);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

}  // namespace lipfit
