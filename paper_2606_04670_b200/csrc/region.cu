// region.cu -- NEXT-4(iii): Eq.(2),(3) under MONOTONICITY ON PARTS OF THE DOMAIN (PAPER.md:147-167,
// section 4.2, cases I-IV; `mon in {0..4}`, `a`, `b` of PAPER.md:230).  The paper withholds the formula
// ("can be expressed through components of the distance vector"); reading R26 of DESIGN.md
// derives it.  Per coordinate i the line is cut into A: t <= a_i, AB: a_i <= t <= b_i, B: t >= b_i; f is
// monotone on A and on B in the direction the case prescribes and unrestricted on AB.  Walking from the
// datum's x^k_i to the query's x_i, f can only grow on the part of the way where it is not known to fall in
// the direction of travel.  With the two NON-DECREASING piecewise-linear transforms
//     psi_up(t) = mid(t) + [f increasing on A] A(t) + [f increasing on B] B(t)
//     psi_dn(t) = mid(t) + [f decreasing on A] A(t) + [f decreasing on B] B(t)
//     mid(t) = clamp(t, a, b) - a,   A(t) = min(t - a, 0),   B(t) = max(t - b, 0)      (t - a = mid + A + B)
// that length is   u_i = w_i max(psi_up(x_i) - psi_up(x^k_i), psi_dn(x^k_i) - psi_dn(x_i))   (upper bound)
// and              l_i = w_i max(psi_up(x^k_i) - psi_up(x_i), psi_dn(x_i) - psi_dn(x^k_i))   (lower bound):
// one of the two differences is the length sought, the other is <= 0.  Unrestricted coordinates have
// psi_up = psi_dn = t (|delta| on both sides), simple monotonicity (Eq.(4)) is a = b.
//
// So the prepack writes TWO transformed values (P, N) = w (psi_up, psi_dn) per coordinate, for data and
// queries alike, and the hot loop is mask-, case- and branch-free ("a suitable modification to
// distance calculation, which avoids branching"):
//     dP = P(q) - P(x),  dN = N(x) - N(q),  u = max(dP, dN),  l = -min(dP, dN).
// Kernel shape as bounds.cu: R queries per thread in registers, records through shared memory in TMA-filled
// double-buffered tiles, broadcast LDS.128, (query block, data chunk) tiles over a persistent grid.
#include <cmath>

#include "kernels.h"

namespace lipfit {

namespace {

// host-built description of the per-coordinate transforms (padding coordinates: w = 0)
struct RegionXform {
    int32_t perm[kMaxDim];              // packed coordinate j = original coordinate perm[j]: restricted ones first
    float w[kMaxDim];
    float alo[kMaxDim], bhi[kMaxDim];   // clamp bounds of mid (may be -inf / +inf)
    float a0[kMaxDim], b0[kMaxDim];     // finite reference points of A(t), B(t) and of mid
    float fa_up[kMaxDim], fb_up[kMaxDim], fa_dn[kMaxDim], fb_dn[kMaxDim];
    int32_t d;
};

__device__ __forceinline__ void region_transform(const RegionXform& rx, int j, float t, float& P, float& N) {
    const float mid = fminf(fmaxf(t, rx.alo[j]), rx.bhi[j]) - rx.a0[j];
    const float A = fminf(t - rx.a0[j], 0.f);
    const float B = fmaxf(t - rx.b0[j], 0.f);
    P = rx.w[j] * (mid + rx.fa_up[j] * A + rx.fb_up[j] * B);
    N = rx.w[j] * (mid + rx.fa_dn[j] * A + rx.fb_dn[j] * B);
}

// rows of [P_0, N_0, .., P_{DP-1}, N_{DP-1}] (+ [y, 0, 0, 0] when y != NULL): data records / packed queries
__global__ void __launch_bounds__(256)
region_pack_kernel(const float* __restrict__ X, const float* __restrict__ y, int n, RegionXform rx, int dp,
                   float* __restrict__ out) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int rf = 2 * dp + (y ? 4 : 0);
    const float* src = X + static_cast<size_t>(k) * rx.d;
    float4* dst = reinterpret_cast<float4*>(out + static_cast<size_t>(k) * rf);
    for (int j = 0; j < dp; j += 2) {
        float P0 = 0.f, N0 = 0.f, P1 = 0.f, N1 = 0.f;
        if (j < rx.d) region_transform(rx, j, src[rx.perm[j]], P0, N0);
        if (j + 1 < rx.d) region_transform(rx, j + 1, src[rx.perm[j + 1]], P1, N1);
        dst[j >> 1] = make_float4(P0, N0, P1, N1);
    }
    if (y) dst[dp >> 1] = make_float4(y[k], 0.f, 0.f, 0.f);
}

struct RegionArgs {
    const float* rec;   // [N][2 DP + 4]
    const float* qp;    // [Q][2 DP]
    float *upper, *lower, *g;
    uint32_t *keyU, *keyL;
    int N, Q, nqb, nch, chunk;
    int nr2;  // the first nr2 PAIRS of packed coordinates hold the restricted ones (mon != 0), the rest are free
    float M;
};

template <int DP>
__host__ __device__ constexpr int region_tile_records() {
    return DP <= 4 ? 256 : (DP <= 8 ? 128 : (DP <= 16 ? 64 : 32));
}

// Pairs of packed coordinates under a UNIFORM condition: restricted pairs take the two-transform arithmetic
// (6 operations per coordinate), pairs of unrestricted coordinates (P = N = w t, so dP = -dN = delta and
// u = l = |delta|) the plain 2 per coordinate.
// NR2: number of leading coordinate pairs that take the restricted arithmetic (compile time).
template <int NORM, int DP, int NR2>
__device__ __forceinline__ void region_pair(const float* q, const float* x, float M, int nr2_rt, float& hi,
                                            float& lo) {
    (void)nr2_rt;
    constexpr int nr2 = NR2;
    float su = 0.f, sl = 0.f;  // Linf: su = max u, sl = min over (dP, dN) (= -max l)
    float2 acc = make_float2(0.f, 0.f);  // L1: (sum u, sum m), m <= 0;  L2: (sum u^2, sum m^2)
    float sf = 0.f;            // unrestricted coordinates: shared by both bounds
#pragma unroll
    for (int c = 0; c < DP / 2; ++c) {
        if (c < nr2) {
#pragma unroll
            for (int j = 2 * c; j < 2 * c + 2; ++j) {
                // (dP, -dN) = (qP - xP, qN - xN): the two transformed values of a coordinate sit side by side in
                // the query and in the record, so both differences are ONE FADD2; the sign of the second rides
                // in the operand modifiers of the min / max, and (u, m) accumulate with one FADD2 / FFMA2
                const float2 d2 = __fadd2_rn(make_float2(q[2 * j], q[2 * j + 1]), make_float2(-x[2 * j], -x[2 * j + 1]));
                const float dP = d2.x, dN = -d2.y;
                if (NORM == 3) {
                    su = fmaxf(fmaxf(su, dP), dN);  // FMNMX3
                    sl = fminf(fminf(sl, dP), dN);
                } else {
                    const float2 um = make_float2(fmaxf(dP, dN), fminf(dP, dN));  // u >= 0 >= m
                    acc = NORM == 1 ? __fadd2_rn(acc, um) : __ffma2_rn(um, um, acc);
                }
            }
        } else {
#pragma unroll
            for (int j = 2 * c; j < 2 * c + 2; ++j) {
                const float dlt = q[2 * j] - x[2 * j];
                if (NORM == 1) sf += fabsf(dlt);
                if (NORM == 2) sf = fmaf(dlt, dlt, sf);
                if (NORM == 3) sf = fmaxf(sf, fabsf(dlt));
            }
        }
    }
    if (NORM == 1) {
        su = acc.x;
        sl = -acc.y;
    } else if (NORM == 2) {
        su = acc.x;
        sl = acc.y;
    }
    const float y = x[2 * DP];
    if (NORM == 2) {
        hi = fmaf(M, fast_sqrt(su + sf), y);
        lo = fmaf(-M, fast_sqrt(sl + sf), y);
    } else if (NORM == 1) {
        hi = fmaf(M, su + sf, y);
        lo = fmaf(-M, sl + sf, y);
    } else {
        hi = fmaf(M, fmaxf(su, sf), y);
        lo = fmaf(-M, fmaxf(-sl, sf), y);
    }
}

template <int NORM, int DP, int R, int NR2>
__global__ void __launch_bounds__(128, 2)
bounds_region_kernel(const RegionArgs a) {
    constexpr int THREADS = 128;
    constexpr int RF = 2 * DP + 4;
    constexpr int TILE = region_tile_records<DP>();
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
        float q[R][2 * DP], U[R], L[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            int qi = (qb * R + r) * THREADS + static_cast<int>(threadIdx.x);
            qi = qi < a.Q ? qi : a.Q - 1;
            const float4* src = reinterpret_cast<const float4*>(a.qp + static_cast<size_t>(qi) * 2 * DP);
#pragma unroll
            for (int c = 0; c < DP / 2; ++c) {
                const float4 v = __ldg(src + c);
                q[r][4 * c] = v.x;
                q[r][4 * c + 1] = v.y;
                q[r][4 * c + 2] = v.z;
                q[r][4 * c + 3] = v.w;
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
            for (int j = 0; j < n; ++j) {
                float x[RF];
#pragma unroll
                for (int c = 0; c < RF / 4; ++c) {
                    const float4 v = reinterpret_cast<const float4*>(s + j * RF)[c];
                    x[4 * c] = v.x;
                    x[4 * c + 1] = v.y;
                    x[4 * c + 2] = v.z;
                    x[4 * c + 3] = v.w;
                }
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    float hi, lo;
                    region_pair<NORM, DP, NR2>(q[r], x, a.M, a.nr2, hi, lo);
                    U[r] = fminf(U[r], hi);
                    L[r] = fmaxf(L[r], lo);
                }
            }
            rs.release(t);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int qi = (qb * R + r) * THREADS + static_cast<int>(threadIdx.x);
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

template <int NORM, int DP, int R, int NR2>
int launch_region_t(const Ctx& c, RegionArgs& a) {
    constexpr int THREADS = 128;
    auto kern = bounds_region_kernel<NORM, DP, R, NR2>;
    int occ = 0;
    LIPFIT_CUDA(occupancy_of(&occ, kern, THREADS, 0));
    if (occ < 1) occ = 1;
    const int slots = c.num_sms * occ;
    constexpr int TILE = region_tile_records<DP>();
    a.nqb = (a.Q + THREADS * R - 1) / (THREADS * R);
    // as bounds.cu: cut the data into chunks until there are >= 16 tiles per resident CTA, chunks >= 4 smem tiles
    int want = (16 * slots + a.nqb - 1) / a.nqb;
    const int max_ch = (a.N + 4 * TILE - 1) / (4 * TILE);
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
    KernelTimer kt(TK_BOUNDS_REGION, c.stream);
    kern<<<static_cast<int>(ntiles < slots ? ntiles : slots), THREADS, 0, c.stream>>>(a);
    kt.stop();
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    if (nch > 1) return launch_bounds_finalize(c, a.keyU, a.keyL, a.Q, a.upper, a.lower, a.g);
    return LIPFIT_OK;
}

template <int NORM, int DP, int R, int NR2>
int launch_region_r(const Ctx& c, RegionArgs& a) {
    if (a.nr2 == NR2) return launch_region_t<NORM, DP, R, NR2>(c, a);
    if constexpr (NR2 > 0) return launch_region_r<NORM, DP, R, NR2 - 1>(c, a);
    return LIPFIT_E_PARAM;
}

template <int NORM>
int launch_region_n(const Ctx& c, RegionArgs& a, int dp, bool small) {
    // throughput flavour: R queries per thread; small Q: one query per thread so that the chip fills.
    // DP <= 8: one kernel per number of restricted coordinate pairs (0 .. DP / 2); DP >= 16: every pair takes the
    // restricted arithmetic (valid for any coordinate; a runtime-uniform count was measured and is SLOWER: ptxas
    // predicates both bodies).
    switch (dp) {
        case 4: return small ? launch_region_r<NORM, 4, 1, 2>(c, a) : launch_region_r<NORM, 4, 4, 2>(c, a);
        case 8: return small ? launch_region_r<NORM, 8, 1, 4>(c, a) : launch_region_r<NORM, 8, 4, 4>(c, a);
        case 16: return small ? launch_region_t<NORM, 16, 1, 8>(c, a) : launch_region_t<NORM, 16, 2, 8>(c, a);
        default: return launch_region_t<NORM, 32, 1, 16>(c, a);
    }
}

}  // namespace

int launch_bounds_region(const Ctx& c, const float* X, const float* y, int64_t N, int32_t d, const float* Xq,
                         int64_t Q, float M, const int32_t* mon, const float* a_host, const float* b_host,
                         int norm, const float* weights, float* upper, float* lower, float* g) {
    RegionXform rx{};
    rx.d = d;
    int order[kMaxDim], nres = 0, nord = 0;
    for (int i = 0; i < d; ++i)
        if (mon && mon[i] != 0) order[nord++] = i;  // restricted coordinates first
    nres = nord;
    for (int i = 0; i < d; ++i)
        if (!(mon && mon[i] != 0)) order[nord++] = i;
    // (an odd number of restricted coordinates: the pair that holds the last one also holds the first free
    // coordinate or padding; it takes the restricted arithmetic, which is valid for any coordinate)
    for (int j = 0; j < kMaxDim; ++j) {
        const int i = j < d ? order[j] : 0;
        rx.perm[j] = i;
        const int m = (j < d && mon) ? mon[i] : 0;
        const float w = j < d ? (weights ? weights[i] : 1.f) : 0.f;
        rx.w[j] = w;
        float a = -INFINITY, b = INFINITY;
        if (m != 0) {
            a = a_host[i];
            b = b_host[i];
        }
        const bool incA = (m == 1 || m == 4), incB = (m == 1 || m == 3);
        const bool hasA = m != 0 && std::isfinite(a), hasB = m != 0 && std::isfinite(b);
        rx.alo[j] = a;
        rx.bhi[j] = b;
        // finite reference points: A(t) = min(t - a0, 0) and B(t) = max(t - b0, 0) only count when the region
        // exists; mid is measured from a0 so that every term scales with the distance to the thresholds
        rx.a0[j] = hasA ? a : (hasB ? b : 0.f);
        rx.b0[j] = hasB ? b : rx.a0[j];
        rx.fa_up[j] = (hasA && incA) ? 1.f : 0.f;
        rx.fa_dn[j] = (hasA && !incA) ? 1.f : 0.f;
        rx.fb_up[j] = (hasB && incB) ? 1.f : 0.f;
        rx.fb_dn[j] = (hasB && !incB) ? 1.f : 0.f;
    }
    const int dp = d <= 4 ? 4 : (d <= 8 ? 8 : (d <= 16 ? 16 : 32));
    const int n = static_cast<int>(N), q = static_cast<int>(Q);
    Workspace wrec, wq;
    int rc;
    if ((rc = wrec.alloc(sizeof(float) * static_cast<size_t>(N) * (2 * dp + 4), c.stream))) return rc;
    if ((rc = wq.alloc(sizeof(float) * static_cast<size_t>(Q) * 2 * dp, c.stream))) return rc;
    region_pack_kernel<<<(n + 255) / 256, 256, 0, c.stream>>>(X, y, n, rx, dp, wrec.as<float>());
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    region_pack_kernel<<<(q + 255) / 256, 256, 0, c.stream>>>(Xq, nullptr, q, rx, dp, wq.as<float>());
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    RegionArgs a{};
    a.rec = wrec.as<float>();
    a.qp = wq.as<float>();
    a.upper = upper;
    a.lower = lower;
    a.g = g;
    a.N = n;
    a.Q = q;
    a.M = M;
    a.nr2 = (nres + 1) / 2;
    const bool small = (Q + 3) / 4 < 2LL * c.num_sms * 128;
    if (norm == 1) return launch_region_n<1>(c, a, dp, small);
    if (norm == 2) return launch_region_n<2>(c, a, dp, small);
    return launch_region_n<3>(c, a, dp, small);
}

}  // namespace lipfit
