// dist.cuh -- per-pair arithmetic of the monotone weighted distance, in registers.
//
// Packed coordinates (common.cuh, Xform): j < DU unconstrained, DU <= j < DU+DC constrained and
// already mirrored/weighted, so with delta_j = q_j - x_j   (query minus datum)
//   u_j = l_j = |delta_j|                       (unconstrained)
//   u_j = max(delta_j, 0),  l_j = max(-delta_j, 0)   (constrained)       Eq.(4)
//   D^u = ||u||_p,  D^l = ||l||_p.
// NORM: 1 = L1, 2 = L2, 3 = Linf.
#pragma once
#include "common.cuh"

namespace lipfit {

// delta_j = q_j - x_j for D coordinates.  Neighbouring coordinates of the query (registers of the thread) and of
// the record (one LDS.128) are register pairs already, so two differences are ONE packed FADD2 (add.rn.f32x2,
// same rounding as the scalar subtraction: bit-identical results): the unpacked kernels are issue-bound, and
// this halves the issue slots of their subtractions without any change of layout.
#ifndef LIPFIT_PACK_DELTAS
#define LIPFIT_PACK_DELTAS 1
#endif
template <int D>
__device__ __forceinline__ void pair_deltas(const float* __restrict__ q, const float* __restrict__ x, float* dl) {
#if LIPFIT_PACK_DELTAS
#pragma unroll
    for (int j = 0; j + 1 < D; j += 2) {
        const float2 t = __fadd2_rn(make_float2(q[j], q[j + 1]), make_float2(-x[j], -x[j + 1]));
        dl[j] = t.x;
        dl[j + 1] = t.y;
    }
    if (D & 1) dl[D - 1] = q[D - 1] - x[D - 1];
#else
#pragma unroll
    for (int j = 0; j < D; ++j) dl[j] = q[j] - x[j];
#endif
}

// Accumulated "pre-norm" quantities: L1 -> sums, L2 -> sums of squares, Linf -> maxima.
// S is the part shared by both sides (unconstrained coordinates); PU / PL the one-sided parts.
template <int NORM, int DU, int DC>
struct PairAcc {
    // q, x: D = DU + DC packed coordinates in registers.
    static __device__ __forceinline__ void run(const float* __restrict__ q,
                                               const float* __restrict__ x, float& au, float& al) {
        float dl[DU + DC > 0 ? DU + DC : 1];
        pair_deltas<DU + DC>(q, x, dl);
        float s = 0.f;
#pragma unroll
        for (int j = 0; j < DU; ++j) {
            float dlt = dl[j];
            if (NORM == 1) s += fabsf(dlt);
            if (NORM == 2) s = fmaf(dlt, dlt, s);
            // the chain of maxima starts from |delta_0|, not from 0: n values then fold into (n - 1) / 2 FMNMX3
            if (NORM == 3) s = (j == 0) ? fabsf(dlt) : fmaxf(s, fabsf(dlt));
        }
        float pu = s, pl = s;
#pragma unroll
        for (int j = DU; j < DU + DC; ++j) {
            float dlt = dl[j];
            if (NORM == 1) {
                float r = fmaxf(dlt, 0.f);
                pu += r;
                pl += r - dlt;  // max(-dlt,0) == max(dlt,0) - dlt exactly (one of the two is 0)
            }
            if (NORM == 2) {
                float r = fmaxf(dlt, 0.f);
                float m = fminf(dlt, 0.f);
                pu = fmaf(r, r, pu);
                pl = fmaf(m, m, pl);
            }
            if (NORM == 3) {
                pu = fmaxf(pu, dlt);  // pu >= 0 already, so max(pu, relu(dlt)) == max(pu, dlt)
                pl = fmaxf(pl, -dlt);
            }
        }
        au = pu;
        al = pl;
    }
    // distance from the accumulated quantity
    static __device__ __forceinline__ float finish(float a) { return NORM == 2 ? fast_sqrt(a) : a; }
};

// One-sided distance only (kNN): D^u accumulated quantity (squared for L2).
template <int NORM, int DU, int DC>
struct PairAccU {
    static __device__ __forceinline__ float run(const float* __restrict__ q,
                                                const float* __restrict__ x) {
        float dl[DU + DC > 0 ? DU + DC : 1];
        pair_deltas<DU + DC>(q, x, dl);
        float s = 0.f;
#pragma unroll
        for (int j = 0; j < DU; ++j) {
            float dlt = dl[j];
            if (NORM == 1) s += fabsf(dlt);
            if (NORM == 2) s = fmaf(dlt, dlt, s);
            if (NORM == 3) s = (j == 0) ? fabsf(dlt) : fmaxf(s, fabsf(dlt));
        }
#pragma unroll
        for (int j = DU; j < DU + DC; ++j) {
            float dlt = dl[j];
            if (NORM == 1) s += fmaxf(dlt, 0.f);
            if (NORM == 2) {
                float r = fmaxf(dlt, 0.f);
                s = fmaf(r, r, s);
            }
            if (NORM == 3) s = fmaxf(s, dlt);
        }
        return s;
    }
};

// Generic (runtime mask) version over DP zero-padded coordinates: `fr[j]` is 1 for an
// unconstrained coordinate and 0 for a constrained (or padding) one, so that
//   u_j = max(delta, -fr*delta)  -> |delta| or relu(delta)
//   l_j = max(-delta, fr*delta)  -> |delta| or relu(-delta)
// without a branch.  Padding coordinates have x = q = 0, hence contribute 0 to every norm.
struct FreeFlags {
    float fr[kMaxDim];
    // chunks of 4 packed coordinates (make_free_flags): the first nfree4 chunks hold unconstrained coordinates
    // only, chunks [nfree4, nall4) hold the rest of the d coordinates, chunks >= nall4 are pure padding
    int32_t nfree4, nall4;
};

template <int NORM, int DP>
struct PairAccGeneric {
    static __device__ __forceinline__ void run(const float* __restrict__ q,
                                               const float* __restrict__ x, const FreeFlags& ff,
                                               float& au, float& al) {
        float dl[DP];
        pair_deltas<DP>(q, x, dl);
        float pu = 0.f, pl = 0.f;
#pragma unroll
        for (int j = 0; j < DP; ++j) {
            float dlt = dl[j];
            float t = ff.fr[j] * dlt;
            float u = fmaxf(dlt, -t);
            float l = fmaxf(-dlt, t);
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
        au = pu;
        al = pl;
    }
    static __device__ __forceinline__ float run_u(const float* __restrict__ q,
                                                  const float* __restrict__ x,
                                                  const FreeFlags& ff) {
        float dl[DP];
        pair_deltas<DP>(q, x, dl);
        float pu = 0.f;
#pragma unroll
        for (int j = 0; j < DP; ++j) {
            float dlt = dl[j];
            float u = fmaxf(dlt, -(ff.fr[j] * dlt));
            if (NORM == 1) pu += u;
            if (NORM == 2) pu = fmaf(u, u, pu);
            if (NORM == 3) pu = fmaxf(pu, u);
        }
        return pu;
    }
    static __device__ __forceinline__ float finish(float a) { return NORM == 2 ? fast_sqrt(a) : a; }
};

// Chunked form of the generic arithmetic for the bounds kernels of d > 8 (bounds.cu GenCore): the DP padded
// coordinates are visited in chunks of 4 under UNIFORM (kernel-parameter) conditions -- chunks of unconstrained
// coordinates take the plain 2 operations per coordinate, the (at most dC/4 + 2) remaining chunks the flag
// arithmetic (6 per coordinate), padding chunks are skipped.  Same values as PairAccGeneric::run (adding the
// zeros of a padding coordinate changes no sum, square sum or maximum).
template <int NORM, int DP>
struct PairAccChunked {
    static __device__ __forceinline__ void run(const float* __restrict__ q, const float* __restrict__ x,
                                               const FreeFlags& ff, float& au, float& al) {
        float s = 0.f, pu = 0.f, pl = 0.f;
#pragma unroll
        for (int c = 0; c < DP / 4; ++c) {
            float dl[4];
            if (c < ff.nall4) pair_deltas<4>(q + 4 * c, x + 4 * c, dl);
            if (c < ff.nfree4) {
#pragma unroll
                for (int j = 4 * c; j < 4 * c + 4; ++j) {
                    const float dlt = dl[j - 4 * c];
                    if (NORM == 1) s += fabsf(dlt);
                    if (NORM == 2) s = fmaf(dlt, dlt, s);
                    if (NORM == 3) s = fmaxf(s, fabsf(dlt));
                }
            } else if (c < ff.nall4) {
#pragma unroll
                for (int j = 4 * c; j < 4 * c + 4; ++j) {
                    const float dlt = dl[j - 4 * c];
                    const float t = ff.fr[j] * dlt;
                    const float u = fmaxf(dlt, -t);
                    const float l = fmaxf(-dlt, t);
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
            }
        }
        if (NORM == 3) {
            au = fmaxf(s, pu);
            al = fmaxf(s, pl);
        } else {
            au = s + pu;
            al = s + pl;
        }
    }
};

// Uniform policy wrappers (used by the smoothing kernel): D coordinates per point, RF floats per
// record, value slot VSLOT, run() -> accumulated (au, al), finish() -> distance.
template <int NORM_, int DU, int DC>
struct SpecAcc {
    static constexpr int D = DU + DC;
    static constexpr int RF = record_floats(D);
    static constexpr int VSLOT = D;
    static constexpr int NORM = NORM_;
    static constexpr bool kGeneric = false;
    static __device__ __forceinline__ void run(const float* q, const float* x, const FreeFlags&,
                                               float& au, float& al) {
        PairAcc<NORM, DU, DC>::run(q, x, au, al);
    }
    // one-sided accumulated quantity of D^u only
    static __device__ __forceinline__ float run_u(const float* q, const float* x, const FreeFlags&) {
        return PairAccU<NORM, DU, DC>::run(q, x);
    }
    static __device__ __forceinline__ float finish(float a) { return NORM == 2 ? fast_sqrt(a) : a; }
};

template <int NORM_, int DP>
struct GenAcc {
    static constexpr int D = DP;
    static constexpr int RF = DP + 4;
    static constexpr int VSLOT = DP;
    static constexpr int NORM = NORM_;
    static constexpr bool kGeneric = true;
    static __device__ __forceinline__ void run(const float* q, const float* x, const FreeFlags& ff,
                                               float& au, float& al) {
        PairAccGeneric<NORM, DP>::run(q, x, ff, au, al);
    }
    static __device__ __forceinline__ float run_u(const float* q, const float* x, const FreeFlags& ff) {
        return PairAccGeneric<NORM, DP>::run_u(q, x, ff);
    }
    static __device__ __forceinline__ float finish(float a) { return NORM == 2 ? fast_sqrt(a) : a; }
};

}  // namespace lipfit
