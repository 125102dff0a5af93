// kernels.h -- host-side launchers implemented in the .cu translation units.
#pragma once
#include "common.cuh"
#include "dist.cuh"

namespace lipfit {

// Builds the Xform for (mask, weights); flip = true negates the mask first (used by kNN side=-1,
// where D^l under mask s equals D^u under mask -s).  symmetric = true ignores the mask (R6).
int make_xform(int32_t d, const int32_t* mono_mask, const float* weights, bool symmetric, bool flip,
               Xform* xf);
FreeFlags make_free_flags(const Xform& xf);

// Record layout chosen by the kernel family that will consume the records: `rf` floats per
// record (multiple of 4), packed coordinates in slots [0, d), the value (y or z) in slot `vslot`,
// zeros elsewhere.
struct RecLayout {
    int rf, vslot;
    int cslot = -1;       // >= 0: slot of c' = 2 value - sum of the constrained coordinates (folded L1 bounds)
    bool mscale = false;  // true: the kernel family wants the coordinates pre-multiplied by M
    bool dup = false;     // true: every float is stored twice (x0,x0,x1,x1,..): operands of packed f32x2 math;
                          //       rf then counts the PHYSICAL floats, vslot / cslot stay logical
    bool packed = false;  // the variant has a packed-f32x2 throughput kernel (bounds_layout sets dup when it is used)
};
RecLayout bounds_layout(const Ctx& c, const Xform& xf, int norm, int64_t Q);
// the transform the all-pairs bounds pass really uses for (xf, norm): xf itself, or xf with zero-weight padding
// coordinates for off-table shapes with d <= 8 (bounds.cu); apply it before bounds_layout / prepack / launch_bounds
Xform bounds_xform(const Xform& xf, int norm);
RecLayout smooth_layout(const Xform& xf, int norm);
RecLayout lipconst_layout(const Xform& xf, int norm);  // records of launch_lipschitz_constant

// a1: build the records; y may be NULL (value 0), eps may be NULL; value = y[k] + eps[k].
// centre: device float[d] in the ORIGINAL coordinate order or NULL.  When given, the packed coordinates are
// sw_j (x - centre): the kernel families that pre-multiply the coordinates by M (layouts with mscale, the
// smoothing records) round M w x before subtracting, an absolute error ~2^-24 M |x| per coordinate -- after
// the translation it scales with the spread of the data instead of their offset from the origin.  The
// callers pass the first datum X[0 .. d) (any point near the data does; distances are translation
// invariant).  The consumer must translate its queries by the same centre.
int launch_prepack(const Ctx& c, const float* X, const float* y, const float* eps, int64_t N,
                   const Xform& xf, RecLayout lay, float* rec, const float* centre = nullptr);

// a2: fused bounds.  rec: packed records; Xq: ORIGINAL row-major queries (transformed on load).
int launch_bounds(const Ctx& c, const float* rec, int64_t N, const float* Xq, int64_t Q,
                  const Xform& xf, int norm, float M, float* upper, float* lower, float* g,
                  const float* centre = nullptr);
const char* bounds_variant_name(const Xform& xf, int norm);
// partial extrema of data chunks (order-preserving keys, atomicMin / atomicMax) -> upper / lower / g
int launch_bounds_finalize(const Ctx& c, const uint32_t* keyU, const uint32_t* keyL, int Q, float* upper,
                           float* lower, float* g);
// NEXT-4(iii): bounds under monotonicity on parts of the domain (region.cu, reading R26).
// mon / a_host / b_host / weights: HOST arrays of length d, already validated by the caller.
int launch_bounds_region(const Ctx& c, const float* X, const float* y, int64_t N, int32_t d, const float* Xq,
                         int64_t Q, float M, const int32_t* mon, const float* a_host, const float* b_host,
                         int norm, const float* weights, float* upper, float* lower, float* g);
// NEXT-2: weighted sums of the k best upper / lower bound values; wk_host: host float[k]
// rec: records in bounds_topk_layout (= bounds_layout; mscale / centre / dup as for lipfit_bounds)
RecLayout bounds_topk_layout(const Ctx& c, const Xform& xf, int norm, int64_t Q);
int launch_bounds_topk(const Ctx& c, const float* rec, int64_t N, const float* Xq, int64_t Q, const Xform& xf,
                       int norm, float M, int k, const float* wk_host, float* upper, float* lower, float* g,
                       const float* centre, bool dup);

// NEXT-4(ii): bounds with exact spatial pruning (prune.cu); X, Xq: ORIGINAL row-major arrays.
// stats_dev: device uint64[3] (zeroed by the caller) or NULL: [0] += tiles of 32 x 32 pairs evaluated,
// [1] += tiles that passed the warp-box test, [2] += lanes whose own test asked for an evaluated tile.
// guard_limit > 0 (LIPFIT_BOUNDS_AUTO): the kernel keeps the running fraction of pairs its finished query groups
// evaluated; above guard_limit (from max(64, groups / 64) finished groups on, while fewer than half are done) the
// groups not yet started return at once.  One read-back + stream synchronisation after the kernel sets *declined:
// the outputs are then incomplete and the caller runs the all-pairs kernels instead.
int launch_bounds_pruned(const Ctx& c, const float* X, const float* y, int64_t N, const float* Xq, int64_t Q,
                         const Xform& xf, int norm, float M, float* upper, float* lower, float* g,
                         unsigned long long* stats_dev, float guard_limit = 0.f, bool* declined = nullptr);

// LIPFIT_BOUNDS_AUTO (include/lipfit.h): the exactly pruned pass when the box tests can pay for themselves --
// few enough coordinates for the boxes to separate (d <= 8: measured 9.7x / 5.3x / 2.0x on the config 2 / 5 /
// 3 workloads, d = 4 / 5 / 8) and enough pairs (>= 2^32, N >= 8192, Q >= 4096) to amortise two radix sorts.
inline bool bounds_prefers_pruned(const Xform& xf, int64_t N, int64_t Q) {
    return xf.d <= 8 && N >= 8192 && Q >= 4096 && N * Q >= (1LL << 32);
}
// ... and only while the finished query groups evaluate at most this fraction of their pairs: the pruned kernel evaluates
// a pair at 0.35-0.55 of the all-pairs kernels' rate (configs 2 / 5 / 3: 1.23 vs 3.1, 0.68 vs 1.19, 1.05 vs 1.84
// Tpairs/s), so beyond ~40 % the all-pairs pass is the faster exact answer.
constexpr float kPrunedGuardLimit = 0.40f;

// Eq.(7) objective / gradient with the same exact pruning (prune.cu).  F_dev: device double (required,
// zeroed here); grad: device float in the original order or NULL; eps may be NULL.
// order_dev: the Morton order of the data from smooth_pruned_order (depends on X only; NULL: computed here).
int launch_smooth_objective_pruned(const Ctx& c, const float* X, const float* y, const float* eps, int64_t N,
                                   const Xform& xf, int norm, float M, float p, double* F_dev, float* grad,
                                   unsigned long long* stats_dev, double* maxviol_dev = nullptr,
                                   const int32_t* order_dev = nullptr);
int smooth_pruned_order(const Ctx& c, const float* X, int64_t N, const Xform& xf, Workspace& dorder);
// lipfit_smooth evaluates Eq.(7) with the pruned pass when it wins: no constrained coordinate (the
// dominated orthant of a monotone mask defeats the box test) and enough data to fill the chip
inline bool smooth_prefers_pruned(const Xform& xf, int64_t N) { return xf.dC == 0 && N >= 8192; }

// a3: fused distance + top-k selection (fp32) followed by the fp64 re-rank.  allow_tc = false keeps the
// selection on the CUDA cores; info (host, may be NULL): per-call diagnostics, the call then synchronises.
int launch_knn(const Ctx& c, const float* X, int64_t N, const float* Xq, int64_t Q, const Xform& xf,
               int norm, int k, int32_t* idx, float* dist, bool allow_tc, lipfit_knn_info* info);
const char* knn_variant_name(const Xform& xf, int norm, bool allow_tc);

// a4: all-pairs objective/gradient.  base: packed records whose coordinates are PRE-MULTIPLIED BY M
// (prepack with scale_xform(xf, M)); their value slot is ignored, z = y + eps is formed per call.
// F_dev: device double (may be NULL); grad: device float (may be NULL); eps may be NULL (= 0).
int launch_smooth_objective(const Ctx& c, const float* base, const float* y, const float* eps, int64_t N,
                            const Xform& xf, int norm, float p, double* F_dev, float* grad,
                            double* maxviol_dev);
// NEXT-3: smallest consistent Lipschitz constant; base = packed records with plain coordinates.
int launch_lipschitz_constant(const Ctx& c, const float* X, const float* base, const float* y, int64_t N,
                              const Xform& xf, int norm, float* L_dev);
// NEXT-1: local Lipschitz interpolation (local.cu).  knots_host: host float[LIPFIT_LOCAL_KNOTS].
int launch_distance_quantiles(const Ctx& c, const float* X, int64_t N, const Xform& xf, int norm,
                              const int32_t* pair_i, const int32_t* pair_k, int64_t S, int J, float* knots_dev,
                              int* bad_dev);
int launch_local_lipschitz(const Ctx& c, const float* X, const float* y, int64_t N, const Xform& xf, int norm,
                           const float* knots_host, float* table);
int launch_values_local(const Ctx& c, const float* X, const float* y, int64_t N, const float* Xq, int64_t Q,
                        const Xform& xf, int norm, const float* knots_host, const float* table, float* upper,
                        float* lower, float* g);
// xf with every coordinate factor multiplied by s
Xform scale_xform(const Xform& xf, float s);

// value-slot refresh: rec[k][vslot] = y[k] + eps[k]
int launch_set_values(const Ctx& c, float* rec, RecLayout lay, const float* y, const float* eps,
                      int64_t N);
// y[k] += eps[k]
int launch_axpy(const Ctx& c, float* y, const float* eps, int64_t N);

// cudaMemPoolTrimTo(private pool of the current device, 0)
int workspace_release();

// small.cu: step a2 for latency-bound calls (all N data fit a CTA's shared memory, <= 2^25 pairs): one kernel
// launch, a1 inside the kernel, no workspace.  X, Xq: ORIGINAL row-major arrays.
bool bounds_small_applies(const Xform& xf, int64_t N, int64_t Q);
int launch_bounds_small(const Ctx& c, const float* X, const float* y, int64_t N, const float* Xq, int64_t Q,
                        const Xform& xf, int norm, float M, float* upper, float* lower, float* g);

// noalloc.cu: all-pairs bounds whose scratch is a fixed file-scope device array (no allocation of any kind);
// LIPFIT_E_LIMIT when N (DP + 4) or Q exceed it.  X, Xq: ORIGINAL row-major arrays.
int launch_bounds_noalloc(const Ctx& c, const float* X, const float* y, int64_t N, const float* Xq, int64_t Q,
                          const Xform& xf, int norm, float M, float* upper, float* lower, float* g);

// diagnostic (pipes.cu): measured issue rate of one fp32 instruction class on the current device
int pipe_throughput(const Ctx& c, int which, double* lane_results_per_clk_sm, double* warp_instr_per_clk_sm);

void timing_set(int on);
int timing_get(int which, double* ms, long long* n);

}  // namespace lipfit
