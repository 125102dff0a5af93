/*
 * lipfit.h -- C ABI of the B200-native (sm_100a) LipFit hot path.
 *
 * Implements the data-parallel hot path of "Fitting scattered data with
 * optional monotonicity constraints on GPU: LipFit package" (PAPER.md =
 * arxiv/paper_2606_04670): evaluation of the optimal Lipschitz interpolant
 * (Eq.(2),(3) with the monotone distance Eq.(4)), neighbour selection by the
 * same fused distance-then-reduce pass, and penalty smoothing (Eq.(5)-(7)).
 *
 * Conventions common to every entry point
 *   - Plain C types only.  Unless a parameter says "host", array pointers are
 *     DEVICE pointers to row-major fp32 (int32 for indices), 4-byte aligned,
 *     caller-owned.  The library never frees or retains caller memory.
 *     `mono_mask` and `weights` are HOST arrays of length d (read during the
 *     call; NULL = all 0 / all 1).  The `*_host` variants take HOST pointers for
 *     everything and do the host<->device copies themselves.
 *   - `cuda_stream` is a cudaStream_t (NULL = default stream).  Internal workspace comes from a
 *     PRIVATE stream-ordered memory pool of the library (cudaMemPoolCreate, one per device, created on
 *     first use), is allocated on that stream and released (stream-ordered) before the call returns.
 *     The pool keeps released workspaces cached across synchronisations (so that back-to-back calls do
 *     not re-map them); lipfit_release_workspace() hands them back to the driver.  The device's default
 *     memory pool and the caller's allocator are never touched.
 *   - Every function returns LIPFIT_OK (0) or a negative lipfit_status; no exception crosses the
 *     boundary.
 *   - Thread safety.  The compute entry points keep no per-call state outside their arguments, so
 *     calls from different host threads on different streams may run concurrently.  Process-wide
 *     state is exactly: (1) the private memory pools and the caches of device attributes / occupancy
 *     (mutex-protected, invisible to results); (2) the monotone launch counter lipfit_launch_count
 *     (atomic); (3) the DIAGNOSTIC timing switch lipfit_set_timing / lipfit_get_timing: process-wide
 *     accumulators under a mutex, every thread's launches add to them while the switch is on, and a
 *     timed launch blocks its calling thread -- meant for single-threaded measurement (bench.py), not
 *     for production use.  Nothing else is global: kernel-selection options and per-call diagnostics
 *     of kNN are arguments of lipfit_knn_ex, not settings.
 *   - lipfit_bounds / lipfit_knn / lipfit_smooth_objective(F==NULL) are
 *     asynchronous on `cuda_stream`; lipfit_smooth and the *_host variants
 *     synchronise the stream before returning.
 *   - Inputs must be finite; NaN/Inf are not scanned for (results undefined,
 *     never a crash).  There is no CPU fallback: without a CUDA device every
 *     compute call returns LIPFIT_E_CUDA.
 *
 * Distance (Eq.(4), sign convention PAPER.md:140):
 *   delta_i = xq_i - x^k_i, mask s_i in {-1,0,+1}, weight w_i >= 0,
 *   u_i = w_i |delta_i| if s_i = 0 else w_i max( s_i delta_i, 0)
 *   l_i = w_i |delta_i| if s_i = 0 else w_i max(-s_i delta_i, 0)
 *   D^u = ||u||_p = d_s(x^k, x)   (used by H^upper)
 *   D^l = ||l||_p = d_s(x, x^k)   (used by H^lower),  p = norm in {1,2,inf}.
 */
#ifndef LIPFIT_H
#define LIPFIT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LIPFIT_MAX_DIM 32
#define LIPFIT_MAX_K 128
#define LIPFIT_MAX_TOPK 8    /* neighbours of the k > 1 approximation (lipfit_bounds_topk) */
#define LIPFIT_LOCAL_KNOTS 16 /* knots of the local Lipschitz step functions M_k */

enum lipfit_norm { LIPFIT_L1 = 1, LIPFIT_L2 = 2, LIPFIT_LINF = 3 };

enum lipfit_status {
    LIPFIT_OK = 0,
    LIPFIT_E_NULL = -1,  /* a required pointer is NULL */
    LIPFIT_E_DIM = -2,   /* d < 1 or d > LIPFIT_MAX_DIM */
    LIPFIT_E_SIZE = -3,  /* N < 1, Q < 0, k < 1, k > N, k > LIPFIT_MAX_K, N or Q > 2^31-1 */
    LIPFIT_E_PARAM = -4, /* M < 0 or non-finite, mask not in {-1,0,1}, w < 0 or non-finite, bad norm/side, p <= 0 */
    LIPFIT_E_CUDA = -5,  /* a CUDA runtime call failed (no device, launch error, ...) */
    LIPFIT_E_NOMEM = -6, /* workspace allocation failed */
    LIPFIT_E_LIMIT = -7  /* sizes beyond the fixed scratch of a no-allocation entry point (lipfit_bounds_noalloc) */
};

/* ---- Eq.(2),(3) PAPER.md:103-116 with the distance of Eq.(4) PAPER.md:142 ------------------
 *   upper[q] = min_k (y[k] + M D^u(q,k)),  lower[q] = max_k (y[k] - M D^l(q,k)),
 *   g[q]     = (upper[q] + lower[q]) / 2.
 * X [N*d], y [N], Xq [Q*d]; upper/lower/g [Q], each may be NULL (at least one non-NULL unless Q=0).
 * Q = 0 returns LIPFIT_OK and writes nothing.  M = 0 is allowed.  Inconsistent data
 * (lower > upper somewhere) are not an error.
 * Steps on the device: a1 prepack (permute / mirror / weight the coordinates, build records)
 * then a2 fused distance + running min/max; the Q x N distance matrix is never formed.
 * Evaluation policy LIPFIT_BOUNDS_AUTO (see lipfit_bounds_ex). */
int lipfit_bounds(const float* X, const float* y, int64_t N, int32_t d,
                  const float* Xq, int64_t Q, float M,
                  const int32_t* mono_mask /* host[d] or NULL */, int32_t norm,
                  const float* weights /* host[d] or NULL */,
                  float* upper, float* lower, float* g, void* cuda_stream);

/* Same, every array pointer a HOST pointer (pageable or pinned); copies X, y, Xq to the
 * device, runs lipfit_bounds, copies the non-NULL outputs back and synchronises. */
int lipfit_bounds_host(const float* X, const float* y, int64_t N, int32_t d,
                       const float* Xq, int64_t Q, float M,
                       const int32_t* mono_mask, int32_t norm, const float* weights,
                       float* upper, float* lower, float* g, void* cuda_stream);

/* ---- Eq.(2),(3) without ANY device allocation ------------------------------------------------------
 * For callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that
 * forbid allocation.  Same upper / lower / g as lipfit_bounds_ex(..., LIPFIT_BOUNDS_BRUTE, ...) (every pair is
 * visited; the generic pair arithmetic for any d <= 32, mask, norm, weights), same arguments, layout, ownership
 * and asynchrony on `cuda_stream` -- but the scratch (packed records, chunk-merge keys) is a FIXED file-scope
 * device array of 8 MiB inside the library (every GPU that loads the library holds it until the process exits)
 * and the call issues kernel launches only: no cudaMalloc / cudaFree / cudaMallocAsync, no allocating routine.
 * Limits (LIPFIT_E_LIMIT beyond them, nothing launched):
 *     N * (DP + 4) <= LIPFIT_NOALLOC_MAX_RECORD_FLOATS,  DP = d rounded up to 4 / 8 / 16 / 32
 *         (N <= 131072 for d <= 4, 87381 for d <= 8, 52428 for d <= 16, 29127 for d <= 32),
 *     Q <= LIPFIT_NOALLOC_MAX_Q = 524288 per call (split larger query sets into several calls).
 * The scratch is SHARED by all calls and keeps the last call's contents; each call rewrites / re-initialises
 * what it reads, so consecutive calls on one stream are independent -- but calls that OVERLAP on the GPU (two
 * streams, two host threads) race on it: serialise them.  The first call on a device looks the array's
 * address up (cudaGetSymbolAddress, with that device current); do that first call outside a graph capture. */
#define LIPFIT_NOALLOC_MAX_RECORD_FLOATS (1 << 20)
#define LIPFIT_NOALLOC_MAX_Q (1 << 19)
int lipfit_bounds_noalloc(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q, float M,
                          const int32_t* mono_mask, int32_t norm, const float* weights,
                          float* upper, float* lower, float* g, void* cuda_stream);

/* ---- Evaluation policy of Eq.(2),(3) -------------------------------------------------------------
 * The result of lipfit_bounds is always the minimum / maximum over ALL N data (within the fp32 tolerance
 * of DESIGN.md section 6, whichever pass computes it); the policy only chooses how many pairs are visited:
 *   LIPFIT_BOUNDS_BRUTE   every (query, datum) pair, the fused all-pairs kernels (step a2): N Q pair
 *                         evaluations "proportional to N" per query as in PAPER.md:130.
 *   LIPFIT_BOUNDS_PRUNED  exact spatial pruning (NEXT-4(ii), see lipfit_bounds_pruned below).
 *   LIPFIT_BOUNDS_AUTO    what lipfit_bounds / lipfit_bounds_host do: a single-launch kernel that keeps all N data
 *                         in shared memory when the call is latency-bound (N (DP + 4) floats <= 46 KB and
 *                         N Q <= 2^25 pairs: BASELINE configs[0] takes 14 us instead of 25 us), else
 *                         PRUNED when d <= 8, N >= 8192,
 *                         Q >= 4096 and N Q >= 2^32 (few enough coordinates for bounding boxes to separate,
 *                         enough pairs to pay for two radix sorts: 9.7x / 5.3x / 2.0x on the config 2 / 5 / 3
 *                         workloads), BRUTE otherwise.  Pruning cannot help when the candidates y + M D of far
 *                         data compete with those of near data everywhere (M D comparable to the spread of y
 *                         across the whole domain): the pruned pass then visits most pairs at about half the
 *                         all-pairs rate.  AUTO guards against that: the pruned kernel keeps the running fraction
 *                         of pairs its finished groups of 32 queries evaluated and, above 40 %, stops handing out
 *                         groups; the call then runs BRUTE instead (ONE stream synchronisation inside the call,
 *                         after the pruned kernel, to read that decision back; only for Q >= 4608 x the number
 *                         of SMs, i.e. when the groups come in enough waves for stopping to save work).  The
 *                         result is the same exact minimum / maximum whichever pass runs.  Callers who must not
 *                         synchronise pass LIPFIT_BOUNDS_BRUTE or LIPFIT_BOUNDS_PRUNED.
 * pairs_evaluated: HOST int64[3] or NULL, as in lipfit_bounds_pruned ([0] = N Q under BRUTE); non-NULL
 * synchronises the stream.  Unknown policy: LIPFIT_E_PARAM. */
enum lipfit_bounds_policy { LIPFIT_BOUNDS_AUTO = 0, LIPFIT_BOUNDS_BRUTE = 1, LIPFIT_BOUNDS_PRUNED = 2 };
int lipfit_bounds_ex(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q, float M,
                     const int32_t* mono_mask, int32_t norm, const float* weights,
                     float* upper, float* lower, float* g, int32_t policy,
                     int64_t* pairs_evaluated /* host[3] or NULL */, void* cuda_stream);
int lipfit_bounds_host_ex(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                          float M, const int32_t* mono_mask, int32_t norm, const float* weights,
                          float* upper, float* lower, float* g, int32_t policy,
                          int64_t* pairs_evaluated /* host[3] or NULL */, void* cuda_stream);

/* ---- NEXT-4(iii): Eq.(2),(3) under monotonicity on PARTS of the domain (section 4.2) ----
 * "Partition the domain with respect to each variable i into the intervals A: x_i <= a_i, AB: a_i <= x_i <= b_i,
 * B: x_i >= b_i" and "Case I: f increasing on A, B, unrestricted on AB.  Case II: f decreasing on A, B ...
 * Case III: f decreasing on A, increasing on B ...  Case IV: f increasing on A, decreasing on B";
 * the package passes `mon in {0,1,2,3,4}^dim` and `a, b in R^dim`.  The paper does not print the
 * modified bounds ("can be expressed through components of the distance vector"); reading R26
 * of DESIGN.md derives them: walking coordinate i from the datum x^k_i to the query x_i,
 *   u_i = w_i (length of the way in AB + length in A / in B where f may GROW in the direction of travel)
 *   l_i = w_i (length of the way in AB + length in A / in B where f may FALL in the direction of travel)
 * ("may grow" = travelling up through an increasing region or down through a decreasing one), and
 *   upper[q] = min_k (y[k] + M ||u||_p),  lower[q] = max_k (y[k] - M ||l||_p),  g = (upper + lower) / 2.
 * mon: HOST int32[d] or NULL (= all 0), 0 = unrestricted, 1..4 = case I..IV.  a, b: HOST float[d], required
 * when some mon[i] != 0, a[i] <= b[i]; a[i] = -inf (no region A) and b[i] = +inf (no region B) are allowed;
 * entries of coordinates with mon[i] = 0 are ignored.  a = b with case I / II is lipfit_bounds with mask
 * +1 / -1 (Eq.(4)).  Every pair is visited (no pruning).  Other arguments, layout, ownership, error
 * behaviour and asynchrony as lipfit_bounds; bad mon / a > b / NaN: LIPFIT_E_PARAM. */
int lipfit_bounds_region(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                         float M, const int32_t* mon /* host[d] or NULL */, const float* a /* host[d] */,
                         const float* b /* host[d] */, int32_t norm, const float* weights /* host[d] or NULL */,
                         float* upper, float* lower, float* g, void* cuda_stream);

/* ---- Approximation with k > 1 neighbours ("Extra features" 2) -------
 *   upper[q] = sum_j wk[j] * (j-th smallest of y[k] + M D^u(q,k)),
 *   lower[q] = sum_j wk[j] * (j-th largest  of y[k] - M D^l(q,k)),   j = 1..k,   g = (upper+lower)/2
 * "the weights of the 'nearest' neighbour, second nearest and so on ... The data set will not be
 * interpolated".  wk: HOST float[k], wk[j] >= 0 finite (assumed to add to 1; not enforced);
 * 1 <= k <= min(N, LIPFIT_MAX_TOPK); k = 1, wk = {1} is lipfit_bounds.  Other arguments, layout and
 * error behaviour as lipfit_bounds; asynchronous on the stream. */
int lipfit_bounds_topk(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                       float M, const int32_t* mono_mask, int32_t norm, const float* weights, int32_t k,
                       const float* wk /* host[k] */, float* upper, float* lower, float* g,
                       void* cuda_stream);

/* ---- NEXT-4(ii): the same upper / lower / g as lipfit_bounds, evaluated with EXACT spatial pruning ----
 * (the paper evaluates every bound in time "proportional to N", and prunes only
 * heuristically, pairs of the smoothing problem).  Data and queries are sorted along a Morton curve of the transformed coordinates; tiles of
 * 32 data carry a bounding box and the range of their values; a tile is skipped for a group of
 * queries when  ymin + M dlb^u >= every running upper bound  and  ymax - M dlb^l <= every running
 * lower bound  of the group (dlb = smallest possible distance between the boxes), which proves that
 * no datum of the tile can change a minimum of Eq.(2) or a maximum of Eq.(3).  The result is the
 * min / max over ALL N data of the per-pair fp32 arithmetic; only the number of pairs evaluated
 * changes (by orders of magnitude for low d, not at all in the worst case).
 * Equivalent to lipfit_bounds_ex(..., LIPFIT_BOUNDS_PRUNED, pairs_evaluated, stream).
 * Arguments, layout, ownership and error behaviour as lipfit_bounds.  pairs_evaluated: HOST int64[3]
 * or NULL; when non-NULL the call synchronises the stream and stores [0] the number of (query, datum)
 * pairs whose distance was actually computed (Q N for the unpruned path), [1] the number of
 * (query group, tile) combinations that passed the box-to-box test, [2] the number of (query, tile)
 * combinations whose own point-to-box test asked for an evaluated tile (diagnostics). */
int lipfit_bounds_pruned(const float* X, const float* y, int64_t N, int32_t d,
                         const float* Xq, int64_t Q, float M,
                         const int32_t* mono_mask, int32_t norm, const float* weights,
                         float* upper, float* lower, float* g, int64_t* pairs_evaluated /* host */,
                         void* cuda_stream);

/* ---- Eq.(7) PAPER.md:197 objective and gradient with the same exact pruning -----------------------
 * Same F and grad as lipfit_smooth_objective (same reading of Eq.(5),(6)).  From datum i's side the two
 * penalty terms of the pair (i,k) are the violations of the upper bound  z_k + M d_s(x^k,x^i)  and of the
 * lower bound  z_k - M d_s(x^i,x^k)  at x^i, so a tile B of data is skipped for the data of a tile A when
 * zmin_B + M dlb^u >= zmax_A  and  zmax_B - M dlb^l <= zmin_A : every term of that tile pair is exactly 0.
 * This is the exact counterpart of the M/3 pair-removal heuristic of PAPER.md:214-218.
 * lipfit_smooth evaluates Eq.(7) with this pass when no coordinate is constrained and N >= 8192 (where it
 * wins by an order of magnitude), with the all-pairs pass otherwise.
 * X [N*d], y [N], eps [N] (device, eps may be NULL = 0); *F HOST double (required; the call
 * synchronises); grad [N] device fp32 or NULL; pairs_evaluated HOST int64 or NULL (ordered pairs whose
 * distances were computed, N(N-1) for the unpruned pass). */
int lipfit_smooth_objective_pruned(const float* X, const float* y, int64_t N, int32_t d, float M,
                                   const int32_t* mono_mask, int32_t norm, const float* weights, float p,
                                   const float* eps, double* F /* host */, float* grad,
                                   int64_t* pairs_evaluated /* host */, void* cuda_stream);

/* ---- k nearest data per query by distance (d_(1) <= d_(2) <= ...) -------------
 * side 0: symmetric weighted norm, mask ignored; +1: D^u; -1: D^l.
 * idx [Q*k] int32 and dist [Q*k] fp32, row-major, ascending distance per query.
 * Selection runs in fp32 (symmetric L2: cross-term key ||x||^2 - 2 q.x) on a pool of k + margin
 * candidates; the pool is re-ranked in fp64 from the original fp32 inputs, sorted by
 * (distance, index); a per-query certificate (exact k-th distance below every pool threshold
 * minus a bound of the fp32 key error) proves the pool contained the answer, and the rare
 * queries where it fails are redone by an exact fp64 scan.  The returned set is therefore the
 * exact fp64 one (ties by lower index); dist is the fp64 distance rounded to fp32. */
int lipfit_knn(const float* X, int64_t N, int32_t d, const float* Xq, int64_t Q,
               const int32_t* mono_mask, int32_t side, int32_t norm, const float* weights,
               int32_t k, int32_t* idx, float* dist, void* cuda_stream);

int lipfit_knn_host(const float* X, int64_t N, int32_t d, const float* Xq, int64_t Q,
                    const int32_t* mono_mask, int32_t side, int32_t norm, const float* weights,
                    int32_t k, int32_t* idx, float* dist, void* cuda_stream);

/* lipfit_knn with per-call options and diagnostics (nothing process-wide is read or written).
 * flags: LIPFIT_KNN_NO_TENSOR_CORES keeps the selection of symmetric L2, d <= 16 on the CUDA cores
 *   (FFMA2 cross-term kernel) instead of the tcgen05 bf16x3 GEMM of csrc/knn_tc.cu; the results are
 *   identical (both feed the same exact re-rank).  Unknown bits: LIPFIT_E_PARAM.
 * info: HOST pointer or NULL.  When non-NULL the call synchronises the stream and fills
 *   fallbacks        queries whose superset certificate failed and that were therefore answered by the
 *                    exact fp64 scan (0 on typical data),
 *   key_error_ratio  largest observed |selection key - exact fp64 key| / the certificate's error bound E
 *                    over every pool candidate of this call (the bound is sound iff <= 1; the tests
 *                    assert it on every kNN case),
 *   tensor_cores     1 if the tcgen05 selection kernel ran. */
#define LIPFIT_KNN_NO_TENSOR_CORES 1
typedef struct lipfit_knn_info {
    int64_t fallbacks;
    double key_error_ratio;
    int32_t tensor_cores;
    int32_t reserved;
} lipfit_knn_info;
int lipfit_knn_ex(const float* X, int64_t N, int32_t d, const float* Xq, int64_t Q,
                  const int32_t* mono_mask, int32_t side, int32_t norm, const float* weights,
                  int32_t k, int32_t* idx, float* dist, int32_t flags, lipfit_knn_info* info /* host */,
                  void* cuda_stream);

/* ---- Penalty smoothing, Eq.(5)-(7) PAPER.md:189-198 ---------------------------------------
 * F(eps) = ||eps||^2/p + sum_{i!=k} (z_i - z_k - M d_s(x^k,x^i))_+^2
 *                      + sum_{i!=k} (z_k - z_i - M d_s(x^i,x^k))_+^2,   z = y + eps,
 * all N(N-1) ordered pairs recomputed on the fly (no N x N matrix).
 * lipfit_smooth_objective: eps [N] device (NULL = 0); *F host double (may be NULL: then the call
 * is asynchronous and only grad is produced); grad [N] device fp32 (may be NULL). */
int lipfit_smooth_objective(const float* X, const float* y, int64_t N, int32_t d, float M,
                            const int32_t* mono_mask, int32_t norm, const float* weights, float p,
                            const float* eps, double* F /* host */, float* grad, void* cuda_stream);

typedef struct lipfit_smooth_info {
    int32_t iters;          /* LBFGS iterations taken */
    int32_t evals;          /* objective/gradient evaluations (device passes) */
    int32_t status;         /* 0 converged (gnorm_inf <= tol_grad), 1 max_iter, 2 no further progress */
    int32_t reserved;
    double F0, F;           /* objective at eps = 0 and at the returned eps */
    double gnorm_inf;       /* ||grad F||_inf at the returned eps */
    double max_violation0;  /* max_{i!=k} (z_i - z_k - M d_s(x^k,x^i))_+ at eps = 0 ... */
    double max_violation;   /* ... and at the returned eps */
} lipfit_smooth_info;

/* Minimises F from eps = 0 by LBFGS on the host, each evaluation one
 * device pass; then y_inout <- y + eps on the device.  eps_out [N] device or
 * NULL; info host or NULL.  Synchronises the stream.  Stops at gnorm_inf <= tol_grad (status 0), at
 * max_iter (status 1), or (status 2) when no decrease can be found / the quasi-Newton model predicts a
 * decrease below 1e-9 |F|, the resolution of the fp32-evaluated objective. */
int lipfit_smooth(const float* X, float* y_inout, int64_t N, int32_t d, float M,
                  const int32_t* mono_mask, int32_t norm, const float* weights, float p,
                  int32_t max_iter, double tol_grad, float* eps_out, lipfit_smooth_info* info,
                  void* cuda_stream);

int lipfit_smooth_host(const float* X, float* y_inout, int64_t N, int32_t d, float M,
                       const int32_t* mono_mask, int32_t norm, const float* weights, float p,
                       int32_t max_iter, double tol_grad, float* eps_out, lipfit_smooth_info* info,
                       void* cuda_stream);

/* ---- Smallest Lipschitz constant consistent with the data ---------------
 *   L = max over ordered pairs i != k with y_i > y_k of (y_i - y_k) / d_s(x^k, x^i)
 * (the least M for which constraint (5) holds; without monotonicity max |y_i-y_k| / ||x^i-x^k||).
 * "N^2 operations, but no storage of the distance matrix": the data are sorted by y
 * and every unordered pair is visited once by the smoothing sweep with a running-maximum filter.
 * L: one fp32 (device for lipfit_lipschitz_constant, asynchronous; host for the _host variant,
 * which copies X, y in and synchronises).  +inf if a pair with y_i > y_k has zero distance, 0 if no
 * pair qualifies (N = 1, constant y).  The fp32 sweep only FILTERS (conservatively: a pair is
 * dropped only if it provably cannot beat the running maximum); surviving pairs are evaluated
 * in fp64 from the original inputs, so L is the exact fp64 maximum rounded to fp32. */
int lipfit_lipschitz_constant(const float* X, const float* y, int64_t N, int32_t d,
                              const int32_t* mono_mask, int32_t norm, const float* weights,
                              float* L /* device[1] */, void* cuda_stream);
int lipfit_lipschitz_constant_host(const float* X, const float* y, int64_t N, int32_t d,
                                   const int32_t* mono_mask, int32_t norm, const float* weights,
                                   float* L /* host */, void* cuda_stream);

/* ---- Local Lipschitz interpolation, PAPER.md:169-183 (section 4.3) --------------------------
 * Radial symmetric weighted distance D(a,b) = ||w (a - b)||_p (no monotonicity: the paper gives no
 * formula for combining the two, R23).  J = LIPFIT_LOCAL_KNOTS for the last two calls.
 *
 * lipfit_distance_quantiles: spline knots = nearest-rank j/J quantiles (j = 1..J) of the S sampled
 *   inter-point distances D(x^{pair_i[s]}, x^{pair_k[s]}) ("quantiles of the distribution
 *   of distances ... approximated from a sample of interpoint distances"; the sample is an INPUT).
 *   pair_i, pair_k: device int32[S]; knots: HOST float[J], 1 <= J <= 1024, J <= S; synchronises.
 * lipfit_local_lipschitz: per-datum non-decreasing step functions
 *   table[k*J+j] = max(|y_k - y_(1)|/d_(1), max_{i != k, D(x^k,x^i) <= knots[j]} |y_k - y_i|/D),
 *   last knot treated as +infinity; +inf where a different value sits at zero distance.
 *   knots: HOST float[J]; table: device float[N*J]; asynchronous.  An all-pairs pass (N^2 pairs).
 * lipfit_values_local: Eq.(2),(3) with M replaced by M_k(D(x, x^k)) = table[k][first j with
 *   D <= knots[j], else J-1]; upper/lower/g as in lipfit_bounds. */
int lipfit_distance_quantiles(const float* X, int64_t N, int32_t d, int32_t norm, const float* weights,
                              const int32_t* pair_i, const int32_t* pair_k, int64_t S, int32_t J,
                              float* knots /* host[J] */, void* cuda_stream);
int lipfit_local_lipschitz(const float* X, const float* y, int64_t N, int32_t d, int32_t norm,
                           const float* weights, const float* knots /* host[J] */, int32_t J,
                           float* table /* device[N*J] */, void* cuda_stream);
int lipfit_values_local(const float* X, const float* y, int64_t N, int32_t d, const float* Xq, int64_t Q,
                        int32_t norm, const float* weights, const float* knots /* host[J] */, int32_t J,
                        const float* table /* device[N*J] */, float* upper, float* lower, float* g,
                        void* cuda_stream);

/* ---- Host optimiser on its own (step a5), exposed so that it can be tested without a GPU ----
 * Minimises a caller-supplied function by the same LBFGS lipfit_smooth uses (history `history`,
 * strong-Wolfe line search).  x: host double[n], start point on entry and
 * result on exit.  fn returns 0 on success; a non-zero value aborts and is returned (negated if
 * positive).  info may be NULL; only iters, evals, status, F0, F, gnorm_inf are filled. */
typedef int (*lipfit_eval_fn)(void* user, const double* x, double* f, double* grad);
int lipfit_lbfgs(int64_t n, double* x, lipfit_eval_fn fn, void* user, int32_t max_iter,
                 double tol_grad, int32_t history, lipfit_smooth_info* info);

/* ---- Introspection ----------------------------------------------------------------------- */
const char* lipfit_status_string(int code);
/* "major.minor.patch" of this library. */
const char* lipfit_version(void);
/* Number of kernel launches this library has issued since load (all threads); used by
 * bench.py's gpu_launches.  Monotone counter, not reset. */
int64_t lipfit_launch_count(void);
/* Returns the cached workspaces of the current device's private pool to the driver
 * (cudaMemPoolTrimTo(pool, 0)); workspaces of calls still in flight are unaffected. */
int lipfit_release_workspace(void);
/* Device timing of the dominant kernels, for roofline reports (bench.py).  PROCESS-WIDE diagnostic
 * (see "Thread safety" above).  lipfit_set_timing(1) resets the accumulators and makes every later launch
 * of the dominant kernels (which: 0 = fused bounds, 1 = kNN selection, 2 = smoothing all-pairs,
 * 3 = Lipschitz-constant all-pairs, 4 = local step tables, 5 = local evaluation, 6 = pruned bounds,
 * 7 = pruned smoothing pass, 8 = kNN re-rank, 9 = top-k bounds, 10 = region-monotone bounds) bracketed by
 * CUDA events on its own stream; such calls wait for that kernel.  lipfit_set_timing(0) switches it off
 * (default).  lipfit_get_timing returns the accumulated device milliseconds and the number of launches. */
void lipfit_set_timing(int32_t on);
int lipfit_get_timing(int32_t which, double* total_ms, int64_t* launches);
/* DIAGNOSTIC behind the "alu" roofline peak (bench.py --pipes): measured issue rate on the
 * current device of one fp32 instruction class, which = 0 FFMA, 1 FADD, 2 FADD2 (packed f32x2), 3 FFMA2,
 * 4 FMNMX, 5 FMNMX3 (3-input), 6 MUFU.SQRT, 7 FFMA and FMNMX interleaved, 8 FADD2 and FMNMX3 interleaved,
 * 9 FADD with the |.| source modifier, 10-15 further FMA-pipe / ALU-pipe mixes (lipfit_pipe_name says which).  32 warps per SM run 8 independent chains each; the two HOST outputs
 * (either may be NULL) are lane-results per clock per SM (a packed instruction retires 2 per lane, FMNMX3 folds
 * 2 comparisons) and warp instructions per clock per SM.  Synchronises the stream; LIPFIT_E_PARAM for an
 * unknown `which` (lipfit_pipe_name returns "" then). */
int lipfit_pipe_throughput(int32_t which, double* lane_results_per_clk_sm /* host */,
                           double* warp_instr_per_clk_sm /* host */, void* cuda_stream);
const char* lipfit_pipe_name(int32_t which);
/* Name of the selection kernel lipfit_knn_ex would use for (d, side, norm, flags). */
int lipfit_knn_variant(int32_t d, int32_t side, int32_t norm, int32_t flags, char* out, int32_t cap);
/* Name of the kernel variant lipfit_bounds would dispatch to for (d, mask, norm), e.g.
 * "bounds<L1,U2,C2,R8>" or "bounds_generic<L2,DP8>"; writes at most `cap` bytes incl. NUL. */
int lipfit_bounds_variant(int32_t d, const int32_t* mono_mask, int32_t norm, char* out, int32_t cap);

#ifdef __cplusplus
}
#endif
#endif /* LIPFIT_H */
