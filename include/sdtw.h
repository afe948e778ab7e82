/*
 * sdtw.h -- C ABI of libsdtw: Soft-DTW value, gradient and fixed-step barycenter descent on one B200 (sm_100a).
 *
 * The operation (arXiv 2404.12134, "Warped Time Series Anomaly Detection", section 3.3; line numbers are those of
 * /root/reference/PAPER.md):
 *
 *   pair k:  x_k in R^{n_k x d} (a cycle),  Z in R^{m x d} (the barycenter / prototype)
 *   Def. 3 (l.119-121)   D_k[i][j] = delta(x_k[i], Z[j]) = sum_c (x_k[i][c] - Z[j][c])^2   (squared Euclidean)
 *   eq. 3  (l.149-152)   min^gamma(a) = -gamma log sum_p exp(-a_p / gamma)
 *   eq. 5  (l.162-167)   r_00 = 0, r_i0 = r_0j = inf, r_ij = D_ij + min^gamma(r_{i-1,j-1}, r_{i-1,j}, r_{i,j-1});
 *                        value_k = Soft-DTW^gamma(x_k, Z) = r_{n_k, m}
 *   eq. 6  (l.175-183)   grad_Z value_k = (dD_k/dZ)^T E_k,  E_k = d value_k / d D_k (the expected alignment matrix,
 *                        obtained by the reverse recurrence of the paper's ref. [19]); with squared-Euclidean delta
 *                        g_k[j][c] = sum_i E_k[i][j] * 2 * (Z[j][c] - x_k[i][c])
 *   eq. 7  (l.187-192)   barycenter objective sum_k value_k(Z) (plain sum: lambda_k = 1, no 1/n_k; C6),
 *                        minimised by fixed-step gradient descent (l.185):  Z <- Z - step * sum_k g_k.
 *
 * Conventions for every entry point
 *   - "dev" pointers are CUDA device pointers owned by the caller (e.g. torch tensors); "host" pointers are ordinary
 *     host memory.  The library never frees or keeps a caller pointer after the enqueued work has run.
 *   - Layout is time-major, channel-minor: Z is [m][d], X_concat is [sum_k n_k][d], both contiguous float32.
 *     offsets is a HOST array of N+1 int64 row indices into X_concat: offsets[0] = 0, strictly increasing,
 *     cycle k = rows offsets[k] .. offsets[k+1]-1.  It is read during the call only.
 *   - stream is a cudaStream_t (NULL = the legacy default stream).  Device entry points only ENQUEUE work on it: no
 *     host synchronisation and no device-to-host copy (exception: the first call with a new (offsets, m, d) shape
 *     uploads a few KB of plan metadata with one pageable cudaMemcpyAsync).  The caller keeps all buffers alive until
 *     the stream has drained.  Results are bitwise reproducible run to run for fixed inputs (no atomics on data).
 *   - Return value: SDTW_OK (0) or a negative SDTW_ERR_* code.  No exception crosses the ABI.  On an argument error
 *     nothing is enqueued and outputs are untouched.  NaN/Inf in the DATA is not scanned for (it propagates).
 *   - d is supported for 1 <= d <= SDTW_MAX_D (compiled maximum; SDTW_DTW_MAX_D for sdtw_dtw_score / sdtw_subdtw);
 *     1 <= n_k, m < 2^30; 1 <= N < 2^24.
 *   - There is no CPU fallback: on a device that is not compute capability 10.x the calls return SDTW_ERR_UNSUPPORTED.
 *   - CO-RESIDENCY.  The forward, reverse and DTW kernels are persistent grids sized by the occupancy query so that every
 *     CTA is resident at once; a CTA that waits for a strip-boundary value spins (with nanosleep back-off) on data words
 *     another resident CTA writes.  That holds when the library has the SMs it was promised: a whole GPU, or a MIG
 *     slice.  Where the CTAs of one grid may NOT all be resident -- another process time-slicing or sharing the SMs
 *     through MPS with a limited active-thread percentage, a debugger single-stepping a CTA, a concurrent kernel of the
 *     caller's that occupies SMs for as long as this grid waits for them -- a waiting CTA can wait for one that is not
 *     scheduled, and the call then does not return: there is no time-out in the wait loops and no SDTW_ERR_* for this.
 *     Kernels of the caller that merely run to completion beside the library's only delay it.
 */
#ifndef SDTW_H_
#define SDTW_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SDTW_OK 0
#define SDTW_ERR_INVALID_ARG (-1) /* NULL required pointer, m/d/N < 1, gamma <= 0 or non-finite, empty cycle, ... */
#define SDTW_ERR_UNSUPPORTED (-2) /* d > SDTW_MAX_D, sizes beyond the stated limits, device is not sm_100        */
#define SDTW_ERR_WORKSPACE (-3)   /* the workspace budget does not hold the call (or, with waves, one pair)      */
#define SDTW_ERR_CUDA (-4)        /* a CUDA runtime call failed; see sdtw_last_cuda_error()                      */
#define SDTW_ERR_STATIC_LIMIT (-5) /* sdtw_value_static: the problem needs more than the built-in scratch array holds */

#define SDTW_MAX_D 4
#define SDTW_DTW_MAX_D 9 /* sdtw_dtw_score / sdtw_subdtw: the paper's Step 1 aligns all 9 robot variables at once (l.300) */

/*
 * sdtw_value_grad -- eq. 5 and eq. 6 for N pairs (x_k, Z), summed over k.
 *   Z          dev  [m][d]            barycenter (read only)
 *   X_concat   dev  [offsets[N]][d]   the N cycles back to back (read only)
 *   offsets    HOST [N+1] int64
 *   gamma      > 0, finite (gamma = 0, the hard-DTW case of eq. 3, is rejected)
 *   out_values dev  [N] float32, value_k in the caller's pair order; may be NULL
 *   out_grad   dev  [m][d] float32, sum_k g_k (plain sum, not averaged); NULL => forward only (no checkpoints are
 *              written and no reverse pass runs -- the scoring-sweep configuration)
 */
int sdtw_value_grad(const float* Z, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                    float gamma, float* out_values, float* out_grad, void* stream);

/*
 * sdtw_barycenter -- `iters` iterations of  Z <- Z - step * sum_k g_k(Z)  (l.185, eq. 7), all on `stream`.
 *   Z_inout       dev [m][d]   Z0 on entry, the last iterate on return (the only buffer written in place)
 *   iters         >= 0 (0 = no-op);  step finite
 *   out_values    dev [N], value_k at the LAST EVALUATED iterate Z^(iters-1); may be NULL
 *   out_objective dev [iters], sum_k value_k(Z^(t)) before the t-th update; may be NULL
 */
int sdtw_barycenter(float* Z_inout, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                    float gamma, int32_t iters, float step, float* out_values, float* out_objective, void* stream);

/*
 * Extended calls: the paper's variants of the same path (Def. 7 / eq. 7, l.187-192; Table 1, l.318-319).
 *   weights  HOST [N] float32 or NULL.  w_k multiplies pair k in the objective and in the gradient:
 *            objective = sum_k w_k value_k,  out_grad = sum_k w_k g_k  (eq. 7 has w_k = lambda_k / n_k; NULL = all 1, the
 *            plain sum of sdtw_value_grad).  out_values[k] stay the UNWEIGHTED Soft-DTW values.  Read during the call
 *            only.  Non-finite weight => SDTW_ERR_INVALID_ARG.
 *   band     Sakoe-Chiba band (Table 1 "Bandwidth", a fraction of the longest length: the caller passes
 *            band = floor(0.6 * max(m, max_k n_k)) for the paper's setting).  Read (C18) as the classic
 *            adjustment window: cell (i, j) belongs to an admissible path iff |i - j| <= band; cells outside are
 *            excluded from eq. 5 (r = +inf) and have E = 0.  band < 0 = no band.
 *            band < |n_k - m| for some k => SDTW_ERR_INVALID_ARG (no complete path fits).  A band that excludes cells
 *            of pair k but is narrower than |n_k - m| + 4 (ceil(n_k / m) + 2) + 2 => SDTW_ERR_UNSUPPORTED (the kernel's
 *            value staircase must fit inside the band).
 *   out_objective  dev [1] (value_grad_ex) / dev [iters] (barycenter_ex) float32, sum_k w_k value_k; may be NULL.
 * Everything else is as in sdtw_value_grad / sdtw_barycenter, which are these calls with weights = NULL, band = -1.
 */
int sdtw_value_grad_ex(const float* Z, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                       float gamma, const float* weights, int64_t band, float* out_values, float* out_grad,
                       float* out_objective, void* stream);
int sdtw_barycenter_ex(float* Z_inout, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                       float gamma, const float* weights, int64_t band, int32_t iters, float step, float* out_values,
                       float* out_objective, void* stream);

/*
 * sdtw_barycenter_backtracking -- gradient descent on eq. 7's objective f(Z) = sum_k w_k Soft-DTW(Z, x_k) with an Armijo
 * backtracking line search: the stand-in for the off-the-shelf optimiser of Table 1 (l.320-332; C22).  It
 * removes the step-size fragility of the fixed-step loop with value-only evaluations and vector operations.
 *   iteration it:  t = step0;  up to max_trials times:  Zt = Z - t G;  accept if f(Zt) <= f(Z) - c1 t ||G||^2, else
 *                  t = shrink t.  Accepted: Z = Zt.  None accepted: the descent stops (later iterations do nothing).
 *   weights, band       as in sdtw_value_grad_ex (NULL / -1 for the plain problem)
 *   step0 > 0, 0 < shrink < 1, c1 >= 0, max_trials >= 1, iters >= 0
 *   out_values          dev  [N]  value_k at the final Z; may be NULL
 *   out_objective       HOST [iters + 1] float64, f at Z(0), ..., Z(iters)            (required)
 *   out_steps           HOST [iters] float32, the accepted step of each iteration (0 = none accepted)
 *   out_trials          HOST [iters] int32, evaluations of f spent in each iteration
 * A rejected trial costs one forward sweep, an accepted one a forward and a reverse sweep.  The accept / reject test is
 * taken on the host in float64 on the kernel's objective, so this call BLOCKS: it synchronises `stream` once per
 * trial (two 8-byte device-to-host copies).  The objective is summed in float64 from the float32 per-pair values.
 */
int sdtw_barycenter_backtracking(float* Z_inout, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets,
                                 int32_t N, float gamma, const float* weights, int64_t band, int32_t iters, float step0,
                                 float shrink, float c1, int32_t max_trials, float* out_values, double* out_objective,
                                 float* out_steps, int32_t* out_trials, void* stream);

/*
 * sdtw_barycenter_lbfgs -- the optimiser Table 1 names (l.320-332: "L-BFGS"; the paper takes it off the shelf, so the
 * recursion is the textbook one, Nocedal & Wright Algorithm 7.4, with the Armijo backtracking of
 * sdtw_barycenter_backtracking as its line search; reading C23) on the objective of eq. 7.
 *   d = -H G by the two-loop recursion over the last `hist` accepted pairs (s = Z' - Z, y = G' - G), H0 = (s.y / y.y of
 *   the newest pair) I; a direction with G.d >= 0 drops the pairs and falls back to -G.  Trial steps t = step0 when no
 *   pair is stored, else 1, shrunk by `shrink` up to max_trials times; accept when f(Z + t d) <= f(Z) + c1 t (G.d).
 *   A pair is stored iff s.y > 1e-10 |s| |y|.  hist = 0 is sdtw_barycenter_backtracking.  hist <= 64.
 * Vectors are float32 on the device; dot products are float64 fixed-shape trees read back by the host, which runs the
 * recursion's scalars and the accept test in double: the call BLOCKS (a stream synchronisation per dot product and per
 * trial).  A trial costs a forward sweep; an accepted trial reuses its checkpoints for the reverse sweep.
 * Arguments as sdtw_barycenter_backtracking (out_objective HOST [iters + 1] double, out_steps / out_trials HOST [iters]).
 */
int sdtw_barycenter_lbfgs(float* Z_inout, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                          float gamma, const float* weights, int64_t band, int32_t iters, int32_t hist, float step0,
                          float shrink, float c1, int32_t max_trials, float* out_values, double* out_objective,
                          float* out_steps, int32_t* out_trials, void* stream);

/*
 * sdtw_dtw_score -- Step 3 of the paper (section 3.4, Def. 8 / eq. 8, l.233-242): the classic DTW of eq. 1 (l.123-127;
 * eq. 5 with gamma = 0, squared-Euclidean delta) between the prototype Z and each cycle x_k, the number of cells
 * |pi_k| of the optimal alignment path, and the similarity score d_score = DTW / |pi|.  When several paths attain the
 * minimum the path is the one obtained by preferring the diagonal predecessor, then (i-1, j), then (i, j-1)
 * (C20; the paper does not say).  Arithmetic is plain float32, one rounding per operation, in the order
 * D = sum_c (x_c - z_c)^2 (c ascending), r = D + min(.), score = DTW / float(|pi|).
 *   out_dtw      dev [N] float32, DTW(x_k, Z) in the caller's pair order; may be NULL
 *   out_pathlen  dev [N] int32, |pi_k|  (max(n_k, m) <= |pi_k| <= n_k + m - 1); may be NULL
 *   out_score    dev [N] float32, out_dtw[k] / out_pathlen[k]; may be NULL
 * Forward only, full matrix (no band), no special functions; same argument / stream / workspace conventions.
 * n_k + m must stay below 2^24 (SDTW_ERR_UNSUPPORTED otherwise; the same holds for sdtw_subdtw).
 */
int sdtw_dtw_score(const float* Z, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                   float* out_dtw, int32_t* out_pathlen, float* out_score, void* stream);

/*
 * sdtw_subdtw -- the primitive of Step 1, segmentation into cycles (section 3.2, eq. 2, l.129-145): Sub-DTW between the
 * reference quasi-period Z (all m samples traversed: i_1 = 1, i_k = M in the paper's notation) and the best
 * subsequence of each window x_k (free first and last index along the window):
 *     value_k = min_{a <= b} DTW(Z, x_k[a..b])      a*_k, b*_k = first / last row of x_k on the optimal path.
 * Ties: b* is the smallest row attaining the minimum, and the path is the diagonal-up-left preference of
 * sdtw_dtw_score (C20).  Same float32 arithmetic, one rounding per operation.
 *   Z          dev [m][d]   the reference cycle;  X_concat dev, offsets HOST: the N windows back to back
 *   out_value  dev [N] float32;  out_a, out_b  dev [N] int32, 0-based, inclusive.  Any of them may be NULL.
 * The sliding-window loop of l.137-143 is sequential (each window starts where the previous cycle ended); the
 * binding's segment_cycles() drives it with one call per window.
 */
int sdtw_subdtw(const float* Z, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                float* out_value, int32_t* out_a, int32_t* out_b, void* stream);

/*
 * sdtw_gd_update -- the descent step alone: Z[t] <- Z[t] - step * G[t] for t < count (= m*d).  Used when the
 * gradient is all-reduced across GPUs between sdtw_value_grad and the update.
 */
int sdtw_gd_update(float* Z_inout, const float* G, int64_t count, float step, void* stream);

/*
 * sdtw_value_static -- the forward-only sweep of sdtw_value_grad (eq. 5, l.162-167: value_k = Soft-DTW^gamma(x_k, Z) for
 * every pair, no gradient) for callers that must not allocate device memory.
 *
 * Who that is: a plug-in running inside a host application that reserved the whole GPU for its own memory pool up front
 * (a cudaMalloc from a guest library then fails, or fragments the pool); a control or monitoring loop with a latency
 * budget, where the implicit device-wide synchronisation of cudaMalloc / cudaFree stalls every other stream; code that
 * runs where the platform forbids allocation after start-up (certified or long-running services that fix their memory
 * footprint at load time).  Every other entry point of this header may allocate: the plan metadata of a new shape and,
 * unless sdtw_set_workspace() registered a buffer, the workspace.  This one never does.
 *
 * How: all scratch of the sweep (scaled input copies, work-queue counters, strip-boundary columns, per-strip value
 * partials, the per-pair schedule table) lives in ONE array of SDTW_STATIC_SCRATCH_BYTES (32 MiB) that is compiled into
 * the library as a static device variable.  Every GPU on which the library's CUDA module is loaded carries those 32 MiB
 * from load until the process exits, whether or not this call is ever made; that is the price of the guarantee.  The
 * call issues kernel launches only (the same prologue / forward / epilogue kernels as sdtw_value_grad with out_grad ==
 * NULL, column layout, so out_values are BITWISE what that call returns): no cudaMalloc, cudaFree, cudaMallocAsync,
 * event or stream creation, no memcpy, no host synchronisation.  Profiling (sdtw_debug.h) is ignored by this call.
 *
 * Limits.  N <= SDTW_STATIC_MAX_PAIRS (64; the schedule table travels as a kernel argument), and the sweep's scratch
 * must fit the array: roughly  4 * (n_k + 128) * ceil(m / 128)  bytes per pair  +  8 * d * (sum_k n_k + m)  bytes.
 * 32 MiB holds one pair of the paper's size (n_k <= 33000 against m = 30000, any d <= SDTW_MAX_D), or 64 pairs of
 * 3000 x 3000.  Beyond either limit: SDTW_ERR_STATIC_LIMIT, nothing enqueued, outputs untouched.  Other argument errors
 * as in sdtw_value_grad.
 *
 * Sharing.  There is one array per GPU and every call on that GPU uses it, from whichever host thread or stream.  A
 * call first re-initialises what has to start clean (queue counters to zero, boundary columns to the "not yet written"
 * pattern), so leftovers of the previous call are harmless -- but two calls whose kernels are in flight at the same
 * time (different streams, or different host threads on different streams) overwrite each other's scratch and return
 * garbage or hang.  Keep calls on one GPU stream-ordered: same stream, or an event between them.  The library does not
 * order them for you (that would need an event, i.e. a resource created at run time).
 *
 * Set-up.  The FIRST call on each device resolves the device address of the array (cudaGetSymbolAddress, with that
 * device current -- the caller makes the device current, as for every call here) and remembers it; later calls on that
 * device skip this step.  Make that first call during start-up, before any stream capture is begun -- and before the
 * host application takes the rest of the GPU's memory: the CUDA driver creates the array when it loads this library's
 * module on the device, which (CUDA loads modules lazily) happens at the first libsdtw call that touches the device.
 * For the same reason the first launch of the sweep for each channel count d makes the driver load that kernel's code
 * (a one-off 2 MiB step in the device's free memory, measured): call once per d you will use, at start-up.
 *
 *   Z, X_concat  dev, offsets HOST [N+1], gamma: as in sdtw_value_grad
 *   out_values   dev [N] float32 (required), value_k in the caller's pair order
 */
#define SDTW_STATIC_SCRATCH_BYTES (32u << 20)
#define SDTW_STATIC_MAX_PAIRS 64
int sdtw_value_static(const float* Z, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                      float gamma, float* out_values, void* stream);

/*
 * Host-buffer variants (all pointers HOST; pinned memory makes the copies asynchronous).  They copy the inputs to
 * the device, run the device entry point, copy the results back and synchronise `stream` before returning.
 * Used by bench.py's end-to-end leg.  Outputs may be NULL as above.
 */
int sdtw_value_grad_host(const float* Z, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                         float gamma, float* out_values, float* out_grad, void* stream);
int sdtw_barycenter_host(float* Z_inout, int64_t m, int32_t d, const float* X_concat, const int64_t* offsets, int32_t N,
                         float gamma, int32_t iters, float step, float* out_values, float* out_objective, void* stream);

/*
 * Workspace.  sdtw_workspace_bytes() is what one call needs to evaluate all its pairs at once (tile-boundary strips,
 * checkpoints of the forward state: 0.375 bytes per DP cell, per-pair gradient partials).  If a workspace has been
 * registered with sdtw_set_workspace() it is used; otherwise the library keeps one grow-only device buffer per GPU
 * (cudaMalloc on first use / when a larger problem arrives -- that call blocks the host while allocating).  Calls
 * that share the buffer from different streams are ordered on it with an event, so they are safe but not concurrent.
 * sdtw_set_workspace(NULL, 0) unregisters the caller's buffer and frees the library-owned one of the current device.
 * The pointer must be 256-byte aligned.  sdtw_workspace_bytes returns 0 on invalid arguments.
 * WAVES.  When that size exceeds the budget -- sdtw_set_workspace_limit(bytes) if set (0 = unset), else the registered
 * workspace, else what the device has free -- sdtw_value_grad[_ex] and sdtw_barycenter[_ex] evaluate the pair set as
 * consecutive waves of pairs in the same workspace (pairs are independent): per-pair values are bitwise
 * the same, the gradients of the waves are added in wave order (float32 round-off against the unsplit call).  Only when
 * a single pair does not fit the budget: SDTW_ERR_WORKSPACE.  sdtw_dtw_score and sdtw_subdtw split the same way (against
 * sdtw_dtw_workspace_bytes; every output is per pair, so every bit is that of the unsplit call).  The two line-search
 * calls (sdtw_barycenter_backtracking, sdtw_barycenter_lbfgs) do NOT split -- an accepted trial's reverse sweep reuses the
 * checkpoints of all pairs -- and return SDTW_ERR_WORKSPACE when a registered workspace is too small.  A split is silent;
 * with the library-owned buffer the budget is the device's free memory at the time of the call, so a co-tenant that
 * holds memory (a caching allocator) makes calls split into more waves: sdtw_last_wave_count() (sdtw_debug.h) tells.
 * THREADS.  Calls are serialised by one library lock while they enqueue.  The two line-search calls (backtracking,
 * L-BFGS) block on the stream once per trial and hold that lock for their whole run: other threads' libsdtw calls, on
 * any device, wait until they return.
 * Forward-only calls (want_grad == 0) without a band keep O(chunks) boundary state per resident strip plus one
 * boundary column per unit of strips; a forward-only call WITH a band that excludes cells keeps a
 * full boundary column per strip: size its workspace with sdtw_workspace_bytes_ex(..., band).  The forward-only size
 * depends on the SM count of the current device (148 is assumed when no device is current).
 */
size_t sdtw_workspace_bytes(int64_t m, int32_t d, const int64_t* offsets, int32_t N, int want_grad);
size_t sdtw_workspace_bytes_ex(int64_t m, int32_t d, const int64_t* offsets, int32_t N, int want_grad, int64_t band);
/* What one sdtw_dtw_score / sdtw_subdtw call of this shape needs (d <= SDTW_DTW_MAX_D); 0 on invalid arguments. */
size_t sdtw_dtw_workspace_bytes(int64_t m, int32_t d, const int64_t* offsets, int32_t N);
int sdtw_set_workspace(void* dev_ptr, size_t bytes);
int sdtw_set_workspace_limit(size_t bytes);

/* Static description of a status code; the cudaError_t behind the last SDTW_ERR_CUDA on this thread. */
const char* sdtw_status_string(int status);
int sdtw_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SDTW_H_ */
