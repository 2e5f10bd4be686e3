/*
 * vegas.h -- C ABI of the B200-native Vegas iteration library (libvegas_b200.so).
 *
 * What it computes.  One Vegas importance-sampling iteration over n events in d dimensions on
 * [0,1]^d ("importance sampling as implemented in Vegas", section 2.2), the grid
 * refinement that follows every iteration ("refine how the random numbers are generated",
 * PAPER.md:49-51) and the value +- error combination of iterations (result format of Table 1,
 * PAPER.md:83-86).  The integrands are the paper's toy functions (Eqs.(1),(3))
 * plus the synthetic stand-in for its LO single-top run named in
 * BASELINE.json:configs.  All numerical conventions the paper leaves open are the readings
 * C1..C11 listed in DESIGN.md ("Readings of the paper"); BASELINE.json:north_star names the calls.
 *
 * Per event e of iteration k (all in registers / shared memory of one fused kernel):
 *   word_j  = Philox4x32-10(counter = (j>>2, k, e lo, e hi), key = (seed lo, seed hi))[j&3]   (C1,C2)
 *   b_j     = (word_j * n_bins) >> 32 ;  r_j = ((word_j * n_bins mod 2^32) + 1/2) * 2^-32      (C3)
 *   x_j     = X[j][b_j] + (X[j][b_j+1] - X[j][b_j]) * r_j ;  J = prod_j n_bins * Delta_j       (C4)
 *   v       = f(x) * J ;  S1 += v ;  S2 += v^2 ;  H[j][b_j] += v^2 for every j                 (C5,C6)
 * and per iteration  I = S1/n,  sigma^2 = (S2/n - I^2)/(n-1)                                    (C7).
 *
 * Conventions for every entry point
 *   - Return value: 0 (VEGAS_OK) or a negative VEGAS_E* code; vegas_strerror() explains it.  No C++
 *     exception crosses this boundary.  Calls on ONE vegas_grid are not thread-safe; different grids are
 *     independent and may be used from different host threads.  The only process-wide state is internal and
 *     lock-protected: per kernel and device, the shared-memory size already configured for it, and the built-in
 *     scratch array of vegas_iterate_static().
 *   - "host" pointers are ordinary host memory owned by the caller (pageable or pinned), row-major,
 *     fp64 unless stated.  "device" pointers are CUDA device memory owned by the caller.
 *   - The library never allocates device memory and never creates streams: the caller provides one
 *     device workspace at vegas_create() (vegas_workspace_bytes() says how large, 256-byte aligned)
 *     and a CUstream / cudaStream_t handle (as void*, NULL = default stream) per call.  With PyTorch:
 *     torch.empty(nbytes, dtype=torch.uint8, device="cuda").data_ptr() and
 *     torch.cuda.current_stream().cuda_stream.
 *   - Calls that return numbers to host pointers synchronise the given stream before returning.
 *     Calls documented as "asynchronous" only enqueue work on the stream.
 *   - There is NO CPU fallback: without a usable CUDA device every compute call returns VEGAS_ECUDA.
 */
#ifndef VEGAS_B200_H
#define VEGAS_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define VEGAS_OK 0
#define VEGAS_EINVAL (-1)   /* bad argument: dim not in [1,32], n_bins not in [2,256], n_events < 2,
                               unknown integrand id / precision, wrong n_params, workspace too small
                               or misaligned, edges not strictly increasing from 0 to 1, alpha < 0,
                               NULL where a pointer is required                                    */
#define VEGAS_ECUDA (-2)    /* a CUDA runtime call or kernel launch failed (message: vegas_strerror
                               on the grid-less code, details via vegas_last_cuda_error())          */
#define VEGAS_ENUMERIC (-3) /* S1 or S2 came out non-finite, or vegas_refine() met a dimension whose
                               smoothed histogram has no finite positive sum (that dimension's grid
                               is left unchanged, the others are refined)                           */

#define VEGAS_ELIMIT (-4)   /* vegas_iterate_static() only: dim * n_bins is larger than VEGAS_STATIC_MAX_ENTRIES, the
                               shape its fixed built-in scratch was sized for; nothing was launched              */

#define VEGAS_MAX_DIM 32
#define VEGAS_MAX_BINS 256
#define VEGAS_MAX_PARAMS 160

/* integrand ids (reading C5) and their host parameter arrays for vegas_set_params():
 *   VEGAS_F_CONST              f = 1                                               n_params = 0
 *   VEGAS_F_GAUSS              PAPER.md:65 Eq.(1): (a sqrt(pi))^-d exp(-sum_j (x_j-1/2)^2/a^2)
 *                              params = { a }                                      n_params = 1
 *   VEGAS_F_GENZ_PRODUCT_PEAK  PAPER.md:74 Eq.(3) with N = 1: prod_j 1/(c_j^-2 + (x_j-w_j)^2)
 *                              params = { c[0..d-1], w[0..d-1] }                   n_params = 2d
 *   VEGAS_F_BW_POLY            BASELINE.json:configs[4]: s = m_min^2 + x_0 (m_max^2 - m_min^2),
 *                              f = M^2 G^2/((s-M^2)^2 + M^2 G^2) * sum_{i=1..d-1} sum_{k=0..4} a[i][k] x_i^k
 *                              params = { M, G, m_min, m_max, a[1][0..4], ..., a[d-1][0..4] }
 *                                                                                  n_params = 4+5(d-1), d >= 2 */
#define VEGAS_F_CONST 0
#define VEGAS_F_GAUSS 1
#define VEGAS_F_GENZ_PRODUCT_PEAK 2
#define VEGAS_F_BW_POLY 3
/*   VEGAS_F_USER               an integrand supplied as CUDA source and compiled at run time for this grid:
 *                              see vegas_set_user_integrand() below; n_params <= VEGAS_USER_MAX_PARAMS */
#define VEGAS_F_USER 4
/*   VEGAS_F_GENZ_DISCONTINUOUS PAPER.md:67-70 Eq.(2) as printed, N = 1 (reading R19): f = 0 where any
 *                              x_j <= a_j, exp(sum_j c_j x_j) elsewhere.  params = { c[0..d-1], a[0..d-1] }, c_j > 0.
 *                              fp64 only: an event within rounding of a cut would be kept or dropped in a different
 *                              precision than the fp64 oracle decides it in (VEGAS_EINVAL for precision 32). */
#define VEGAS_F_GENZ_DISCONTINUOUS 5
#define VEGAS_USER_MAX_PARAMS 64

/* precision of the per-event arithmetic (reading C11): 64 = everything fp64; 32 = grid table, r, x,
 * J, f and v in fp32, v widened to fp64 before S1 += v, S2 += v^2, H += v^2.  Words, bins, the master
 * grid, the sums, the histogram and the refinement are identical / fp64 in both.  What must fit the fp32 range is
 * v = f J / C with a per-integrand constant C applied after the widening (GAUSS: ln N is folded into the exponent, so
 * f = N exp(-E) is formed in one piece; product peak: the product is formed in four partial quotients, prod c_j is C);
 * intermediate factors do not have to.  Where v itself exceeds 3.4e38 the sums become non-finite and the iteration
 * reports VEGAS_ENUMERIC, nothing is clamped; where it falls below 1.2e-38 it loses digits and then vanishes (the
 * estimate stays finite and is biased low: an un-adapted narrow Gaussian in many dimensions): use VEGAS_FP64 there. */
#define VEGAS_FP64 64
#define VEGAS_FP32 32

typedef struct vegas_grid vegas_grid; /* opaque host object; owns no device memory */

/* Device bytes the caller must provide to vegas_create() for this (dim, n_bins).  0 if invalid. */
size_t vegas_workspace_bytes(int dim, int n_bins);

/* Create a grid on the CURRENT CUDA device with the uniform start grid X[j][i] = i/n_bins (C4),
 * written into the workspace on the default stream (synchronous).  dev_workspace: device pointer,
 * 256-byte aligned, at least vegas_workspace_bytes() bytes, must outlive the grid.  *out receives the
 * handle (host object, released by vegas_destroy).  The integrand defaults to VEGAS_F_CONST. */
int vegas_create(int dim, int n_bins, void* dev_workspace, size_t bytes, vegas_grid** out);
int vegas_destroy(vegas_grid* g);

/* Copy the integrand parameter array (host, fp64, layout above) into the grid object; it is passed
 * to the kernels by value at every launch.  Required before iterating with that integrand id
 * (except VEGAS_F_CONST).  Parameters of several ids can be set; each id keeps its own array. */
int vegas_set_params(vegas_grid* g, int integrand_id, const double* params_host, int n_params);

/* User-supplied integrand (integrands "written in Fortran, C/C++ or even CUDA" are the paper's
 * usability claim).  cuda_source (host, NUL-terminated) is CUDA C++ that defines
 *
 *     struct vegas_user_integrand {
 *         __device__ void   begin(int dim, const double* p);          // start of an event
 *         __device__ void   dim(int j, double x, const double* p);    // once per dimension j, x = x_j in (0,1);
 *                                                                     // the ORDER of the calls is unspecified
 *         __device__ double finish(const double* p);                  // f(x); must be finite on (0,1)^d
 *     };
 *
 * (any members, helper functions and constants it needs; no #include of host headers; p points to the
 * n_params doubles given here, read-only).  The library compiles it with NVRTC for sm_100a into the SAME fused
 * iterate kernel the built-in integrands use (streaming form: x is consumed dimension by dimension, nothing per
 * event is stored) for this grid's dim, in both precisions, and selects it with integrand_id = VEGAS_F_USER in
 * vegas_iterate / vegas_accumulate / vegas_integrate.  With precision VEGAS_FP32 the sampling map, the Jacobian and
 * v = f*J are fp32 (C11) around the same user code: dim() receives the fp32 x widened to double, finish()'s value is
 * rounded to fp32 (it must then lie in the fp32 range).  vegas_set_params(g, VEGAS_F_USER, ...) replaces the
 * parameters without recompiling.  log (host, may be NULL) receives the NUL-terminated compiler log, truncated
 * to log_bytes.  Needs libnvrtc.so.12 at run time (loaded on first use).
 * Errors: VEGAS_EINVAL (NULL source, n_params out of range, compile error -> see log; dim * n_bins too large for
 * the fused kernel's shared memory), VEGAS_ECUDA (NVRTC or the CUDA runtime unavailable / module load failed).
 * vegas_debug_sample() does not take VEGAS_F_USER. */
int vegas_set_user_integrand(vegas_grid* g, const char* cuda_source, const double* params_host, int n_params,
                             char* log, size_t log_bytes);

/* Histogram of an observable during the integration ("exporting histograms during integration").
 * If the user integrand's struct also defines
 *         __device__ double observable(const double* p);     // called after finish(), same event
 * and vegas_set_observable(g, lo, hi, n_obs_bins) was called with 1 <= n_obs_bins <= 128, every iteration with
 * VEGAS_F_USER also accumulates  O[k] += v  (v = f*J of the event) for k = floor((observable - lo) / (hi - lo) *
 * n_obs_bins) in [0, n_obs_bins); events outside [lo, hi) are not counted.  vegas_get_observable_hist() copies the n_obs_bins
 * sums of the LAST iteration to the host (divide by n_events and the bin width for dI/dO); one shared-memory add per
 * event in the fused kernel and one global add per bin per CTA per launch, so the last bits depend on the CTA order.
 * n_obs_bins = 0 switches it off.  Errors: VEGAS_EINVAL (hi <= lo, n_obs_bins out of range, nothing to get). */
int vegas_set_observable(vegas_grid* g, double lo, double hi, int n_obs_bins);
int vegas_get_observable_hist(vegas_grid* g, double* obs_hist_host, void* cuda_stream);

/* Host-callback integrands (integrands written "in Fortran, C/C++" reach the paper's library through
 * CFFI, second half).  One iteration like vegas_iterate(), but f is evaluated by a HOST function
 * on batches of points: per batch of at most batch_events events the library samples x on the device (S1-S3), copies
 * x [n][dim] (row-major fp64) to the host, calls fn(x, n, dim, f, user) -- which must fill f[0..n-1] -- copies f back
 * and accumulates S1, S2 and the histogram on the device (S5-S6).  Same sample, same sums as a device integrand with
 * the same f; fp64; this is a convenience path bound by the host function and the PCIe copies, not the hot path.
 * dev_scratch: device memory, 256-byte aligned, caller-owned.  vegas_callback_scratch_bytes(dim, batch_events) bytes
 * (about batch_events * (40 dim + 32)) hold TWO batches: the device samples batch k+1 and copies its points to the host
 * while the host evaluates batch k (one stream; the host waits on events, not on the stream); with half of that the
 * batches are processed strictly one after the other.  The callback runs on the calling thread; it must not call
 * into this grid.  Host staging is page-locked memory owned by the library (2 x batch_events x (dim + 1) doubles).
 * Errors: VEGAS_EINVAL (NULL fn / scratch, n_events < 2, batch_events = 0, scratch too small or misaligned),
 * VEGAS_ECUDA, VEGAS_ENUMERIC (a non-finite f makes the sums non-finite; I, sigma are still written). */
typedef void (*vegas_host_integrand)(const double* x, uint64_t n, int dim, double* f, void* user);
size_t vegas_callback_scratch_bytes(int dim, uint32_t batch_events);
int vegas_iterate_callback(vegas_grid* g, uint64_t n_events, uint32_t batch_events, uint64_t seed, uint32_t iteration,
                           vegas_host_integrand fn, void* user, void* dev_scratch, size_t scratch_bytes,
                           void* cuda_stream, double* I, double* sigma, double* hist_host);

/* Inject / read the master grid: edges_host is [dim][n_bins+1] fp64, every row strictly increasing
 * with first element 0 and last element 1 (checked -> VEGAS_EINVAL).  Synchronous on `stream`. */
int vegas_set_edges(vegas_grid* g, const double* edges_host, void* cuda_stream);
int vegas_get_edges(vegas_grid* g, double* edges_host, void* cuda_stream);
/* Read the histogram [dim][n_bins] left on the device by the last iteration (sum of v^2, C6). */
int vegas_get_hist(vegas_grid* g, double* hist_host, void* cuda_stream);

/* One Vegas iteration (steps S1-S7 of SURVEY.md 8(a)): n_events events with global indices
 * 0..n_events-1 of iteration `iteration`, processed in launches of at most chunk_events events
 * (0 = a single launch; the result does not depend on it beyond summation order, every event's RNG
 * counter is its global index, C2; the fast path additionally splits a launch at multiples of 2^32 of
 * the event index).  Writes I and sigma (host doubles, C7) and, if hist_host is not
 * NULL, the histogram [dim][n_bins] (host); the histogram also stays on the device for
 * vegas_refine(g, NULL, ...).  Synchronises `stream` before returning.
 * Errors: VEGAS_EINVAL (n_events < 2, unknown id/precision, params not set), VEGAS_ECUDA,
 * VEGAS_ENUMERIC (I, sigma are still written). */
int vegas_iterate(vegas_grid* g, uint64_t n_events, uint64_t chunk_events, uint64_t seed,
                  uint32_t iteration, int integrand_id, int precision, void* cuda_stream, double* I,
                  double* sigma, double* hist_host);

/* The same iteration split into its asynchronous pieces, for sharding events over several GPUs /
 * processes: every rank calls begin, accumulate on ITS event range
 * [first_event, first_event+count), reduce; the ranks then sum the vegas_totals_count() doubles at
 * vegas_totals_device() (one all-reduce); every rank calls finalize with the GLOBAL event count.
 * begin/accumulate/reduce only enqueue work; finalize synchronises like vegas_iterate. */
int vegas_begin_iteration(vegas_grid* g, void* cuda_stream);
int vegas_accumulate(vegas_grid* g, uint64_t first_event, uint64_t count, uint64_t chunk_events,
                     uint64_t seed, uint32_t iteration, int integrand_id, int precision,
                     void* cuda_stream);
int vegas_reduce(vegas_grid* g, void* cuda_stream);
int vegas_finalize(vegas_grid* g, uint64_t n_events_total, void* cuda_stream, double* I, double* sigma,
                   double* hist_host);
/* vegas_finalize and vegas_refine in one call, for the sharded iteration: after the ranks' all-reduce of the totals,
 * enqueue S7 (I, sigma) and, if alpha >= 0, S8 (refinement from the summed histogram; alpha < 0: none) back to back on
 * `stream`, then read { I, sigma, status } (and the histogram, if hist_host is not NULL) with ONE synchronisation -- a
 * sharded iteration costs one host synchronisation like a single-GPU one, instead of one for finalize and one for refine
 * (the multi-GPU runs; what matters for the small configs, whose iteration is tens of
 * microseconds).  Every rank calls it with the GLOBAL event count and the same alpha, and ends with the same grid.
 * Errors: as vegas_finalize and vegas_refine (VEGAS_ENUMERIC: non-finite sums, or a dimension kept its grid). */
int vegas_finish_sharded(vegas_grid* g, uint64_t n_events_total, double alpha, void* cuda_stream, double* I, double* sigma,
                         double* hist_host);
/* Device address / length (in doubles) of the reduced totals { S1_hi, S1_lo, S2_hi, S2_lo,
 * H[dim][n_bins] } that vegas_reduce() writes and vegas_finalize() / vegas_refine() read. */
void* vegas_totals_device(vegas_grid* g);
size_t vegas_totals_count(const vegas_grid* g);

/* One iteration for callers that have no device memory to give beyond the data itself (steps S1-S7 as vegas_iterate).
 *
 * Who this is for.  Every other compute call needs a vegas_grid, and a vegas_grid needs a device workspace that the caller
 * allocates.  Some callers cannot do that.  The typical one is code running as an op or callback inside a framework that
 * owns the GPU's memory -- a TensorFlow custom op (the paper's library lives on TensorFlow) or a PyTorch
 * extension that gets handed its input and output buffers and nothing else: the framework's pool has usually claimed most
 * of the card already, so a cudaMalloc from inside the op fails or eats into someone else's budget, and it stalls every
 * stream on the device while it runs.  Others are a service loop that must not see that device-wide stall on its latency
 * path, and a process that was given a fixed slice of device memory at start-up with no headroom for a workspace whose
 * size depends on the grid shape.  For them this call needs only what they already hold: the grid edges going in, the
 * result and the histogram coming out.  It calls no cudaMalloc / cudaFree / cudaMallocHost and no library routine that
 * allocates; the per-CTA partial sums and the reduced totals that the kernels need as working memory live in an array
 * compiled into the library.
 *
 * The price of that array.  It is 2 642 976 bytes (161 rows of 4 + VEGAS_STATIC_MAX_ENTRIES doubles), it exists once per
 * GPU in every process that loads this library, from the moment the library's device code is loaded on that GPU until the
 * process exits, whether or not this call is ever used.  Shapes with dim * n_bins > VEGAS_STATIC_MAX_ENTRIES (2048: e.g.
 * 20 x 100, 16 x 128, 8 x 256; all five BASELINE.json configs fit) are refused with VEGAS_ELIMIT before anything is
 * launched -- use a vegas_grid for those.
 *
 * Arguments.  edges_dev: DEVICE, [dim][n_bins+1] fp64, every row increasing from 0 to 1 (read only; not checked -- it is
 * on the device).  params_host / n_params: HOST, the integrand's parameter array exactly as vegas_set_params() takes it
 * (VEGAS_F_USER is not served: compiling one allocates).  result_dev: DEVICE, 3 doubles, receives { I, sigma, status }
 * with status 0.0 or -3.0 (VEGAS_ENUMERIC: the sums came out non-finite).  hist_dev: DEVICE, [dim][n_bins] fp64, receives
 * the histogram of v^2 (C6); may be NULL.  Both outputs are caller-owned and fully overwritten.  The call runs on the
 * CURRENT device and only enqueues work on `cuda_stream`: the outputs are valid once the stream has reached that point.
 * Same sample as vegas_iterate with the same (seed, iteration) (C2); it runs the library's generic fused kernel in one
 * launch plus the fixed-order reduction, so I, sigma and H agree with vegas_iterate to rounding (summation order), and
 * repeated calls with the same arguments give the same bits.
 *
 * First call on each GPU.  It looks up the device address of the built-in array and the device's limits and keeps them
 * for later calls (guarded by a lock).  Make that first call at start-up, outside of any stream capture.
 *
 * Sharing.  All calls on one GPU -- from any thread, on any stream -- use the SAME array, and it still holds whatever
 * the previous call left there.  Each call therefore zeroes, in stream order, the rows it is about to use before its
 * kernels run.  Two calls that can execute at the same time on the GPU (different streams without an event between them,
 * or two host threads) overwrite each other's partial sums and both results are garbage: keep all calls on one stream, or
 * order them with events.  Calls that follow each other on one stream are safe; no host synchronisation is needed.
 *
 * Errors: VEGAS_EINVAL (NULL edges_dev / result_dev, n_events < 2, bad shape, id, precision or parameters -- the same
 * rules as vegas_set_params / vegas_iterate), VEGAS_ELIMIT (see above), VEGAS_ECUDA (no device, launch failure). */
#define VEGAS_STATIC_MAX_ENTRIES 2048
int vegas_iterate_static(const double* edges_dev, int dim, int n_bins, uint64_t n_events, uint64_t seed,
                         uint32_t iteration, int integrand_id, const double* params_host, int n_params, int precision,
                         void* cuda_stream, double* result_dev, double* hist_dev);

/* Refine the grid (step S8, reading C8: smooth, normalise, compress with damping alpha, rebin), per
 * dimension, fp64.  hist_host NULL = use the histogram the last iteration left on the device;
 * otherwise [dim][n_bins] fp64 is uploaded first.  Synchronises `stream`.
 * Errors: VEGAS_EINVAL (alpha < 0 or NaN), VEGAS_ECUDA, VEGAS_ENUMERIC (see above). */
int vegas_refine(vegas_grid* g, const double* hist_host, double alpha, void* cuda_stream);

/* n_iter iterations (iteration indices 0..n_iter-1), each followed by a refinement (also the skipped
 * ones; alpha < 0 disables refinement = importance sampling on a fixed grid), then the
 * inverse-variance combination of iterations k >= n_skip (step S9, reading C9):
 * W = sum 1/sigma_k^2, I = sum(I_k/sigma_k^2)/W, sigma = W^-1/2, chi2_dof = sum (I_k-I)^2/sigma_k^2/(K-1);
 * if an included sigma_k is 0: plain mean, sigma = 0.  All launches are enqueued back to back; the
 * stream is synchronised once at the end.  per_iter_host: [n_iter][2] = (I_k, sigma_k) or NULL.
 * Errors: VEGAS_EINVAL (n_iter < 1 or > 4096, n_skip not in [0,n_iter), ...), VEGAS_ECUDA,
 * VEGAS_ENUMERIC (outputs still written). */
int vegas_integrate(vegas_grid* g, int n_iter, int n_skip, uint64_t n_events, uint64_t chunk_events,
                    uint64_t seed, double alpha, int integrand_id, int precision, void* cuda_stream,
                    double* I, double* sigma, double* chi2_dof, double* per_iter_host);

/* The same, continuing a run: the n_iter iterations carry the indices first_iteration .. first_iteration+n_iter-1
 * in the RNG counter (C2) and start from the grid as it stands.  With the grid (vegas_get_edges / vegas_set_edges),
 * the seed and the next iteration index saved, a run is resumed bit for bit: the RNG is counter-based, nothing else
 * is state.  n_skip counts from first_iteration.  vegas_integrate(...) = vegas_integrate_from(g, 0, ...).
 * Additional error: VEGAS_EINVAL if first_iteration + n_iter exceeds 0xFFFFFFFF (reserved, reading C10). */
int vegas_integrate_from(vegas_grid* g, uint32_t first_iteration, int n_iter, int n_skip, uint64_t n_events,
                         uint64_t chunk_events, uint64_t seed, double alpha, int integrand_id, int precision,
                         void* cuda_stream, double* I, double* sigma, double* chi2_dof, double* per_iter_host);

/* Step S9 alone on host arrays (no device work). */
int vegas_combine(int n_iter, int n_skip, const double* I_k, const double* sigma_k, double* I,
                  double* sigma, double* chi2_dof);

/* Parity hook (kernel K4): for events first_event .. first_event+count-1 of `iteration`, run exactly
 * the device functions of the fused kernel and return, to HOST arrays (any may be NULL):
 *   words [count][dim] u32 (C2), bins [count][dim] i32 (C3), x [count][dim] fp64 (C4; fp32 values
 *   widened when precision = 32), fJ [count] fp64 (v = f*J).  dev_scratch: device memory of at least
 *   vegas_debug_scratch_bytes(dim, count) bytes, caller-owned.  Synchronises `stream`. */
size_t vegas_debug_scratch_bytes(int dim, uint32_t count);
int vegas_debug_sample(vegas_grid* g, uint64_t first_event, uint32_t count, uint64_t seed,
                       uint32_t iteration, int integrand_id, int precision, void* dev_scratch,
                       void* cuda_stream, uint32_t* words, int32_t* bins, double* x, double* fJ);

/* Launch shape of the fused kernel.  0 = automatic for any field.  blocks: CTAs per launch (default: one per SM, at
 * most 1024); threads: per CTA, a multiple of 32 up to 1024 -- a REQUEST that each kernel clamps to its own launch bound:
 * the generic kernel runs at most 512 threads, a fast-path kernel at most 12, 16 or 24 warps (384 / 512 / 768 threads)
 * depending on integrand and dimension (automatic = that maximum, or the warp count below it that gives the most
 * histogram copies), and a user integrand's kernel 12 warps.  vegas_get_launch reports the EFFECTIVE shape, which is the
 * only way to know what a call will run with.  The library has two fused kernels
 * (DESIGN.md "Kernels"): the fast path (path 1: compile-time dimension, affine pre-composed table, bank
 * rotation, exclusive-owner histograms; every built-in integrand at every dimension -- Genz discontinuous in fp64 only --
 * and user integrands, when the table plus one histogram copy fit the shared memory)
 * and the generic path (path 0: every built-in integrand, any shape).  table_copies / hist_copies are the
 * bank-interleaved replicas of the grid table / histogram of the GENERIC kernel (powers of two, <= 32);
 * setting either to a non-zero value pins the generic path.  VEGAS_EINVAL if the combination does not fit
 * the device's shared memory.  vegas_get_launch reports what a call with (integrand_id, precision) will use. */
int vegas_set_launch(vegas_grid* g, int blocks, int threads, int table_copies, int hist_copies);
int vegas_get_launch(vegas_grid* g, int integrand_id, int precision, int* path, int* blocks, int* threads,
                     int* table_copies, int* hist_copies, size_t* shared_bytes);

/* Variants of the sampling map (readings C3' and C4'; "how to
 * generate the random numbers" and PAPER.md:88 "number of subdivisions of the grid" are all the paper fixes).  Opt-in, per
 * grid, for every later iterate / accumulate / integrate / debug_sample call:
 *   VEGAS_VARIANT_NONE  the method as vegas_iterate describes it (32 random bits per event and dimension, fp64 table).
 *   VEGAS_VARIANT_U53   C3': 53-bit uniforms from two Philox words per draw.  One Philox block serves two dimensions:
 *                       counter = (j>>1, iteration, e lo, e hi); U = out[2(j&1)] * 2^21 + (out[2(j&1)+1] >> 11);
 *                       P = U * n_bins, bin = P >> 53, r = (P mod 2^53) * 2^-53 in [0,1).  A different sample from the
 *                       same seed; twice the generator work per event.
 *   VEGAS_VARIANT_Q32   C4': the fused kernel's grid table holds the per-bin pair (X_b, Delta_b = X_{b+1} - X_b) rounded
 *                       to fp32 (half the table read); x = X~_b + Delta~_b * r and J = prod n_bins * Delta~_b in fp64.
 *                       The master grid, the histogram and the refinement stay fp64.  The rounded bins do not tile [0,1)
 *                       exactly: a relative bias of up to dim * 2^-24 on I (measured: DESIGN.md section 11).
 * Both are fp64 modes of CONST, GAUSS, GENZ_PRODUCT_PEAK and BW_POLY on the fast path: with a variant set, a call with
 * precision 32, with VEGAS_F_USER or VEGAS_F_GENZ_DISCONTINUOUS, or for a shape that only the generic kernel serves
 * returns VEGAS_EINVAL.  vegas_debug_sample reports
 * the top 32 bits of U in `words` under VEGAS_VARIANT_U53. */
#define VEGAS_VARIANT_NONE 0
#define VEGAS_VARIANT_U53 1
#define VEGAS_VARIANT_Q32 2
int vegas_set_variant(vegas_grid* g, int variant);
int vegas_get_variant(const vegas_grid* g);

const char* vegas_strerror(int code);
/* Text of the last CUDA error seen by a call on this grid ("" if none); valid until the next call. */
const char* vegas_last_cuda_error(const vegas_grid* g);
/* Library version / build string, e.g. "vegas_b200 0.1 sm_100a". */
const char* vegas_version(void);

#ifdef __cplusplus
}
#endif
#endif /* VEGAS_B200_H */
