/*
 * hpsd.h -- C ABI of the B200-native Hermitian PSD-cone projection library.
 *
 * The operation ("computing an eigendecomposition and setting
 * all negative eigenvalues to zero"):
 *
 *     X = V diag(lambda) V^H   ->   P(X) = V diag(max(lambda, 0)) V^H
 *
 * for every Hermitian block of a cone list, on the real-vector encoding vec_R
 * of Eq. (D10), which preserves the trace inner product
 * (PAPER.md:1224-1226).  This is the step u = Pi_C(u~ - v) of each ADMM
 * iteration, Eq. (D33).
 *
 * svec layout (the library's own):
 *   - block b of size n_b starts at double offset sum_{c<b} n_c^2;
 *   - inside a block the LOWER triangle is stored column by column; column j
 *     starts at off(j) = j (2 n - j) and holds
 *       [ X_jj, s Re X_{j+1,j}, s Im X_{j+1,j}, ..., s Re X_{n-1,j}, s Im X_{n-1,j} ],
 *     s = sqrt(2); n^2 doubles per block.
 *
 * Conventions for every entry point
 *   - "device pointer" = plain CUDA device address on the current device;
 *     "host pointer"   = ordinary host memory.  No torch types cross this ABI.
 *   - stream is a cudaStream_t passed as void* (NULL = legacy default stream).
 *   - Calls with device pointers only ENQUEUE work on `stream` and return; they
 *     do not synchronise the host once the library workspace and the plan for
 *     this size list exist (first call with a new size list allocates and may
 *     synchronise; later calls are capturable in a CUDA graph).
 *   - The caller owns every buffer it passes.  The library never frees caller
 *     memory.  in_svec == out_svec (exact aliasing) is allowed; partial overlap
 *     is not.
 *   - Return value: HPSD_OK (0) or a negative HPSD_E* code; never throws.
 *     Numerical trouble (an iteration that did not converge) cannot be
 *     returned synchronously: it sets info_dev[b] != 0 on the device.
 *   - NaN/Inf in the input (the paper is silent): a block that holds a non-finite
 *     value gets an all-NaN output block (with hpsd_admm_step also an all-NaN v
 *     block) and info[b] = 2; the other blocks of the call are unaffected.  Finite
 *     entries whose squares overflow are outside the supported range.
 *   - n_b = 0 blocks are skipped; n_b = 1 gives out = max(in, 0).
 *   - There is no CPU fallback: without a CUDA device every compute call
 *     returns HPSD_ECUDA.
 */
#ifndef HPSD_H
#define HPSD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HPSD_OK          0
#define HPSD_EINVAL     -1   /* bad argument: negative count/size, NULL with non-empty work */
#define HPSD_EWORKSPACE -2   /* caller workspace too small or misaligned (256 B) */
#define HPSD_ECUDA      -3   /* a CUDA runtime call or kernel launch failed */
#define HPSD_EALLOC     -4   /* device or host allocation failed */
#define HPSD_ETOOLARGE  -5   /* hpsd_project_static: n or count beyond the fixed capacity of the static scratch */

/* Library version: major*10000 + minor*100 + patch. */
int hpsd_version(void);

/* Static string for a return code. */
const char *hpsd_strerror(int code);

/* Projection of a cone list (Eq. D33).
 *   n_blocks  number of Hermitian blocks (>= 0)
 *   sizes     HOST array, sizes[b] = n_b >= 0
 *   in_svec   DEVICE pointer, sum_b n_b^2 doubles, layout above (read only)
 *   out_svec  DEVICE pointer, same length (may equal in_svec)
 *   stream    cudaStream_t
 * Uses a library-owned, per-device workspace that grows on demand and a cached plan per size list.  Calls on
 * different streams (or from different host threads) are safe: they are ordered on the shared workspace with an
 * event, i.e. they serialise; use one hpsd_plan (or hpsd_project_ws with a workspace) per stream for concurrency.
 * A call captured by the caller into a CUDA graph is the caller's to order against other users of the library. */
int hpsd_project(int n_blocks, const int *sizes,
                 const double *in_svec, double *out_svec, void *stream);

/* Bytes of workspace hpsd_project_ws needs for this size list. */
int hpsd_workspace_size(int n_blocks, const int *sizes, size_t *bytes);

/* Same as hpsd_project with a caller-owned DEVICE workspace `ws` of at least
 * hpsd_workspace_size() bytes, 256-byte aligned (e.g. a torch tensor), and an
 * optional DEVICE array info_dev[n_blocks] (may be NULL) that receives 0 per
 * block, or a positive code if an iteration in that block did not converge. */
int hpsd_project_ws(int n_blocks, const int *sizes,
                    const double *in_svec, double *out_svec,
                    void *ws, size_t ws_bytes, int *info_dev, void *stream);

/* Explicit plan handle: what an ADMM loop keeps across iterations.  A plan owns the routing of
 * its size list (size class per block, svec offsets, lanes), the options in force when it was created (later
 * hpsd_set_option calls do not touch it), its own DEVICE workspace, the per-block status words and the CUDA graphs
 * captured for the buffers it has been run with.  hpsd_plan_create allocates and may synchronise; the execute calls
 * only enqueue on `stream` (first call with a new set of buffers: plain launches; second: capture; later: one
 * cudaGraphLaunch), may be captured by the caller, and never run route or size computations on the host.
 * Calls on ONE plan from different streams are ordered with an event (they share its workspace); different plans
 * are independent and may run concurrently.  Destroying a plan synchronises the device.
 *   hpsd_plan_project    out = Pi_C(in)                         (Eq. D33)
 *   hpsd_plan_admm_step  u = Pi_C(u~ - v), v <- v - u~ + u     (Eqs. D33-D34)
 *   hpsd_plan_info       DEVICE pointer to the n_blocks status words of the last execution (0, 1/4 = an iteration
 *                        did not converge, 2 = non-finite input) and the plan's workspace size in bytes
 * All pointers passed to the execute calls are DEVICE pointers with the layout and aliasing rules of hpsd_project. */
typedef struct hpsd_plan hpsd_plan;
int hpsd_plan_create(int n_blocks, const int *sizes, hpsd_plan **plan);
int hpsd_plan_destroy(hpsd_plan *plan);
int hpsd_plan_project(hpsd_plan *plan, const double *in_svec, double *out_svec, void *stream);
int hpsd_plan_admm_step(hpsd_plan *plan, const double *utilde, double *v, double *u, void *stream);
int hpsd_plan_info(hpsd_plan *plan, const int **info_dev, size_t *workspace_bytes);
/* Copies the n_blocks status words to HOST memory on `stream` and synchronises that stream. */
int hpsd_plan_read_info(hpsd_plan *plan, int *info_host, void *stream);
/* Measurement aid: HOST microseconds per hpsd_plan_project call, averaged over `reps` back-to-back calls on `stream`
 * (enqueue only, the stream is synchronised before and after the loop; the plan's CUDA graph is warm). */
int hpsd_plan_host_overhead(hpsd_plan *plan, const double *in_svec, double *out_svec, int reps, void *stream, double *enqueue_us);

/* complex64 STORAGE ("a fixed number of initial iterations is performed in single
 * precision", complex64 column of Table III).  The same operations as hpsd_project, hpsd_admm_step,
 * hpsd_plan_project and hpsd_plan_admm_step on svecs stored as FP32: same layout (n^2 floats per block, sqrt(2)-scaled
 * lower triangle), DEVICE pointers, same aliasing rules, same plans, routes and options, same NaN contract.  Every load
 * widens to FP64, the path in between is the FP64 one, every store rounds to nearest FP32: the result is the FP32 rounding
 * of the FP64 projection of the FP32 input, i.e. at least as accurate as a complex64 eigensolver (relative error 2^-24 per
 * entry against n 2^-24 norm-wise), at the FP64 path's speed with half the svec traffic; FP32 ARITHMETIC is not built
 * (DESIGN.md §10).  The single -> double switch of PAPER.md:1544 is the caller's: run the first iterations through the
 * _c64 calls, widen the iterate once (hpsd_svec_convert), continue with the FP64 calls on the same plan. */
int hpsd_project_c64(int n_blocks, const int *sizes, const float *in_svec, float *out_svec, void *stream);
int hpsd_admm_step_c64(int n_blocks, const int *sizes, const float *utilde, float *v, float *u, void *stream);
int hpsd_plan_project_c64(hpsd_plan *plan, const float *in_svec, float *out_svec, void *stream);
int hpsd_plan_admm_step_c64(hpsd_plan *plan, const float *utilde, float *v, float *u, void *stream);
/* dst[i] = src[i] for count svec entries between the two storage types (to_f32 != 0: double -> float, else float ->
 * double); DEVICE pointers, no overlap, enqueue-only. */
int hpsd_svec_convert(size_t count, const void *src, void *dst, int to_f32, void *stream);

/* Allocation-free exact projection (same operation and svec layout as hpsd_project) of `count` blocks of
 * ONE size n, stored back to back: block i at in_svec + i n^2.  For callers that cannot call cudaMalloc (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid it): the call makes no cudaMalloc / cudaFree and calls no
 * allocating library routine, on the first call or any later one.  Its scratch is a fixed array of
 * HPSD_STATIC_SCRATCH_BYTES in the library's device image, held by every GPU that loads the library until exit.
 *   limits     2 <= n <= HPSD_STATIC_MAX_N and 0 <= count <= HPSD_STATIC_MAX_COUNT; beyond either: HPSD_ETOOLARGE,
 *              nothing enqueued.  n < 2, count < 0, NULL svec with count > 0: HPSD_EINVAL.
 *   in_svec    DEVICE, count n^2 doubles, read only.   out_svec  DEVICE, same size, may alias in_svec.
 *   info_dev   DEVICE, count ints, or NULL: per-block status as in hpsd_project_ws (0 ok, 2 non-finite input -> NaN block).
 *   stream     enqueue-only on this stream; no synchronisation.
 * Every call shares the one array and finds the previous call's contents there; what must start at zero is cleared by
 * each call on `stream`.  Two calls that overlap on the GPU (different streams without an event between them) RACE on
 * the array: serialise them.  The result equals hpsd_project's to rounding (the route is the batched divide-and-conquer
 * medium path for every n here, where hpsd_project takes the Jacobi kernel for n <= 32). */
#define HPSD_STATIC_MAX_N          83
#define HPSD_STATIC_MAX_COUNT      16
#define HPSD_STATIC_SCRATCH_BYTES  (6u << 20)
int hpsd_project_static(int n, int count, const double *in_svec, double *out_svec, int *info_dev, void *stream);

/* The affine-projection step of the SCS iteration on the device:
 *     z_x = (a_x - A^T a_y) / 2,      z_y = a_y + A z_x,
 * with A x = - sum_mu x_mu F_mu and (A^T Z)_mu = - tr[F_mu Z] (Eq. D3) over the orthonormal
 * product basis F_mu of generalized Gell-Mann matrices (Eq. A10) on A_i (x) A_o (x) B_i (x) B_o, all of
 * local dimension d, restricted to the allowed multi-indices of Eq. (B14) without the all-identity
 * index; A^T A = 1 (D4), so no linear solve is involved.  n = d^4 is the matrix size, m = 2 d^6 - 3 d^4 + 2 d^2 - 1
 * the number of coefficients (column m of Table II).
 *   Basis order (the paper fixes none): sigma_0 = 1/sqrt d; sigma_{1+l} the diagonal elements l = 0..d-2;
 *   then (|j><k| + |k><j|)/sqrt 2 and then -i(|j><k| - |k><j|)/sqrt 2, each over j < k in lexicographic order;
 *   multi-indices (alpha, beta, gamma, delta) in lexicographic order.
 *   x, a_x, z_x: DEVICE vectors of m doubles.  y_svec, a_y, z_y: DEVICE svec vectors (n^2 doubles, layout above) of
 *   Hermitian n x n matrices.  z_x may alias a_x and z_y may alias a_y.  2 <= d <= 9.
 * hpsd_affine_create allocates device tables and workspace (40 n^2 bytes) on the current device and synchronises;
 * the apply / project calls only enqueue on `stream` (one plan serves one stream at a time). */
typedef struct hpsd_affine hpsd_affine;
int hpsd_affine_create(int d, hpsd_affine **plan);
int hpsd_affine_destroy(hpsd_affine *plan);
int hpsd_affine_dims(const hpsd_affine *plan, int *n, int *m);
int hpsd_affine_apply_a(hpsd_affine *plan, const double *x, double *y_svec, void *stream);
int hpsd_affine_apply_at(hpsd_affine *plan, const double *y_svec, double *x, void *stream);
int hpsd_affine_project(hpsd_affine *plan, const double *a_x, const double *a_y, double *z_x, double *z_y, void *stream);

/* Factorisation-free APPROXIMATE projection of ONE Hermitian block ("a
 * composite matrix polynomial constructed solely from matrix-matrix products").  The paper's optimised coefficients
 * are in its ref. [81], which this build does not have; the composite polynomial used is the `iterations`-fold
 * composition of the Newton-Schulz cubic g(t) = (3t - t^3)/2 on X / ||X||_F:
 *     S_0 = X / ||X||_F,   S_{k+1} = (3 S_k - S_k^3) / 2,   out = vec_R((X + X S_K) / 2),
 * i.e. the filter lambda -> lambda (1 + g^K(lambda/||X||_F)) / 2 on the spectrum; the Frobenius error against the exact
 * projection is 1/2 || lambda (1 - |g^K(lambda/||X||_F)|) ||_2 and tends to 0 as K grows (K ~ 1.7 log2(||X||_F / |lambda|) + 6
 * settles an eigenvalue lambda).  2 K + 1 complex n^3 GEMMs on the FP64 tensor pipe; no eigensolver.
 *   in_svec, out_svec: DEVICE svec of n^2 doubles (may alias); library workspace (64 n^2 bytes); enqueue-only. */
int hpsd_project_approx(int n, const double *in_svec, double *out_svec, int iterations, void *stream);

/* One ADMM cone step, Eqs. (D33)-(D34), fused into the projection:
 *     u = Pi_C(u~ - v),      v <- v - u~ + u
 * on the PSD part of the cone.  utilde (read only), v (read and updated in place) and u (written) are DEVICE
 * svec vectors of sum_b n_b^2 doubles; u may alias utilde.  The difference u~ - v is formed while unpacking (S1)
 * and the v update is written by the same epilogue that packs u (S8), so neither costs a pass over memory.
 * Same workspace, stream and error conventions as hpsd_project. */
int hpsd_admm_step(int n_blocks, const int *sizes, const double *utilde, double *v, double *u, void *stream);

/* The same projection through HOST buffers: copies in_host to the device,
 * projects, copies the result back and synchronises `stream` before
 * returning.  This is the end-to-end call bench.py's "e2e" times; the paper
 * pays this host<->device round trip every iteration. */
int hpsd_project_host(int n_blocks, const int *sizes,
                      const double *in_host, double *out_host, void *stream);

/* vec_R, Eq. (D10): lower triangle of a column-major complex
 * FP64 matrix A (DEVICE, interleaved re/im, leading dimension lda >= n, in
 * complex elements) -> svec (DEVICE, n^2 doubles).  Step S8 of SURVEY.md §8(a). */
int hpsd_pack(int n, const void *A, int lda, double *svec, void *stream);

/* mat_R, inverse of (D10): svec (DEVICE) -> full Hermitian column-major complex
 * FP64 matrix A (DEVICE, lda >= n): both triangles written, Im(diag) = 0.
 * Step S1 of SURVEY.md §8(a). */
int hpsd_unpack(int n, const double *svec, void *A, int lda, void *stream);

/* S2+S3 of SURVEY.md §8(a) alone: reduce one Hermitian block (svec, DEVICE) to a
 * REAL symmetric tridiagonal matrix unitarily similar to it: diagonal d (DEVICE,
 * n doubles) and sub-diagonal e (DEVICE, n-1 doubles).  First half of the
 * "eigendecomposition" of PAPER.md:1536; lets tests check the reduction alone. */
int hpsd_tridiagonalize(int n, const double *in_svec, double *d, double *e, void *stream);

/* S2 of SURVEY.md §8(a) alone (two-stage reduction, option "two_stage"): reduce one
 * Hermitian block (svec, DEVICE, n >= 2) to a Hermitian BAND matrix of width
 * b = hpsd_band_width() unitarily similar to it.  band (DEVICE) receives 2b x n
 * complex FP64 elements, column-major with leading dimension 2b: element (i, j),
 * j <= i <= j + b, of the band matrix at band[(i - j) + j * 2b] (rows b+1 .. 2b-1 of
 * every column are zero: room for the bulge of S3).  HPSD_ECUDA when the device
 * cannot launch the 16-CTA cluster the panel factorisation needs. */
int hpsd_reduce_to_band(int n, const double *in_svec, double *band, void *stream);
int hpsd_band_width(void);

/* Eigenvalues of one Hermitian block given as svec (DEVICE), ascending, into
 * lambda (DEVICE, n doubles).  Diagnostic/NEXT-2 entry:
 * lambda_min for the post-processing mix. */
int hpsd_eigvalsh(int n, const double *in_svec, double *lambda, void *stream);

/* Tuning/testing knobs.
 *   "jacobi_max_n" (1..84, default 32): blocks with 2 <= n <= value use the one-CTA
 *       cyclic Jacobi kernel (S9).
 *   "medium_max_n" (0..116, default 116): blocks with jacobi_max_n < n <= value use the
 *       one-CTA Householder + implicit-QL kernel (S10); larger ones the multi-kernel
 *       Householder / divide-and-conquer path.  jacobi_max_n = 1 with medium_max_n = 0
 *       forces every block through the large path (used by the edge-case tests).
 *   "medium_dc" (0/1, default 1): medium blocks with n <= 83 solve their tridiagonal eigenproblems with
 *       the batched device-side divide & conquer (whole group as one virtual problem) instead of the
 *       in-CTA implicit QL.
 *   "cluster_tridiag" (0/1, default 1): blocks whose packed lower triangle fits in the shared memory of one
 *       16-CTA cluster (116 < n <= ~631) are tridiagonalised by the cluster-resident kernel (S1+S2+S3 in one
 *       launch); 0 forces the grid-wide panel kernel.
 *   "overlap_factors" (0/1, default 1): the compact-WY factors of the back-transform (they depend on the
 *       reflectors only) run on an internal side stream next to the divide & conquer; fork and join are events
 *       on the caller's stream, so the call stays asynchronous and capturable.
 *   "large_lanes" (0/1, default 1): two or more blocks of one call whose reduction runs on a single 16-CTA cluster
 *       (sizes up to ~631) are processed next to each other on up to 8 internal lane streams, each with its own part of
 *       the workspace (hpsd_workspace_size accounts for it); fork and join are events on the caller's stream.
 *   "panel_lanes" (0/1, default 1): two or more blocks of one call above the cluster limit (n <= 2600; they take the
 *       grid-wide cooperative panel kernel, which is bound by per-column latency, not by throughput) are dealt to two
 *       lanes: lane 1 runs on an internal stream with 64 CTAs, lane 0 on the caller's stream keeps every SM until its
 *       remaining work equals lane 1's and then continues on the other SMs.  One more scratch area (accounted for by
 *       hpsd_workspace_size); fork and join are events on the caller's stream.
 *   "medium_reroute" (0/1, default 1): a group of at most 32 blocks of one size in 84..116 (the in-CTA QL range), or of
 *       at most 4 blocks of one size in 64..83, goes through the large path (cluster-resident reduction, lanes) instead
 *       of the one-CTA medium kernels (5 and 1 blocks when "large_lanes" is off).
 *   "graph_replay" (0/1, default 1): the second call with the same size list AND the same buffers (an ADMM
 *       loop) is captured into a CUDA graph on an internal stream; that call and the following ones are one
 *       cudaGraphLaunch on the caller's stream (same kernels, same order).  Off while "profile" is on or when the
 *       caller's stream is itself capturing.  Any hpsd_set_option call discards the cached graphs.
 *   "profile" (0/1): record CUDA events on the caller's stream around every stage
 *       of the path (S1..S10) for hpsd_profile_read.  Off by default. */
int hpsd_set_option(const char *name, int value);

/* Stage timers (measurement): number of stages, their names, and the
 * device time in milliseconds each stage took in the LAST hpsd_project* call made with
 * "profile" = 1 (summed over its launches; spans[i] = number of timed spans, may be
 * NULL).  ms and spans are HOST arrays of at least hpsd_profile_stage_count() entries.
 * hpsd_profile_read synchronises on the recorded events. */
int hpsd_profile_stage_count(void);
const char *hpsd_profile_stage_name(int stage);
int hpsd_profile_read(double *ms, int *spans, int n);

/* Number of kernel launches the library issued in the last hpsd_project*
 * call on this thread (bench.py reports it as gpu_launches). */
int hpsd_last_launch_count(void);

/* Release the library-owned workspace and cached plans of the current device. */
int hpsd_release(void);

/* Measurement aid for the FP64 roofline denominator, which
 * MEASURED_PEAKS.json lacks: runs `iters` rounds of independent FP64 FMA
 * chains (kind 0: DFMA; kind 1: DMMA m8n8k4) on every SM on `stream` and
 * writes the flop count of one launch to *flops (HOST).  bench.py times the
 * launch with CUDA events.  Not on the projection path. */
int hpsd_fp64_peak_probe(int kind, int iters, double *flops, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* HPSD_H */
