/* nk.h -- C-ABI of libnk.so: the Nekbone conjugate-gradient hot path on one B200 (sm_100a), fp64.
 *
 * What it computes (citations: "P:n" = /root/reference/PAPER.md line n; "S" = SURVEY.md section;
 * "BJ" = BASELINE.json north_star):
 *   P:225-226, P:290  3-D Poisson problem on E hexahedral spectral elements with (N+1)^3 points
 *                     each, solved by unpreconditioned conjugate gradients, fixed iteration count.
 *   P:314             `ax`: action of the Poisson operator (matrix-free local Laplacian, S 8(c) O3).
 *   P:183-187         `gs`: gather-scatter (direct-stiffness sum QQ^T) over copies of shared nodes.
 *   P:312, Table V    "streaming" (axpy) and "reduction" (dot product) kernels of CG.
 *   BJ                Dirichlet mask; fused axpy+dot; residual history.
 *
 * Layout.  n = N+1, P = n^3, L = E*P.  A "local vector" is L doubles, element-local layout:
 * index l = e*P + i + n*j + n^2*k with i <-> r (fastest), j <-> s, k <-> t.  Copies of a node
 * shared between elements are stored once per touching element.
 *
 * Pointers.  Each argument says HOST or DEVICE.  DEVICE pointers must be 16-byte aligned and are
 * owned by the caller (PyTorch tensors' data_ptr()); nothing passed in is retained except the
 * workspace, which must outlive the context.  `stream` is a cudaStream_t passed as void* (NULL =
 * the legacy default stream).  All work is enqueued on `stream`; only nk_setup, the *_host calls
 * and nk_get_scalars synchronise.  One in-flight call per context; calls on one context must be
 * stream-ordered.
 *
 * Errors.  Every call returns 0 (NK_OK) or a negative NK_ERR_* code; it never throws, aborts or
 * prints.  There is no CPU fallback anywhere: without a CUDA device every compute call returns
 * NK_ERR_CUDA.
 */
#ifndef NK_H
#define NK_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NK_OK              0
#define NK_ERR_ARG        -1   /* null/misaligned pointer, E <= 0, N outside [1,15], niter < 0, L >= 2^31 */
#define NK_ERR_WORKSPACE  -2   /* workspace too small or not 256-byte aligned */
#define NK_ERR_ID         -3   /* negative glo_num */
#define NK_ERR_MASK       -4   /* mask value not exactly 0.0/1.0, or copies of one node disagree */
#define NK_ERR_GEOM       -5   /* Jacobian determinant <= 0 or non-finite at some point */
#define NK_ERR_CUDA       -6   /* CUDA runtime error; nk_last_cuda_error() has the cudaError_t */
#define NK_ERR_ALLOC      -7   /* host allocation failed */
#define NK_ERR_MULT       -8   /* more than 127 distinct node multiplicities (unsupported) */
#define NK_ERR_SIZE       -9   /* nk_dot_static: more entries than its fixed scratch serves (nk_dot_static_max_n) */

#define NK_MAX_ORDER      15

typedef struct nk_ctx nk_ctx;   /* opaque; one per mesh */

/* Upper bound, from (E, N) only, on the DEVICE workspace nk_setup needs (S 8(b)). */
int nk_workspace_bytes(int64_t E, int N, size_t *bytes);

/* Set-up (S 8(a) row a0; "setup on CPU amortised", P:63 derivative matrices depend on N only).
 * Computes the GLL basis for order N, the six geometric factors per point
 *   G_ab = w_i w_j w_k * J * (grad a . grad b),  a,b in {r,s,t}   (S 8(c) O2)
 * on the device, the gather-scatter plan (CSR of local indices grouped by global id), the
 * multiplicity and the inverse-multiplicity weights c.  Synchronises `stream` before returning.
 *   coords   HOST  3 planes x|y|z, each L doubles, local layout
 *   glo_num  HOST  L int64, arbitrary ids >= 0 (need not be contiguous)
 *   mask     HOST  L doubles, each exactly 0.0 (Dirichlet) or 1.0; equal on all copies of a node
 *   workspace DEVICE, caller-owned, 256-byte aligned, >= nk_workspace_bytes(E,N)
 * On error *ctx is NULL.  NK_ERR_GEOM for an inverted / left-handed element. */
int nk_setup(nk_ctx **ctx, int64_t E, int N, const double *coords, const int64_t *glo_num,
             const double *mask, void *workspace, size_t workspace_bytes, void *stream);
void nk_free(nk_ctx *ctx);
/* Host threads the set-up's plan building uses from now on (it runs on all cores by default: a parallel radix
 * sort of (global id, local index), the group walk, the packing); n < 1 restores the default.  Every array
 * nk_setup builds is independent of this number. */
int nk_set_host_threads(int n);
/* Which builder nk_setup uses for the gather-scatter plan from now on: 0 (default) = on the device (ids and mask are
 * uploaded, then a stable radix sort of (global id, local index), scans and per-point kernels; the host only turns
 * the list of distinct multiplicities into the 1/multiplicity table); 1 = on the host cores.  Both produce the same
 * arrays bit for bit.  NK_ERR_ARG for any other value. */
int nk_set_plan_builder(int which);

/* w = A_L u : element-local Laplacian, no gs, no mask (S 8(a) a1).  u, w DEVICE, L; u != w. */
int nk_ax_e(nk_ctx *ctx, const double *u, double *w, void *stream);
/* v = Q Q^T v in place, NO mask (S 8(a) a2).  v DEVICE, L. */
int nk_gs(nk_ctx *ctx, double *v, void *stream);
/* w = M Q Q^T A_L u : ax_e, then gs fused with the Dirichlet mask (S 8(a) a1-a3).  u != w. */
int nk_ax(nk_ctx *ctx, const double *u, double *w, void *stream);
/* out[0] = <a,b>_c = sum_l c_l a_l b_l, c = 1/multiplicity (S 8(a) a4).  a, b, out DEVICE.
 * Deterministic: per-block partials, ordered finish; no floating-point atomics. */
int nk_dot(nk_ctx *ctx, const double *a, const double *b, double *out, void *stream);

/* The weighted dot product WITHOUT a context, a workspace or any allocation, for callers that cannot call cudaMalloc
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
 *   out[0] = sum_{i<n} c_i a_i b_i      (c == NULL: plain dot product; with c = 1/multiplicity it is nk_dot, S 8(a) a4)
 * a, b, c, out DEVICE; a, b, c hold n doubles (16-byte aligned pointers take the vector loads), out one double.
 * Scratch (per-block partial sums and a ticket counter) is a file-scope __device__ array inside the library, about
 * 128 KB that every GPU which loads the library holds until the process exits.  It serves
 * n <= nk_dot_static_max_n() = 2^27 entries; a larger n returns NK_ERR_SIZE and launches nothing.  n = 0 stores 0.
 * Deterministic: a block sums a fixed run of 8192 entries and the last block adds the partials in index order, so the
 * result depends on n and the data only, not on the GPU.  Enqueues one memset node (the counter) and one kernel on
 * `stream`, never synchronises.  Every call shares the one array: calls that OVERLAP on the GPU (different streams
 * with no ordering between them) race on it -- order them; calls on one stream are safe.
 * nk_static_setup() looks the array's device address up for the CURRENT device (cudaGetSymbolAddress; once per
 * device); nk_dot_static does so itself on the first call of a device, so call nk_static_setup beforehand where that
 * first call would fall inside a stream capture.  NK_ERR_ARG: null pointer, n < 0, device ordinal >= 64. */
int nk_static_setup(void);
int64_t nk_dot_static_max_n(void);
int nk_dot_static(const double *a, const double *b, const double *c, int64_t n, double *out, void *stream);

/* Unpreconditioned CG (S 8(c) O8): x0 = 0 (incoming x ignored), r0 = mask o f, recursive
 * residual.  res_hist[k] = sqrt(<r_k, r_k>_c), k = 0..niter (DEVICE, niter+1 doubles).
 * f must be equal on all copies of a node (unchecked).  f, x DEVICE, L.  niter = 0 is legal.
 * Guards: an iteration with rho = 0 or pap = 0 takes alpha = beta = 0 (f = 0 gives x = 0, no NaN).
 * Never synchronises; alpha, beta, rho stay on the device. */
int nk_cg(nk_ctx *ctx, const double *f, double *x, int niter, double *res_hist, void *stream);
/* Same with HOST f, x, res_hist: copies f in, runs nk_cg on workspace buffers, copies x and the
 * history out, synchronises.  Needs extra staging vectors nk_workspace_bytes already counts. */
int nk_cg_host(nk_ctx *ctx, const double *f_host, double *x_host, int niter,
               double *res_hist_host, void *stream);

/* nrhs solves in a row, HOST buffers, pipelined: while solve j runs on `stream`, right-hand side j+1 is copied in and
 * solution j-1 (with its history) copied out on two internal copy streams, through two sets of staging buffers in the
 * workspace.  f_host, x_host, res_hist_host: HOST arrays of nrhs HOST pointers (L, L, niter+1 doubles each; pinned
 * memory is what makes the copies overlap; the same buffer may appear more than once in f_host).  Every solve is
 * exactly nk_cg on its right-hand side: results equal nk_cg_host's bit for bit.  Synchronises before returning. */
int nk_cg_host_batch(nk_ctx *ctx, int nrhs, const double *const *f_host, double *const *x_host, int niter,
                     double *const *res_hist_host, void *stream);

/* Jacobi-preconditioned CG, the original Nekbone's iteration, which the paper's variant omits (P:225,
 * P:290; S 8(f) f-3): z = r / diag, diag = Q Q^T diag(A_L), z = 0 on Dirichlet nodes; rho = <r,z>_c;
 * res_hist[k] = sqrt(<r_k, r_k>_c) as in nk_cg.  Same arguments, guards and residency as nk_cg; the
 * preconditioner is built on the first call and kept in the workspace.  Enqueued launch by launch. */
int nk_pcg(nk_ctx *ctx, const double *f, double *x, int niter, double *res_hist, void *stream);
/* diag (DEVICE out, L) = Q Q^T diag(A_L) in local layout. */
int nk_get_diag(nk_ctx *ctx, double *diag, void *stream);

/* Test entry points for lock-step parity (S 8(c) protocol 2): the CG state lives in the context.
 *   nk_cg_init       r = mask o f, x = 0, p = r, rho = <r,r>_c  (x DEVICE L, caller-owned, kept)
 *   nk_cg_load_state copies r, p (DEVICE, L) into the context and sets rho (x is the caller's)
 *   nk_cg_step       one iteration on (x, ctx r, ctx p); leaves w = ax(p) in the context
 *   nk_cg_get_state  copies ctx r, p and w = M Q Q^T A_L p out (DEVICE, L each; any may be NULL)
 *   nk_get_scalars   HOST out[5] = rho (entering the last step), pap, alpha, rho', beta; synchronises */
int nk_cg_init(nk_ctx *ctx, const double *f, double *x, void *stream);
int nk_cg_load_state(nk_ctx *ctx, const double *r, const double *p, double rho, void *stream);
int nk_cg_step(nk_ctx *ctx, double *x, void *stream);
int nk_cg_get_state(nk_ctx *ctx, double *r, double *p, double *w, void *stream);
int nk_get_scalars(nk_ctx *ctx, double *out5_host, void *stream);

/* ---- Distributed gs / CG over an element partition, one rank per GPU ------------------------------------
 * (PAPER.md:336 lists multi-rank runs as future work; the original Nekbone is MPI,
 * PAPER.md:225.)  Every rank calls nk_setup on ITS OWN elements with GLOBAL node ids; ax_e and the vector kernels
 * are rank-local.  gs needs one neighbour-wise exchange of the partial sums of INTERFACE nodes (nodes another rank
 * holds too), each of the two dot products of an iteration one all-gather of a double; all sums over ranks run
 * in ascending rank order, so every rank holds the same bits and reruns are bitwise equal.  The library builds the
 * plan, enqueues every kernel and drives the sequence; the transfers are the caller's, through a callback.
 *
 *   nk_dist_candidates  HOST: the distinct global ids of the points on element boundaries (i, j or k in {0, N}),
 *                       ascending -- the only nodes another rank can hold.  ids_out needs room for
 *                       E ((N+1)^3 - (N-1)^3) ids.  Needs no context and no device.
 *   nk_dist_setup       builds the plan from ALL ranks' candidate lists (HOST: cand_ids = the lists concatenated in
 *                       rank order, cand_counts[world] their lengths; the caller gathers them, e.g. all_gather).
 *                       glo_num HOST, L, as given to nk_setup.  Plan arrays are device memory the LIBRARY allocates
 *                       (cudaMalloc; the one exception to "the caller owns all device memory"), freed by nk_free.
 *                       Synchronises.  For the halo exchange to overlap ax_e inside nk_dist_cg, put the elements
 *                       that touch another rank's FIRST in the rank's element order (nk_dist_info reports how far
 *                       elements holding an interface node reach).
 *   nk_dist_info        neighbours, doubles in the send (= receive) buffer, interface nodes, leading elements that
 *                       hold interface nodes.  Any out pointer may be NULL.
 *   nk_dist_neighbors   HOST out, one entry per neighbour (ascending rank): its rank, and offset and count of its
 *                       segment in BOTH the send and the receive buffer (the two ranks list the nodes they share in
 *                       ascending global id, so the layouts agree).
 *   nk_dist_set_buffers DEVICE, caller-owned: send, recv (n_exchange doubles each; may be NULL if 0), scalar_send (1),
 *                       scalar_gathered (world).
 *   nk_dist_set_mult    replaces the LOCAL multiplicities by the given global ones (integers 1..127 as doubles, L of
 *                       them: nk_dist_gs of ones): the weights c = 1/mult of every dot product.  Synchronises.
 *   nk_exchange_fn      the caller's transfers, enqueued on `stream` (a cudaStream_t; inside nk_dist_cg the halo
 *                       exchange gets a stream of the library's own).  kind & 1: for every neighbour send its
 *                       segment of `send` and receive its segment of `recv` (one grouped NCCL send/recv);
 *                       kind & 2: all-gather scalar_send[0] into scalar_gathered[0..world).  Return 0 on success.
 *                       Not called where there is nothing to move (one rank; no neighbour).
 *   nk_dist_gs          v <- Q Q^T v over ALL ranks, in place (and the Dirichlet mask if with_mask).
 *   nk_dist_dot         out_dev[0] = <a,b>_c over all ranks.
 *   nk_dist_cg          as nk_cg, over all ranks: per iteration ax_e on the interface elements, their partial sums
 *                       out on a second stream while ax_e runs on the interior elements; all-gather of pap; the
 *                       rank's own gs and mask; totals over the holders; r update; all-gather of rho'; x, p update.
 *                       Three transfers and eight launches per iteration, no host synchronisation.  With one rank
 *                       it IS nk_cg.  Errors as elsewhere; NK_ERR_ARG before nk_dist_setup / nk_dist_set_buffers.
 */
typedef int (*nk_exchange_fn)(void *user, int kind, void *stream);
int nk_dist_candidates(int64_t E, int N, const int64_t *glo_num_host, int64_t *ids_out_host, int64_t *n_out_host);
int nk_dist_setup(nk_ctx *ctx, int rank, int world, const int64_t *glo_num_host, const int64_t *cand_ids_host,
                  const int64_t *cand_counts_host, void *stream);
int nk_dist_info(nk_ctx *ctx, int *n_neighbors, int64_t *n_exchange, int64_t *n_interface_nodes,
                 int64_t *n_interface_elements);
int nk_dist_neighbors(nk_ctx *ctx, int *ranks_host, int64_t *offsets_host, int64_t *counts_host);
int nk_dist_set_buffers(nk_ctx *ctx, double *send_dev, double *recv_dev, double *scalar_send_dev,
                        double *scalar_gathered_dev);
int nk_dist_set_mult(nk_ctx *ctx, const double *mult_dev, void *stream);
int nk_dist_gs(nk_ctx *ctx, double *v, int with_mask, nk_exchange_fn exchange, void *user, void *stream);
int nk_dist_dot(nk_ctx *ctx, const double *a, const double *b, double *out_dev, nk_exchange_fn exchange, void *user,
                void *stream);
int nk_dist_cg(nk_ctx *ctx, const double *f, double *x, int niter, double *res_hist, nk_exchange_fn exchange,
               void *user, void *stream);

/* Options:
 *   "fuse_pap"     1 (default) = pap accumulated inside ax_e through the dot-fusion identity
 *                  <M QQ^T A_L p, p>_c = sum_l (A_L p)_l p_l; 0 = separate weighted dot after gs
 *   "fuse_p"       1 = p = r + beta p folded into the load of the next ax_e; 0 = own kernel;
 *                  2 (default) = the library's choice: 1 at every size (with "defer_x" it moves fewer bytes than the
 *                  separate update and saves a launch)
 *   "fuse_gs"      1 = inside nk_cg the gather-scatter and the mask are folded into the residual
 *                  update: w = M Q Q^T A_L p is only ever read by r -= alpha w, so that kernel streams the
 *                  UNSUMMED ax_e output and sums the copies of every shared node on the fly (in ascending
 *                  local index, as nk_gs: r and x are, entry by entry, what 0 gives for the same alpha; rho'
 *                  adds the same terms in another fixed order, so iterates agree to rounding, not bitwise).
 *                  gs's write-back, its re-read and one launch per iteration are gone.  Needs "fuse_pap" = 1
 *                  (the separate weighted dot reads the summed w); 0 = nk_gs as its own kernel; 2 (default)
 *                  = 1 for meshes of 2^20 local points or more (below, everything sits in L2 and the
 *                  separate kernel is as fast or faster), else 0.
 *   "defer_x"      1 (default) = two iterations share one pass over x, which nothing reads before the solve ends:
 *                  the first of a pair leaves x alone and keeps alpha, the second applies
 *                  x = fma(alpha', p', fma(alpha, p, x)) -- bit for bit what two separate updates give.  The direction
 *                  of the first iteration has to survive the second, so it lives in two vectors: with "fuse_p" and
 *                  "fuse_gs" (the default from 2^20 points on) the second ax_e writes its direction out of place and
 *                  the fused gs update takes both directions (80 B per point and pair instead of 96); without
 *                  "fuse_p" the first forms p' = r + beta p in the second vector (72 instead of 80).  x, r, p are
 *                  complete when nk_cg returns (an odd last iteration is a plain one); 0 = x updated every iteration.
 *   "coop"         1 = nk_cg runs the whole solve as ONE cooperative launch: a persistent CTA per SM does all
 *                  iterations (ax_e with pap and the p update folded in | grid barrier | x, r update with gs
 *                  and the mask folded in, rho' | grid barrier), scalars never leave the chip.  For meshes
 *                  that sit in L2, where launch gaps and kernel tails are most of an iteration.  Orders
 *                  N <= 13; otherwise, and under "profile", the next rule applies.  Sums run in fixed but
 *                  different orders than launch by launch: the two agree to rounding, each is bitwise
 *                  reproducible.  Up to 2^15 points the launch is one 16-CTA thread-block cluster (exchanges through
 *                  distributed shared memory: 1.6-2x the graph replay), above that one CTA per SM with grid
 *                  barriers (1.1-1.3x).  0 = never; 2 (default) = 1 for meshes of up to 2^19 local points
 *                  (slower than the graph replay from about 0.8 M points on).
 *   "graph"        0 = nk_cg enqueues its launches one by one; 1 = records them into a CUDA graph
 *                  (cached per f, x, res_hist, niter; updated in place when the pointers change) and
 *                  replays it; 2 (default) = 1 for meshes of up to 2^24 local points, where launch gaps
 *                  matter, else 0
 *   "pdl"          1 = inside nk_cg, ax_e and the vector kernels are launched as programmatic
 *                  dependents of their predecessor (cudaLaunchAttributeProgrammaticStreamSerialization):
 *                  each runs its prologue early and executes griddepcontrol.wait before the first read of
 *                  anything the predecessor wrote, so results are bit-identical to 0 = plain launches.
 *                  2 = gs as well (on large meshes slower: its gathers need the L1 that ax_e's
 *                  shared-memory carve-out takes away); 3 (default) = 2 for meshes of up to 2^24 local
 *                  points, else 1.  Ignored under "profile".
 *   "profile"      1 = record a CUDA event on `stream` between consecutive launches so that
 *                  nk_get_kernel_times can report device time per kernel class (nk_cg then
 *                  enqueues its launches directly whatever "graph" says)
 * Unknown name or bad value: NK_ERR_ARG. */
int nk_set_option(nk_ctx *ctx, const char *name, int value);
int nk_get_option(nk_ctx *ctx, const char *name, int *value);

/* Introspection. */
int nk_get_sizes(nk_ctx *ctx, int64_t *n_local, int64_t *n_unique, int64_t *n_shared_unique,
                 int64_t *n_masked_unique);
/* gs plan sizes: CSR rows, listed local copies, rows that are summed (shared, unmasked). */
int nk_get_gs_sizes(nk_ctx *ctx, int64_t *n_rows, int64_t *n_listed, int64_t *n_sum_rows);
/* What nk_setup did: the plan builder that ran (0 device, 1 host: chosen by nk_set_plan_builder, or the fallback for
 * meshes with more than 8192 nodes of more than 4096 copies each), wall seconds of the plan part (uploads of ids and
 * mask included) and of the whole call.  Any pointer may be NULL. */
int nk_get_setup_info(nk_ctx *ctx, int *plan_builder, double *plan_seconds, double *total_seconds);
/* Where one array of the gather-scatter plan lives inside the caller's workspace (DEVICE pointer, bytes in use):
 * which = 0 per-point code (multiplicity-table index | 0x80 Dirichlet), 1 CSR row offsets, 2 CSR local indices,
 * 3 packed rows, 4 their chunk descriptors, 5 per-point gather code of the fused update, 6 its rows of three or more
 * copies, 7 the list of those rows, 8 that list cut per block, 9 the 1/multiplicity table, 10 the multiplicity table.
 * For tests and tools (the two plan builders are compared through it); NK_ERR_ARG for another `which`. */
int nk_get_plan_array(nk_ctx *ctx, int which, const void **dev, size_t *bytes);
int nk_get_mult(nk_ctx *ctx, double *mult, void *stream);   /* DEVICE out, L: multiplicity per point */
int nk_get_geom(nk_ctx *ctx, double *G6, void *stream);     /* DEVICE out, planes rr|rs|rt|ss|st|tt, each L */
/* HOST out: D[(N+1)^2] row-major D[i*(N+1)+m] = l_m'(xi_i); xi[N+1]; w[N+1].  Any may be NULL. */
int nk_get_D(nk_ctx *ctx, double *D_host, double *xi_host, double *w_host);
/* Device time per kernel class since the last call, measured with CUDA events on the launching
 * stream while the "profile" option is 1 (S 8(d): per-kernel time inside the timed region).
 * HOST out: ms[6], count[6], classes NK_K_*: 0 ax_e (with whatever is fused into it), 1 gs(+mask),
 * 2 dot, 3 the residual update with rtr (update_r; update x,r on the fuse_p path), 4 the direction
 * update (x and p, or the pending direction update at the end of a solve on the fuse_p path), 5 cg init.  Synchronises `stream`; resets
 * the record. */
#define NK_K_CLASSES 6
int nk_get_kernel_times(nk_ctx *ctx, double *ms_host, int64_t *count_host, void *stream);
/* How ax_e is scheduled (for tests and reports): the persistent kernel works on batches of
 * nk_ax_batch_elements(N) elements (a compile-time constant per order; NK_ERR_ARG for N outside [1,15]);
 * nk_get_ax_launch gives that number, the CTAs one launch uses on this context's device and the number
 * of batches the busiest CTA runs (> 1: the shared-memory ring wraps and its mbarrier phases flip). */
int nk_ax_batch_elements(int N);
int nk_get_ax_launch(nk_ctx *ctx, int *batch_elements, int *ctas, int64_t *max_batches_per_cta);
/* Which way nk_cg runs with the current options on this mesh: path 0 = its kernels enqueued one by one,
 * 1 = the same launches replayed as one CUDA graph, 2 = one cooperative launch for the whole solve ("coop");
 * pdl_mode (may be NULL) = "pdl" resolved (0, 1 or 2; paths 0 and 1). */
int nk_get_cg_path(nk_ctx *ctx, int *path, int *pdl_mode);
/* Kernel launches enqueued by this context so far (for bench.py's gpu_launches). */
int nk_get_launch_count(nk_ctx *ctx, int64_t *count);

/* The fp64 ceiling of the current device, measured with a DFMA-only microbenchmark (the
 * secondary roofline of ax_e, whose primary bound is HBM): HOST out tflops = 2 flops x DFMA per second at
 * full occupancy, best of 5 runs of about a millisecond; dfma_per_clk_per_sm (may be NULL) = the same rate
 * per SM and per cycle of the device's MAXIMUM SM clock.  Needs no context; allocates 8 bytes for the
 * duration of the call; synchronises. */
int nk_fp64_peak(double *tflops_host, double *dfma_per_clk_per_sm_host, void *stream);

const char *nk_strerror(int code);
int nk_last_cuda_error(void);   /* cudaError_t of the last NK_ERR_CUDA on this thread, else 0 */
const char *nk_version(void);

#ifdef __cplusplus
}
#endif
#endif
