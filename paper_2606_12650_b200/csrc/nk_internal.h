// nk_internal.h -- shared declarations of libnk.so's translation units (product code only;
// nothing here is used by, or taken from, oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/nk.h"

// Scalar block on the device (doubles).  Written only by reduction epilogues.
enum { NK_S_RHO = 0, NK_S_PAP = 1, NK_S_ALPHA = 2, NK_S_RHO_NEW = 3, NK_S_BETA = 4, NK_S_RHO_OLD = 5,
       NK_S_ALPHA_PREV = 6,     // alpha of the first iteration of a pair whose x update is deferred ("defer_x")
       NK_S_COUNT = 8 };

// What the last block of a reduction does with the ordered total (S 8(a) a7).
enum { NK_EPI_STORE = 0,   // out[0] = total
       NK_EPI_RHO0 = 1,    // rho = total; hist[0] = sqrt(total); beta = 0
       NK_EPI_PAP = 2,     // pap = total; alpha = rho/pap (guarded)
       NK_EPI_RHO = 3 };   // rho' = total; hist[k] = sqrt; beta = rho'/rho (guarded); rho_old = rho; rho = rho'

#define NK_MAX_PARTIALS 65536      // upper bound on blocks of any reducing kernel
#define NK_VEC_THREADS 512         // P: Table V "local group size 512" for streaming kernels
#define NK_CODE_MASKED 0x80u       // bit 7 of the per-point code: Dirichlet node
#define NK_HIST_MAX 8192               // residual-history capacity of nk_cg_host
#define NK_GRAPH_AUTO_MAX_L (1 << 24)   // "graph" = 2: nk_cg replays a CUDA graph up to this many local points
#define NK_COOP_AUTO_MAX_L (1 << 19)     // "coop" = 2: one cooperative launch per solve up to this many local points
                                        // (measured crossover against the graph replay: 0.7 - 0.9 M points, N = 3..11)
#ifndef NK_CLUSTER_AUTO_MAX_L
#define NK_CLUSTER_AUTO_MAX_L (1 << 15)  // within "coop": up to this many points the solve runs on ONE 16-CTA cluster
#endif
#define NK_FUSE_GS_AUTO_MIN_L (1 << 20)  // "fuse_gs" = 2: gs rides in the residual update from this many local points on
#define NK_GS_CHUNK 32768          // rows per gs chunk (128 blocks of 256 threads)
#define NK_CTAB 128                // code & 0x7f indexes ctab[] = 1/multiplicity

// kernel classes of nk_get_kernel_times
enum { NK_K_AX = 0, NK_K_GS = 1, NK_K_DOT = 2, NK_K_UPDATE_XR = 3, NK_K_UPDATE_P = 4, NK_K_INIT = 5, NK_K_COUNT = 6 };
struct nk_prof;     // nk_api.cu
struct nk_dist;     // nk_dist.cu

// Layout of the geometric factors in HBM: G[e][k][c2][t2] as double2, c2 = 0 (rr,rs),
// 1 (rt,ss), 2 (st,tt), t2 = i + n j.  One element is one contiguous 48 P-byte chunk and one k-plane
// of it a contiguous 48 n^2-byte chunk, always 16-byte aligned: the unit a TMA bulk copy moves.
__host__ __device__ __forceinline__ int64_t nk_g_index(int64_t e, int k, int c2, int t2, int n)
{
    return ((e * n + k) * 3 + c2) * (int64_t)(n * n) + t2;
}

struct nk_reduce_ws {
    double *partials;      // NK_MAX_PARTIALS doubles
    unsigned *counter;     // one ticket counter, self-resetting (atomicInc wrap)
    double *scal;          // NK_S_COUNT doubles
    double *raw;           // NULL, or (distributed CG) where the rank-local total goes INSTEAD of the epilogue
};

struct nk_ctx {
    int64_t E, P, L;
    int N, n;
    int device;
    int sm_count;
    // host copies of the basis (long double evaluated, rounded once)
    double D[16 * 16], xi[16], wq[16];
    // workspace carve-up (all DEVICE)
    void *ws;
    size_t ws_bytes;
    double2 *g;                  // geometric factors, 3 L double2, layout nk_g_index(): per element and
                                 // k-plane one contiguous chunk [c2][i + n j] of (rr,rs) (rt,ss) (st,tt)
    double *r, *p, *w;           // CG state, L each (coords staging aliases these during set-up)
    double *hf, *hx;             // staging for nk_cg_host, L each
    double *pc;                  // where the current direction lives: p, except inside a "defer_x" pair on the "fuse_p" path
    double *p2;                  // second direction vector: the deferred x update needs p_k and p_k+1 at once ("defer_x")
    double *hf2, *hx2, *hist2;   // second set: nk_cg_host_batch copies RHS j+1 in and solution j-1 out while solve j runs
    double *dinv;                // Jacobi preconditioner 1 / (Q Q^T diag A_L), 0 on Dirichlet nodes (lazy)
    int have_dinv;
    uint8_t *code;               // L: multiplicity-table index | NK_CODE_MASKED
    int32_t *row_off;            // n_rows + 1
    int32_t *row_idx;            // n_listed local indices, rows in [0,n_sum_rows) are summed,
                                 // rows in [n_sum_rows, n_rows) are masked nodes
    // the summed rows once more, in chunks of NK_GS_CHUNK rows, packed by length inside a chunk (2, 4, 8
    // copies: faces, edges, corners of a conforming hex mesh): a thread fetches its indices with one
    // vector load and no offset lookup, and a chunk stays in one neighbourhood of memory
    int32_t *pk, *gs_desc;
    // gs folded into the residual update (nk_vec.cu, "fuse_gs"): per local point l
    //   nbr[l] == l   its node has no other copy (or only masked ones): the value stands
    //   nbr[l] >= 0   the ONE other copy of a node of multiplicity 2 (faces: 95 % of all shared points)
    //   nbr[l] == -1  Dirichlet node: the sum is replaced by 0
    //   nbr[l] <= -2  all copies of the node (edges, corners, irregular meshes) are listed in gx: with
    //                 p = -nbr[l]-2, gx[4p-1] = their number and gx[4p ..] their local indices, ascending
    //                 (16-byte aligned so that the first eight come with two vector loads)
    int32_t *nbr, *gx, *gx_rows;   // gx_rows[k] = p of the k-th such node (one thread each in the fused kernel)
    int32_t *gx_blk;               // nk_vec_blocks(L/2) + 1 ints: block b of the fused kernel takes nodes [gx_blk[b], gx_blk[b+1])
    int64_t n_gx_rows;
    int64_t n_gs_chunks;
    int64_t n_pk;                // ints of pk in use
    int plan_builder;            // who built the plan: 0 device (nk_plan.cu), 1 host (nk_setup.cu)
    double setup_plan_s, setup_total_s;   // wall time of the plan part and of all of nk_setup
    double *ctab;                // NK_CTAB doubles: 1/multiplicity
    double *mtab;                // NK_CTAB doubles: multiplicity
    double *hist;                // NK_HIST_MAX doubles (nk_cg_host)
    double *res_dummy;           // 1 double (history sink for nk_cg_step)
    int *errflag;                // geometry error flag
    unsigned *coop_bar;          // grid-barrier counter of the cooperative solve (nk_ax_tma.cu cg_coop_kernel)
    int coop_ok;                 // the device supports cooperative launches
    int cluster_ok;              // ... and has placed a 16-CTA cluster of the solve kernel so far (cleared on the first failure)
    nk_reduce_ws red;
    // sizes
    int64_t n_unique, n_shared_unique, n_masked_unique;
    int64_t n_rows, n_listed, n_sum_rows, n_sum_listed;
    // options / state
    int opt_fuse_pap, opt_fuse_p, opt_fuse_gs, opt_coop, opt_graph, opt_profile, opt_pdl, opt_defer_x;
    int pdl_now;                 // nk_pdl_mode while nk_cg enqueues its loop (every kernel there waits), else 0
    int p_pending;               // 1: p = r + beta p has not been applied yet (fuse_p)
    int w_unsummed;              // 1: ctx w holds the unsummed ax_e output of the last iteration (fuse_gs)
    int64_t launches;
    // per-kernel-class device timing ("profile" option): chained events, interval i = kernel class cls[i]
    nk_prof *prof;
    // distributed gs / CG (nk_dist.cu; S 8(e), 8(f) f-4): the interface plan, library-owned
    struct nk_dist *dist;
    int dist_mult;               // 1: the weights c = 1/multiplicity are GLOBAL (nk_dist_set_mult); rank-local shortcuts are off
    // cached graph for nk_cg
    struct graph_slot {
        cudaGraphExec_t exec;
        const double *f; double *x; double *hist; int niter; int key;
        unsigned long long stamp;                    // last use (the older slot is replaced)
    } graph[2];                                      // two: nk_cg_host_batch alternates between two sets of buffers
    unsigned long long graph_clock;
    // nk_cg_host_batch: copy streams and events, created on first use
    cudaStream_t copy_in, copy_out;
    cudaEvent_t ev_f[2], ev_solve[2], ev_out[2], ev_start;
    int batch_ready;
};
// "pdl" resolved: 0 = plain launches, 1 = ax_e and the vector kernels are programmatic dependents, 2 = gs too.
// gs as a dependent saves a launch gap where gaps matter (config 1: -5 % per solve) and costs 95 us at
// config 5 (its gathers land on SMs whose L1 is still carved out for ax_e): auto = 2 up to 2^24 points.
static inline int nk_pdl_mode(const nk_ctx *c) { return c->opt_pdl == 3 ? (c->L <= NK_GRAPH_AUTO_MAX_L ? 2 : 1) : c->opt_pdl; }

// Programmatic dependent launch (PDL): a kernel launched with `pdl` may start while its predecessor on
// the stream is still draining; it runs its prologue (shared tables, mbarrier set-up, the first TMA
// requests for the STATIC geometric factors) and then waits (nk_pdl_wait) before it touches anything the
// predecessor wrote.  Without the attribute the two device calls are no-ops.
#ifdef __CUDACC__
__device__ __forceinline__ void nk_pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void nk_pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
template <typename... KArgs, typename... Args>
inline cudaError_t nk_launch(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, int pdl,
                             Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
#endif

// Grid of the streaming kernels (nk_vec.cu) and of the row cut nk_setup makes for the fused gs (gx_blk): at least two
// blocks per SM when there is work for them, then 8 pairs per thread (fewer, fatter blocks: less reduction tail on
// mid-size meshes; config 3: 12.4 -> 11.7 ms per solve), capped at 4 resident blocks/SM x 4 waves.
// Fixed grid => fixed partial sums => run-to-run bitwise reproducible.
static inline int nk_vec_blocks(int sm_count, int64_t pairs)
{
    const int64_t one = (pairs + NK_VEC_THREADS - 1) / NK_VEC_THREADS;
    const int64_t floor2 = (int64_t)sm_count * 2, cap = (int64_t)sm_count * 4 * 4;
    int64_t want = (pairs + NK_VEC_THREADS * 8 - 1) / (NK_VEC_THREADS * 8);
    const int64_t lo = one < floor2 ? one : floor2;
    if (want < lo) want = lo;
    if (want > cap) want = cap;
    if (want < 1) want = 1;
    return (int)want;
}

// The fused gs + residual update (nk_vec.cu gs_update_kernel) has its own block geometry: NK_GSU_THREADS threads,
// NK_GSU_MINB resident blocks per SM, NK_GSU_WAVES chunks per resident slot on large meshes.
#ifndef NK_GSU_THREADS
#define NK_GSU_THREADS 512
#endif
#ifndef NK_GSU_MINB
#define NK_GSU_MINB 2
#endif
#ifndef NK_GSU_WAVES
#define NK_GSU_WAVES 8
#endif
static inline int nk_gsu_blocks(int sm_count, int64_t pairs)
{
    const int64_t one = (pairs + NK_GSU_THREADS - 1) / NK_GSU_THREADS;
    const int64_t floor2 = (int64_t)sm_count * 2, cap = (int64_t)sm_count * NK_GSU_MINB * NK_GSU_WAVES;
    int64_t want = (pairs + NK_GSU_THREADS * 8 - 1) / (NK_GSU_THREADS * 8);
    const int64_t lo = one < floor2 ? one : floor2;
    if (want < lo) want = lo;
    if (want > cap) want = cap;
    if (want < 1) want = 1;
    return (int)want;
}

// ---- kernels' host launchers (each returns a cudaError_t from the launch) -----------------------
// nk_dist.cu
// nk_plan.cu: the gather-scatter plan built on the device (nk_setup.cu falls back to its host builder on NK_PLAN_FALLBACK:
// more than 8192 groups longer than 4096 copies).  ctab / mtab: NK_CTAB doubles each, host, filled here.
#define NK_PLAN_FALLBACK (-1000)
int nk_plan_device(nk_ctx *c, const int64_t *glo_num, const double *mask, double *ctab, double *mtab, cudaStream_t st);
void nk_dist_release(nk_ctx *c);              // frees the distributed plan (nk_free)
// nk_basis.cpp
void nk_host_basis(int N, double *xi, double *w, double *D);
void nk_host_basis_dd(int N, double *xi, double *w, double *D, double *Dlo);   // D = D + Dlo (long double split)
// nk_ax_tma.cu : w = A_L u (TMA-pipelined persistent kernel).  If r_in != NULL: u := r_in + beta*u is applied
// first and written back to u.  If dot: sum_l u_l w_l is reduced with epilogue NK_EPI_PAP.
cudaError_t nk_launch_ax_tma(nk_ctx *c, double *u_rw, const double *u_ro, const double *r_in, double *w,
                             int dot, cudaStream_t st);
// the same on elements [e_begin, e_begin + e_count) only (distributed path: interface elements first, then the rest)
cudaError_t nk_launch_ax_tma_range(nk_ctx *c, double *u_rw, const double *u_ro, const double *r_in, double *w, int dot,
                                   int64_t e_begin, int64_t e_count, cudaStream_t st);
cudaError_t nk_upload_D_tables_tma(void);
int nk_ax_tma_epb(int N);
int nk_coop_supported(int N);
// the whole CG solve as one cooperative launch (cg_coop_kernel): x, hist as nk_cg; leaves r, p, the unsummed w and
// the scalars of the last iteration in the context
cudaError_t nk_launch_cg_coop(nk_ctx *c, const double *f, double *x, int niter, double *hist, cudaStream_t st);                       // elements per batch of order N, 0 if N is out of range
// nk_geom.cu
cudaError_t nk_launch_geom(nk_ctx *c, const double *coords_dev, const double *D_dev, const double *Dlo_dev,
                           const double *wq_dev, cudaStream_t st);
cudaError_t nk_launch_get_geom(nk_ctx *c, double *G6, cudaStream_t st);
// nk_gs.cu
cudaError_t nk_launch_gs(nk_ctx *c, double *v, int with_mask, cudaStream_t st);
// nk_vec.cu
cudaError_t nk_launch_dot(nk_ctx *c, const double *a, const double *b, double *out, int epi, cudaStream_t st);
cudaError_t nk_launch_cg_init(nk_ctx *c, const double *f, double *x, double *hist, cudaStream_t st);
// gs != 0: w is the UNSUMMED ax_e output and the copies of shared nodes are summed on the fly (r -= alpha M Q Q^T w
// without gs ever writing w back): r, x entry by entry as nk_launch_gs + gs == 0, rho' summed in another fixed order
cudaError_t nk_launch_update_xr(nk_ctx *c, double *x, double *hist_k, int gs, cudaStream_t st);
cudaError_t nk_launch_update_p(nk_ctx *c, cudaStream_t st);
cudaError_t nk_launch_update_r(nk_ctx *c, double *hist_k, int gs, cudaStream_t st);     // r -= alpha w, rho'
cudaError_t nk_launch_update_px(nk_ctx *c, double *x, cudaStream_t st);         // x += alpha p; p = r + beta p
cudaError_t nk_launch_update_r_first(nk_ctx *c, double *hist_k, cudaStream_t st);          // fused gs update, alpha kept
cudaError_t nk_launch_update_xxr(nk_ctx *c, double *x, const double *pa, const double *pb, double *hist_k, cudaStream_t st);
cudaError_t nk_launch_update_p2(nk_ctx *c, cudaStream_t st);                    // p2 = r + beta p; alpha kept for the next one
cudaError_t nk_launch_update_pxx(nk_ctx *c, double *x, cudaStream_t st);        // x += alpha' p + alpha p2; p = r + beta p2
cudaError_t nk_launch_get_mult(nk_ctx *c, double *mult, cudaStream_t st);
// preconditioned CG
cudaError_t nk_launch_diag(nk_ctx *c, double *diag, cudaStream_t st);          // nk_geom.cu: diag(A_L), local
cudaError_t nk_launch_invert_diag(nk_ctx *c, double *d, cudaStream_t st);      // d = masked ? 0 : 1/d
cudaError_t nk_launch_pcg_init(nk_ctx *c, const double *f, double *x, double *hist, cudaStream_t st);
cudaError_t nk_launch_update_xrz(nk_ctx *c, double *x, double *hist_k, cudaStream_t st);
cudaError_t nk_launch_update_pz(nk_ctx *c, double *x, cudaStream_t st);   // x += alpha p; p = dinv r + beta p
