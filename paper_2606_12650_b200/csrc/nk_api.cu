// nk_api.cu -- the C-ABI of include/nk.h: argument checks, context, set-up (host side of the
// gather-scatter plan), the CG driver.  Every numerical step runs in the kernels of nk_ax_tma.cu,
// nk_gs.cu, nk_vec.cu, nk_geom.cu; nothing here computes on vectors and there is no CPU fallback.
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "nk_host.h"

namespace {
thread_local int t_last_cuda = 0;
}  // namespace

// "profile" option: one cudaEvent between consecutive launches on the caller's stream; the
// interval ending at event i is the device time of the launch of class cls[i] (-1: not a kernel).
struct nk_prof {
    std::vector<cudaEvent_t> ev;
    std::vector<int> cls;
    size_t used = 0;
    ~nk_prof() { for (cudaEvent_t e : ev) cudaEventDestroy(e); }
};

namespace {
cudaError_t prof_mark(nk_ctx *c, int cls, cudaStream_t st)
{
    if (!c->opt_profile) return cudaSuccess;
    if (!c->prof) c->prof = new nk_prof();
    nk_prof *p = c->prof;
    if (p->used == p->ev.size()) {
        cudaEvent_t e;
        cudaError_t rc = cudaEventCreate(&e);
        if (rc != cudaSuccess) return rc;
        p->ev.push_back(e);
        p->cls.push_back(-1);
    }
    p->cls[p->used] = cls;
    return cudaEventRecord(p->ev[p->used++], st);
}
#define NK_LAUNCH(cls, call)                                          \
    do {                                                              \
        if ((e = (call)) != cudaSuccess) return e;                    \
        if ((e = prof_mark(c, (cls), st)) != cudaSuccess) return e;   \
    } while (0)
}  // namespace

void nk_set_last_cuda(int e) { t_last_cuda = e; }

extern "C" {

const char *nk_strerror(int code)
{
    switch (code) {
        case NK_OK: return "ok";
        case NK_ERR_ARG: return "invalid argument";
        case NK_ERR_WORKSPACE: return "workspace too small or misaligned";
        case NK_ERR_ID: return "negative global id";
        case NK_ERR_MASK: return "mask not 0/1 or inconsistent between copies of a node";
        case NK_ERR_GEOM: return "non-positive or non-finite Jacobian";
        case NK_ERR_CUDA: return t_last_cuda ? cudaGetErrorString((cudaError_t)t_last_cuda) : "CUDA error";
        case NK_ERR_ALLOC: return "host allocation failed";
        case NK_ERR_MULT: return "too many distinct multiplicities";
        case NK_ERR_SIZE: return "more entries than the fixed scratch of nk_dot_static serves";
    }
    return "unknown error";
}

int nk_last_cuda_error(void) { return t_last_cuda; }
const char *nk_version(void) { return "nk 0.1 (sm_100a, fp64)"; }

int nk_workspace_bytes(int64_t E, int N, size_t *bytes)
{
    int64_t L;
    if (!bytes || !nk_valid_EN(E, N, &L)) return NK_ERR_ARG;
    *bytes = nk_carve_sizes(L).total;
    return NK_OK;
}

void nk_free(nk_ctx *c)
{
    if (!c) return;
    for (auto &sl : c->graph)
        if (sl.exec) cudaGraphExecDestroy(sl.exec);
    if (c->batch_ready) {
        cudaStreamDestroy(c->copy_in);
        cudaStreamDestroy(c->copy_out);
        for (int s = 0; s < 2; ++s) {
            cudaEventDestroy(c->ev_f[s]);
            cudaEventDestroy(c->ev_solve[s]);
            cudaEventDestroy(c->ev_out[s]);
        }
        cudaEventDestroy(c->ev_start);
    }
    nk_dist_release(c);
    delete c->prof;
    delete c;
}

}  // extern "C"

namespace {

inline cudaStream_t S(void *stream) { return static_cast<cudaStream_t>(stream); }

// "fuse_p" = 2 (default): fold p = r + beta p into ax_e's load.  On at every size since the x update is deferred
// ("defer_x": the fused path then moves 127 B per point and iteration against 131 for the separate direction update,
// with one launch fewer); measured per iteration, fused against separate: 4.1 M points 97.8 vs 100.5 us, 8.2 M 183 vs
// 198, 16.8 M 359 vs 378, 28.3 M 583 vs 607, config 5 (56.6 M) 1.177 vs 1.204 ms.  (Before the deferral it paid off
// only up to 2^24 points: -6..-9 % on configs 1-2, -2.5 % on config 3, +-0 at config 5.)
inline bool fuse_p_on(const nk_ctx *c)
{
    return c->opt_fuse_p != 0;
}

// "fuse_gs" = 2 (default): gs rides in the residual update from 2^20 local points on (measured per iteration, graph
// replay, fused against separate: N=7 1.05 M points 30.4 vs 33.1 us, 2.1 M 51.7 vs 55.1; N=11 1.77 M 49.1 vs 51.6;
// N=9 2.05 M 54.9 vs 57.1, config 5 1.25 vs 1.28 ms; below, on meshes that sit in L2, the separate kernel is as fast
// or faster: N=9 1.02 M 32.4 vs 31.8, N=7 0.52 M 21.9 vs 21.2).  The separate weighted dot needs the summed w, so
// without "fuse_pap" gs stays a kernel of its own.
inline bool fuse_gs_on(const nk_ctx *c)
{
    return c->opt_fuse_pap && (c->opt_fuse_gs == 1 || (c->opt_fuse_gs == 2 && c->L >= NK_FUSE_GS_AUTO_MIN_L));
}

// One CG iteration, enqueued (S 3 call stack (3)).  hist_k: where sqrt(rho') goes (DEVICE).
// "defer_x" (default on): two iterations share one pass over x.  pair = 0: a plain iteration; 1: the first of a pair
// (x untouched, alpha kept); 2: the second (x takes both steps).  The direction of the first iteration must survive
// the second, so the direction lives in two vectors (p, p2):
//   without "fuse_p" (large meshes): first  p2 = r + beta p; second runs on p2, then x and p = r + beta' p2
//                                    (nk_vec.cu update_p2_kernel / update_pxx_kernel);
//   with "fuse_p" and "fuse_gs":     the second ax_e forms its direction OUT OF PLACE (reads c->pc, writes the other
//                                    vector) and the fused gs update applies x = fma(alpha', p', fma(alpha, p, x));
//                                    c->pc follows the current direction, the pending update at the end lands in p.
// x, r, p and the history are bit for bit those of plain iterations.
inline bool defer_x_on(const nk_ctx *c) { return c->opt_defer_x && (!fuse_p_on(c) || fuse_gs_on(c)); }

cudaError_t enqueue_iteration(nk_ctx *c, double *x, double *hist_k, cudaStream_t st, int pair = 0)
{
    cudaError_t e;
    const int fuse_pap = c->opt_fuse_pap;
    const bool fuse_p = fuse_p_on(c);
    double *const pa = c->pc;                                         // the direction before this iteration's update
    double *const pb = (fuse_p && pair == 2) ? (pa == c->p ? c->p2 : c->p) : pa;     // where this iteration's direction goes
    const double *const dir = fuse_p ? pb : (pair == 2 ? c->p2 : c->p);              // what ax_e is applied to
    if (c->p_pending) {          // p = r + beta p folded into this ax_e's load
        NK_LAUNCH(NK_K_AX, nk_launch_ax_tma(c, pb, pb == pa ? nullptr : pa, c->r, c->w, fuse_pap, st));
        c->p_pending = 0;
    } else {
        NK_LAUNCH(NK_K_AX, nk_launch_ax_tma(c, nullptr, dir, nullptr, c->w, fuse_pap, st));
    }
    // "fuse_gs": gs and the mask ride in the residual update, which gathers the copies of shared nodes from the
    // unsummed w (nk_vec.cu); the separate weighted dot needs the summed w, so it keeps gs in place
    const int fuse_gs = fuse_gs_on(c);
    if (!fuse_gs) NK_LAUNCH(NK_K_GS, nk_launch_gs(c, c->w, 1, st));
    if (!fuse_pap) NK_LAUNCH(NK_K_DOT, nk_launch_dot(c, c->w, dir, nullptr, NK_EPI_PAP, st));
    c->w_unsummed = fuse_gs;
    if (fuse_p) {
        if (pair == 1) NK_LAUNCH(NK_K_UPDATE_XR, nk_launch_update_r_first(c, hist_k, st));
        else if (pair == 2) NK_LAUNCH(NK_K_UPDATE_XR, nk_launch_update_xxr(c, x, pa, pb, hist_k, st));
        else NK_LAUNCH(NK_K_UPDATE_XR, nk_launch_update_xr(c, x, hist_k, fuse_gs, st));
        c->pc = pb;
        c->p_pending = 1;
    } else {
        // r first, then x and p together: p is read once per iteration instead of twice (65 vs 73 B/pt)
        NK_LAUNCH(NK_K_UPDATE_XR, nk_launch_update_r(c, hist_k, fuse_gs, st));
        if (pair == 1) NK_LAUNCH(NK_K_UPDATE_P, nk_launch_update_p2(c, st));
        else if (pair == 2) NK_LAUNCH(NK_K_UPDATE_P, nk_launch_update_pxx(c, x, st));
        else NK_LAUNCH(NK_K_UPDATE_P, nk_launch_update_px(c, x, st));
    }
    return cudaSuccess;
}

cudaError_t enqueue_cg(nk_ctx *c, const double *f, double *x, int niter, double *res_hist, cudaStream_t st)
{
    cudaError_t e;
    c->p_pending = 0;
    c->pc = c->p;
    struct pc_scope { nk_ctx *c; ~pc_scope() { c->pc = c->p; } } pcs{c};
    if ((e = prof_mark(c, -1, st)) != cudaSuccess) return e;
    NK_LAUNCH(NK_K_INIT, nk_launch_cg_init(c, f, x, res_hist, st));
    // "pdl": every kernel of the loop waits (griddepcontrol.wait) before it reads what its predecessor
    // wrote, so the launches may overlap tail and prologue; the event pairs of "profile" would serialise them
    struct pdl_scope { nk_ctx *c; ~pdl_scope() { c->pdl_now = 0; } } scope{c};
    c->pdl_now = c->opt_profile ? 0 : nk_pdl_mode(c);
    const bool defer = defer_x_on(c);
    for (int k = 1; k <= niter; ++k) {
        // pairs (k, k+1) from the front; an odd last iteration is a plain one, so x, r, p are complete at the end
        const int pair = !defer ? 0 : (k % 2 == 1 ? (k < niter ? 1 : 0) : 2);
        if ((e = enqueue_iteration(c, x, res_hist + k, st, pair)) != cudaSuccess) return e;
    }
    if (c->p_pending) {          // leave the context with p up to date, in c->p wherever the direction was last
        NK_LAUNCH(NK_K_UPDATE_P, nk_launch_update_p(c, st));
        c->p_pending = 0;
    }
    return cudaSuccess;
}

// The operator calls launch their kernels as programmatic dependents too (unless "pdl" = 0 or "profile"): every
// kernel here executes griddepcontrol.wait before it touches a vector, so whatever precedes it on the stream --
// one of ours or anybody's -- has completed and flushed by then; what overlaps is the launch latency and, in
// ax_e, the producer warp's first bulk copies of the (static) geometric factors.
struct pdl_call_scope {
    nk_ctx *c;
    explicit pdl_call_scope(nk_ctx *ctx) : c(ctx) { c->pdl_now = c->opt_profile ? 0 : nk_pdl_mode(c); }
    ~pdl_call_scope() { c->pdl_now = 0; }
};

}  // namespace

extern "C" {

int nk_ax_e(nk_ctx *c, const double *u, double *w, void *stream)
{
    if (!c || !u || !w || u == w || !nk_aligned16(u) || !nk_aligned16(w)) return NK_ERR_ARG;
    pdl_call_scope scope(c);
    NK_CUDA(prof_mark(c, -1, S(stream)));
    NK_CUDA(nk_launch_ax_tma(c, nullptr, u, nullptr, w, 0, S(stream)));
    NK_CUDA(prof_mark(c, NK_K_AX, S(stream)));
    return NK_OK;
}

int nk_gs(nk_ctx *c, double *v, void *stream)
{
    if (!c || !v || !nk_aligned16(v)) return NK_ERR_ARG;
    pdl_call_scope scope(c);
    NK_CUDA(prof_mark(c, -1, S(stream)));
    NK_CUDA(nk_launch_gs(c, v, 0, S(stream)));
    NK_CUDA(prof_mark(c, NK_K_GS, S(stream)));
    return NK_OK;
}

int nk_ax(nk_ctx *c, const double *u, double *w, void *stream)
{
    if (!c || !u || !w || u == w || !nk_aligned16(u) || !nk_aligned16(w)) return NK_ERR_ARG;
    pdl_call_scope scope(c);
    NK_CUDA(prof_mark(c, -1, S(stream)));
    NK_CUDA(nk_launch_ax_tma(c, nullptr, u, nullptr, w, 0, S(stream)));
    NK_CUDA(prof_mark(c, NK_K_AX, S(stream)));
    NK_CUDA(nk_launch_gs(c, w, 1, S(stream)));
    NK_CUDA(prof_mark(c, NK_K_GS, S(stream)));
    return NK_OK;
}

int nk_dot(nk_ctx *c, const double *a, const double *b, double *out, void *stream)
{
    if (!c || !a || !b || !out || !nk_aligned16(a) || !nk_aligned16(b)) return NK_ERR_ARG;
    NK_CUDA(nk_launch_dot(c, a, b, out, NK_EPI_STORE, S(stream)));
    return NK_OK;
}

// "graph" = 2 (default): replay a CUDA graph where launch gaps matter (measured: config 2 3.8 -> 1.9 ms,
// config 3 15.0 -> 13.0 ms per 100 iterations), enqueue directly on large meshes
// "coop" = 2 (default): the whole solve as one cooperative launch on meshes that sit in L2, where an iteration is
// a few microseconds of work and even a replayed graph of programmatic dependents costs 10-16 us per iteration
// (measured: 7.8-13 us here, profiles/r2_sweep_coop.csv)
static bool cg_uses_coop(const nk_ctx *c)
{
    return !c->opt_profile && c->coop_ok && nk_coop_supported(c->N) && !c->dist_mult &&
           (c->opt_coop == 1 || (c->opt_coop == 2 && c->L <= NK_COOP_AUTO_MAX_L));
}

static bool cg_uses_graph(const nk_ctx *c)
{
    return !c->opt_profile && !cg_uses_coop(c) &&
           (c->opt_graph == 1 || (c->opt_graph == 2 && c->L <= NK_GRAPH_AUTO_MAX_L));
}

int nk_get_cg_path(nk_ctx *c, int *path, int *pdl_mode)
{
    if (!c || !path) return NK_ERR_ARG;
    *path = cg_uses_coop(c) ? 2 : cg_uses_graph(c) ? 1 : 0;
    if (pdl_mode) *pdl_mode = c->opt_profile ? 0 : nk_pdl_mode(c);
    return NK_OK;
}

int nk_cg(nk_ctx *c, const double *f, double *x, int niter, double *res_hist, void *stream)
{
    if (!c || !f || !x || !res_hist || niter < 0 || f == x || !nk_aligned16(f) || !nk_aligned16(x))
        return NK_ERR_ARG;
    cudaStream_t st = S(stream);
    if (niter > 0 && cg_uses_coop(c)) {
        NK_CUDA(nk_launch_cg_coop(c, f, x, niter, res_hist, st));
        c->p_pending = 0;
        c->w_unsummed = 1;
        return NK_OK;
    }
    const bool use_graph = niter > 0 && cg_uses_graph(c);
    if (!use_graph) {
        NK_CUDA(enqueue_cg(c, f, x, niter, res_hist, st));
        return NK_OK;
    }
    // Record the launch sequence once per (f, x, res_hist, niter, options) and replay it: the CG
    // loop of the small configs is launch-bound (S 7 hard part 4).
    // one bit field per option (1, 2, 2, 2, 1 bits): two option sets never share a key
    const int key = c->opt_fuse_pap | (c->opt_fuse_p << 1) | (c->opt_fuse_gs << 3) | (c->opt_pdl << 5) | (c->opt_defer_x << 7);
    nk_ctx::graph_slot *g = nullptr;
    for (auto &sl : c->graph)
        if (sl.exec && sl.f == f && sl.x == x && sl.hist == res_hist && sl.niter == niter && sl.key == key) g = &sl;
    if (!g) {
        // two slots (nk_cg_host_batch alternates between two sets of buffers); the one used longest ago goes
        g = c->graph[0].stamp <= c->graph[1].stamp ? &c->graph[0] : &c->graph[1];
        cudaStream_t cap;
        NK_CUDA(cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
        cudaGraph_t graph = nullptr;
        cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
        const int64_t launches_before = c->launches;
        if (e == cudaSuccess) {
            const cudaError_t e1 = enqueue_cg(c, f, x, niter, res_hist, cap);
            const cudaError_t e2 = cudaStreamEndCapture(cap, &graph);
            e = (e1 != cudaSuccess) ? e1 : e2;
        }
        c->launches = launches_before;
        if (e == cudaSuccess && g->exec) {             // same topology, new pointers: update in place
            cudaGraphExecUpdateResultInfo info;
            if (cudaGraphExecUpdate(g->exec, graph, &info) != cudaSuccess) {
                (void)cudaGetLastError();
                cudaGraphExecDestroy(g->exec);
                g->exec = nullptr;
            }
        }
        if (e == cudaSuccess && !g->exec) e = cudaGraphInstantiate(&g->exec, graph, 0);
        if (graph) cudaGraphDestroy(graph);
        cudaStreamDestroy(cap);
        if (e != cudaSuccess) {
            if (g->exec) cudaGraphExecDestroy(g->exec);
            g->exec = nullptr;
            return nk_cuda_fail(e);
        }
        g->f = f; g->x = x; g->hist = res_hist; g->niter = niter; g->key = key;
    }
    g->stamp = ++c->graph_clock;
    NK_CUDA(cudaGraphLaunch(g->exec, st));
    int per_iter = 3 + (c->opt_fuse_pap ? 0 : 1) + (fuse_p_on(c) ? 0 : 1) - (fuse_gs_on(c) ? 1 : 0);
    c->launches += 1 + (int64_t)niter * per_iter + ((fuse_p_on(c) && niter > 0) ? 1 : 0);
    c->p_pending = 0;
    return NK_OK;
}

int nk_cg_host(nk_ctx *c, const double *f_host, double *x_host, int niter, double *res_hist_host, void *stream)
{
    if (!c || !f_host || !x_host || !res_hist_host || niter < 0 || niter + 1 > NK_HIST_MAX) return NK_ERR_ARG;
    cudaStream_t st = S(stream);
    const size_t bytes = (size_t)c->L * sizeof(double);
    NK_CUDA(cudaMemcpyAsync(c->hf, f_host, bytes, cudaMemcpyHostToDevice, st));
    const int rc = nk_cg(c, c->hf, c->hx, niter, c->hist, stream);
    if (rc != NK_OK) return rc;
    NK_CUDA(cudaMemcpyAsync(x_host, c->hx, bytes, cudaMemcpyDeviceToHost, st));
    NK_CUDA(cudaMemcpyAsync(res_hist_host, c->hist, (size_t)(niter + 1) * sizeof(double), cudaMemcpyDeviceToHost, st));
    NK_CUDA(cudaStreamSynchronize(st));
    return NK_OK;
}

// Several right-hand sides, pipelined: RHS j+1 goes in and solution j-1 comes out (two copy streams, two sets of
// staging buffers) while solve j runs on `stream`.
int nk_cg_host_batch(nk_ctx *c, int nrhs, const double *const *f_host, double *const *x_host, int niter,
                     double *const *res_hist_host, void *stream)
{
    if (!c || nrhs < 0 || niter < 0 || niter + 1 > NK_HIST_MAX) return NK_ERR_ARG;
    if (nrhs > 0 && (!f_host || !x_host || !res_hist_host)) return NK_ERR_ARG;
    for (int j = 0; j < nrhs; ++j)
        if (!f_host[j] || !x_host[j] || !res_hist_host[j]) return NK_ERR_ARG;
    cudaStream_t st = S(stream);
    if (!c->batch_ready) {
        NK_CUDA(cudaStreamCreateWithFlags(&c->copy_in, cudaStreamNonBlocking));
        NK_CUDA(cudaStreamCreateWithFlags(&c->copy_out, cudaStreamNonBlocking));
        for (int s = 0; s < 2; ++s) {
            NK_CUDA(cudaEventCreateWithFlags(&c->ev_f[s], cudaEventDisableTiming));
            NK_CUDA(cudaEventCreateWithFlags(&c->ev_solve[s], cudaEventDisableTiming));
            NK_CUDA(cudaEventCreateWithFlags(&c->ev_out[s], cudaEventDisableTiming));
        }
        NK_CUDA(cudaEventCreateWithFlags(&c->ev_start, cudaEventDisableTiming));
        c->batch_ready = 1;
    }
    const size_t bytes = (size_t)c->L * sizeof(double);
    double *fb[2] = {c->hf, c->hf2}, *xb[2] = {c->hx, c->hx2}, *hb[2] = {c->hist, c->hist2};
    NK_CUDA(cudaEventRecord(c->ev_start, st));                     // the copies start after what precedes on `stream`
    NK_CUDA(cudaStreamWaitEvent(c->copy_in, c->ev_start, 0));
    NK_CUDA(cudaStreamWaitEvent(c->copy_out, c->ev_start, 0));
    for (int j = 0; j < nrhs; ++j) {
        const int s = j & 1;
        // staging set s is free once solve j-2 has read f (ev_solve) and its x and history have left (ev_out)
        if (j >= 2) NK_CUDA(cudaStreamWaitEvent(c->copy_in, c->ev_solve[s], 0));
        NK_CUDA(cudaMemcpyAsync(fb[s], f_host[j], bytes, cudaMemcpyHostToDevice, c->copy_in));
        NK_CUDA(cudaEventRecord(c->ev_f[s], c->copy_in));
        NK_CUDA(cudaStreamWaitEvent(st, c->ev_f[s], 0));
        if (j >= 2) NK_CUDA(cudaStreamWaitEvent(st, c->ev_out[s], 0));
        const int rc = nk_cg(c, fb[s], xb[s], niter, hb[s], stream);
        if (rc != NK_OK) { cudaDeviceSynchronize(); return rc; }
        NK_CUDA(cudaEventRecord(c->ev_solve[s], st));
        NK_CUDA(cudaStreamWaitEvent(c->copy_out, c->ev_solve[s], 0));
        NK_CUDA(cudaMemcpyAsync(x_host[j], xb[s], bytes, cudaMemcpyDeviceToHost, c->copy_out));
        NK_CUDA(cudaMemcpyAsync(res_hist_host[j], hb[s], (size_t)(niter + 1) * sizeof(double), cudaMemcpyDeviceToHost,
                                c->copy_out));
        NK_CUDA(cudaEventRecord(c->ev_out[s], c->copy_out));
    }
    for (int s = 0; s < 2 && s < nrhs; ++s) NK_CUDA(cudaStreamWaitEvent(st, c->ev_out[s], 0));
    NK_CUDA(cudaStreamSynchronize(st));
    return NK_OK;
}

}  // extern "C"

extern "C" {

int nk_cg_init(nk_ctx *c, const double *f, double *x, void *stream)
{
    if (!c || !f || !x || f == x || !nk_aligned16(f) || !nk_aligned16(x)) return NK_ERR_ARG;
    c->p_pending = 0;
    NK_CUDA(nk_launch_cg_init(c, f, x, c->res_dummy, S(stream)));
    return NK_OK;
}

int nk_cg_load_state(nk_ctx *c, const double *r, const double *p, double rho, void *stream)
{
    if (!c || !r || !p) return NK_ERR_ARG;
    cudaStream_t st = S(stream);
    const size_t bytes = (size_t)c->L * sizeof(double);
    double scal[NK_S_COUNT] = {0};
    scal[NK_S_RHO] = rho; scal[NK_S_RHO_OLD] = rho; scal[NK_S_RHO_NEW] = rho;
    c->p_pending = 0;
    c->w_unsummed = 0;
    NK_CUDA(cudaMemcpyAsync(c->r, r, bytes, cudaMemcpyDeviceToDevice, st));
    NK_CUDA(cudaMemcpyAsync(c->p, p, bytes, cudaMemcpyDeviceToDevice, st));
    NK_CUDA(cudaMemcpyAsync(c->red.scal, scal, sizeof(scal), cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaStreamSynchronize(st));      // scal[] is a stack buffer
    return NK_OK;
}

int nk_cg_step(nk_ctx *c, double *x, void *stream)
{
    if (!c || !x || !nk_aligned16(x)) return NK_ERR_ARG;
    NK_CUDA(enqueue_iteration(c, x, c->res_dummy, S(stream)));
    return NK_OK;
}

int nk_cg_get_state(nk_ctx *c, double *r, double *p, double *w, void *stream)
{
    if (!c) return NK_ERR_ARG;
    cudaStream_t st = S(stream);
    const size_t bytes = (size_t)c->L * sizeof(double);
    if (c->p_pending) {
        NK_CUDA(nk_launch_update_p(c, st));
        c->p_pending = 0;
    }
    if (r) NK_CUDA(cudaMemcpyAsync(r, c->r, bytes, cudaMemcpyDeviceToDevice, st));
    if (p) NK_CUDA(cudaMemcpyAsync(p, c->p, bytes, cudaMemcpyDeviceToDevice, st));
    if (w) {
        NK_CUDA(cudaMemcpyAsync(w, c->w, bytes, cudaMemcpyDeviceToDevice, st));
        // "fuse_gs" leaves the UNSUMMED ax_e output in the context (the update gathered from it): what is handed
        // out is w = M Q Q^T A_L p as documented, summed and masked on the copy
        if (c->w_unsummed) NK_CUDA(nk_launch_gs(c, w, 1, st));
    }
    return NK_OK;
}

int nk_get_scalars(nk_ctx *c, double *out5_host, void *stream)
{
    if (!c || !out5_host) return NK_ERR_ARG;
    cudaStream_t st = S(stream);
    double scal[NK_S_COUNT];
    NK_CUDA(cudaMemcpyAsync(scal, c->red.scal, sizeof(scal), cudaMemcpyDeviceToHost, st));
    NK_CUDA(cudaStreamSynchronize(st));
    out5_host[0] = scal[NK_S_RHO_OLD];
    out5_host[1] = scal[NK_S_PAP];
    out5_host[2] = scal[NK_S_ALPHA];
    out5_host[3] = scal[NK_S_RHO_NEW];
    out5_host[4] = scal[NK_S_BETA];
    return NK_OK;
}

static int *option_slot(nk_ctx *c, const char *name, int *lo, int *hi)
{
    if (!std::strcmp(name, "fuse_pap")) { *lo = 0; *hi = 1; return &c->opt_fuse_pap; }
    if (!std::strcmp(name, "fuse_p")) { *lo = 0; *hi = 2; return &c->opt_fuse_p; }
    if (!std::strcmp(name, "fuse_gs")) { *lo = 0; *hi = 2; return &c->opt_fuse_gs; }
    if (!std::strcmp(name, "graph")) { *lo = 0; *hi = 2; return &c->opt_graph; }
    if (!std::strcmp(name, "coop")) { *lo = 0; *hi = 2; return &c->opt_coop; }
    if (!std::strcmp(name, "defer_x")) { *lo = 0; *hi = 1; return &c->opt_defer_x; }
    if (!std::strcmp(name, "pdl")) { *lo = 0; *hi = 3; return &c->opt_pdl; }
    if (!std::strcmp(name, "profile")) { *lo = 0; *hi = 1; return &c->opt_profile; }
    return nullptr;
}

int nk_set_option(nk_ctx *c, const char *name, int value)
{
    if (!c || !name) return NK_ERR_ARG;
    int lo, hi;
    int *slot = option_slot(c, name, &lo, &hi);
    if (!slot || value < lo || value > hi) return NK_ERR_ARG;
    *slot = value;
    return NK_OK;
}

int nk_get_option(nk_ctx *c, const char *name, int *value)
{
    if (!c || !name || !value) return NK_ERR_ARG;
    int lo, hi;
    int *slot = option_slot(c, name, &lo, &hi);
    if (!slot) return NK_ERR_ARG;
    *value = *slot;
    return NK_OK;
}

int nk_get_sizes(nk_ctx *c, int64_t *n_local, int64_t *n_unique, int64_t *n_shared_unique, int64_t *n_masked_unique)
{
    if (!c) return NK_ERR_ARG;
    if (n_local) *n_local = c->L;
    if (n_unique) *n_unique = c->n_unique;
    if (n_shared_unique) *n_shared_unique = c->n_shared_unique;
    if (n_masked_unique) *n_masked_unique = c->n_masked_unique;
    return NK_OK;
}

int nk_get_setup_info(nk_ctx *c, int *plan_builder, double *plan_seconds, double *total_seconds)
{
    if (!c) return NK_ERR_ARG;
    if (plan_builder) *plan_builder = c->plan_builder;
    if (plan_seconds) *plan_seconds = c->setup_plan_s;
    if (total_seconds) *total_seconds = c->setup_total_s;
    return NK_OK;
}

int nk_get_plan_array(nk_ctx *c, int which, const void **dev, size_t *bytes)
{
    if (!c || !dev || !bytes) return NK_ERR_ARG;
    const int nvb = nk_gsu_blocks(c->sm_count, c->L >> 1);
    const void *p = nullptr;
    size_t n = 0;
    switch (which) {
    case 0: p = c->code; n = (size_t)c->L; break;
    case 1: p = c->row_off; n = ((size_t)c->n_rows + 1) * 4; break;
    case 2: p = c->row_idx; n = (size_t)c->n_listed * 4; break;
    case 3: p = c->pk; n = (size_t)c->n_pk * 4; break;
    case 4: p = c->gs_desc; n = (size_t)(c->n_gs_chunks > 0 ? c->n_gs_chunks : 1) * 32; break;
    case 5: p = c->nbr; n = (size_t)c->L * 4; break;
    case 6: p = c->gx; n = (size_t)(c->gx_rows - c->gx) * 4; break;
    case 7: p = c->gx_rows; n = (size_t)c->n_gx_rows * 4; break;
    case 8: p = c->gx_blk; n = ((size_t)nvb + 1) * 4; break;
    case 9: p = c->ctab; n = NK_CTAB * sizeof(double); break;
    case 10: p = c->mtab; n = NK_CTAB * sizeof(double); break;
    default: return NK_ERR_ARG;
    }
    *dev = p;
    *bytes = n;
    return NK_OK;
}

int nk_get_gs_sizes(nk_ctx *c, int64_t *n_rows, int64_t *n_listed, int64_t *n_sum_rows)
{
    if (!c) return NK_ERR_ARG;
    if (n_rows) *n_rows = c->n_rows;
    if (n_listed) *n_listed = c->n_listed;
    if (n_sum_rows) *n_sum_rows = c->n_sum_rows;
    return NK_OK;
}

int nk_get_mult(nk_ctx *c, double *mult, void *stream)
{
    if (!c || !mult) return NK_ERR_ARG;
    NK_CUDA(nk_launch_get_mult(c, mult, S(stream)));
    return NK_OK;
}

int nk_get_geom(nk_ctx *c, double *G6, void *stream)
{
    if (!c || !G6) return NK_ERR_ARG;
    NK_CUDA(nk_launch_get_geom(c, G6, S(stream)));
    return NK_OK;
}

int nk_get_D(nk_ctx *c, double *D_host, double *xi_host, double *w_host)
{
    if (!c) return NK_ERR_ARG;
    if (D_host) std::memcpy(D_host, c->D, sizeof(double) * c->n * c->n);
    if (xi_host) std::memcpy(xi_host, c->xi, sizeof(double) * c->n);
    if (w_host) std::memcpy(w_host, c->wq, sizeof(double) * c->n);
    return NK_OK;
}

int nk_get_kernel_times(nk_ctx *c, double *ms_host, int64_t *count_host, void *stream)
{
    if (!c || !ms_host || !count_host) return NK_ERR_ARG;
    for (int k = 0; k < NK_K_COUNT; ++k) { ms_host[k] = 0.0; count_host[k] = 0; }
    NK_CUDA(cudaStreamSynchronize(S(stream)));
    nk_prof *p = c->prof;
    if (!p) return NK_OK;
    for (size_t i = 1; i < p->used; ++i) {
        const int k = p->cls[i];
        if (k < 0) continue;
        float ms = 0.f;
        NK_CUDA(cudaEventElapsedTime(&ms, p->ev[i - 1], p->ev[i]));
        ms_host[k] += (double)ms;
        count_host[k] += 1;
    }
    p->used = 0;
    return NK_OK;
}

int nk_ax_batch_elements(int N)
{
    const int epb = nk_ax_tma_epb(N);
    return epb > 0 ? epb : NK_ERR_ARG;
}

int nk_get_ax_launch(nk_ctx *c, int *batch_elements, int *ctas, int64_t *max_batches_per_cta)
{
    if (!c) return NK_ERR_ARG;
    const int epb = nk_ax_tma_epb(c->N);
    const int64_t nb = (c->E + epb - 1) / epb;
    const int64_t grid = nb < (int64_t)c->sm_count ? nb : (int64_t)c->sm_count;
    if (batch_elements) *batch_elements = epb;
    if (ctas) *ctas = (int)grid;
    // every CTA takes a contiguous range of floor or ceil(E / ctas) elements, in batches
    if (max_batches_per_cta) *max_batches_per_cta = ((c->E + grid - 1) / grid + epb - 1) / epb;
    return NK_OK;
}

int nk_get_launch_count(nk_ctx *c, int64_t *count)
{
    if (!c || !count) return NK_ERR_ARG;
    *count = c->launches;
    return NK_OK;
}

}  // extern "C"

// ---- Jacobi-preconditioned CG ---------------------------------------------------------
namespace {
cudaError_t ensure_dinv(nk_ctx *c, cudaStream_t st)
{
    if (c->have_dinv) return cudaSuccess;
    cudaError_t e;
    if ((e = nk_launch_diag(c, c->dinv, st)) != cudaSuccess) return e;
    if ((e = nk_launch_gs(c, c->dinv, 0, st)) != cudaSuccess) return e;
    if ((e = nk_launch_invert_diag(c, c->dinv, st)) != cudaSuccess) return e;
    c->have_dinv = 1;
    return cudaSuccess;
}
}  // namespace

extern "C" {

int nk_get_diag(nk_ctx *c, double *diag, void *stream)
{
    if (!c || !diag || !nk_aligned16(diag)) return NK_ERR_ARG;
    NK_CUDA(nk_launch_diag(c, diag, S(stream)));
    NK_CUDA(nk_launch_gs(c, diag, 0, S(stream)));
    return NK_OK;
}

int nk_pcg(nk_ctx *c, const double *f, double *x, int niter, double *res_hist, void *stream)
{
    if (!c || !f || !x || !res_hist || niter < 0 || f == x || !nk_aligned16(f) || !nk_aligned16(x))
        return NK_ERR_ARG;
    cudaStream_t st = S(stream);
    cudaError_t e;
    NK_CUDA(ensure_dinv(c, st));
    c->p_pending = 0;
    c->w_unsummed = 0;
    NK_CUDA(prof_mark(c, -1, st));
    NK_CUDA(nk_launch_pcg_init(c, f, x, res_hist, st));
    NK_CUDA(prof_mark(c, NK_K_INIT, st));
    struct pdl_scope { nk_ctx *c; ~pdl_scope() { c->pdl_now = 0; } } scope{c};
    c->pdl_now = c->opt_profile ? 0 : nk_pdl_mode(c);      // as in nk_cg: every kernel of the loop waits before its first dependent read
    for (int k = 1; k <= niter; ++k) {
        NK_CUDA(nk_launch_ax_tma(c, nullptr, c->p, nullptr, c->w, c->opt_fuse_pap, st));
        NK_CUDA(prof_mark(c, NK_K_AX, st));
        NK_CUDA(nk_launch_gs(c, c->w, 1, st));
        NK_CUDA(prof_mark(c, NK_K_GS, st));
        if (!c->opt_fuse_pap) {
            NK_CUDA(nk_launch_dot(c, c->w, c->p, nullptr, NK_EPI_PAP, st));
            NK_CUDA(prof_mark(c, NK_K_DOT, st));
        }
        NK_CUDA(nk_launch_update_xrz(c, x, res_hist + k, st));
        NK_CUDA(prof_mark(c, NK_K_UPDATE_XR, st));
        NK_CUDA(nk_launch_update_pz(c, x, st));
        NK_CUDA(prof_mark(c, NK_K_UPDATE_P, st));
    }
    (void)e;
    return NK_OK;
}

}  // extern "C"
