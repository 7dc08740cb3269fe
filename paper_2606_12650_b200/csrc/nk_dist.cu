// nk_dist.cu -- gs and the CG iteration over an element partition, one rank per GPU (
// PAPER.md:336 "multiple GPU support (through MPI) is necessary" -- the paper's future work; the original Nekbone is
// MPI).  Every rank sets the library up on ITS elements with GLOBAL node ids; ax_e and the vector
// kernels are rank-local and unchanged.  What crosses ranks:
//
//   * gs: ONE neighbour-wise exchange.  An INTERFACE node is a node another rank holds too (they all lie on
//     element boundaries: nk_dist_candidates).  Each rank adds up its own copies of every interface node
//     (dist_partial_kernel, ascending local index), sends each neighbour the partial sums of the nodes the two
//     share -- ascending global id, so both sides agree on the order without exchanging it -- receives theirs, and
//     adds, per node, the partial sums of all holders IN ASCENDING RANK ORDER (dist_unpack_kernel): every rank gets
//     the same bits, reruns are bitwise equal.  Only shared values move: 8 B per node and neighbour.
//   * the two dot products of an iteration: each rank's partial total is all-gathered (one double) and added in
//     rank order by one thread, which then runs the epilogue the single-GPU kernels run in their last block.
//
// The library enqueues kernels and owns the plan; the transfers themselves are the caller's, through a callback
// (nk_exchange_fn: NCCL grouped send/recv and all-gather via torch.distributed in dist.py) that the library
// invokes in the right places -- so the per-iteration sequence lives here, not in Python.  Inside nk_dist_cg the
// halo exchange runs on a second stream and overlaps the interior elements' ax_e: the rank's elements that hold an
// interface node come FIRST in its local order (the caller's job; nk_dist_setup measures how far they reach), so
// "interface" and "interior" are two contiguous element ranges.
//
// Nothing here has run on more than one GPU (one per box): verified with ranks as host threads of one process,
// transfers replaced by device copies (tests/test_gpu_dist.py), and over gloo / a size-1 NCCL group.
#include <algorithm>
#include <new>
#include <vector>

#include "nk_internal.h"
#include "nk_host.h"
#include "nk_reduce.cuh"
#include "../../include/nk.h"

struct nk_dist {
    int rank = 0, world = 1;
    // host side of the plan
    std::vector<int> nbr_rank;                 // neighbour ranks, ascending
    std::vector<int64_t> nbr_off, nbr_cnt;     // their segments of the send / receive buffer
    int64_t n_if = 0, n_send = 0, n_iface_elems = 0, n_copies = 0;
    // device side (cudaMalloc'ed here, freed in nk_dist_release)
    int32_t *cp_off = nullptr, *cp_idx = nullptr;     // local copies of interface node i: cp_idx[cp_off[i] .. cp_off[i+1])
    int32_t *snd_off = nullptr, *snd_pos = nullptr;   // where its partial sum goes in the send buffer (one per neighbour holding it)
    int32_t *src_off = nullptr, *src = nullptr;       // its holders in ascending rank order: -1 = this rank, else position in recv
    double *own = nullptr;                            // n_if partial sums
    double *tmp = nullptr;                            // 4 doubles: rank-local totals of split launches
    // caller-owned exchange buffers (nk_dist_set_buffers)
    double *send = nullptr, *recv = nullptr, *ssend = nullptr, *sgath = nullptr;
    cudaStream_t comm = nullptr;
    cudaEvent_t ev_packed = nullptr, ev_halo = nullptr;
};

void nk_dist_release(nk_ctx *c)
{
    nk_dist *d = c->dist;
    if (!d) return;
    cudaFree(d->cp_off); cudaFree(d->cp_idx); cudaFree(d->snd_off); cudaFree(d->snd_pos);
    cudaFree(d->src_off); cudaFree(d->src); cudaFree(d->own); cudaFree(d->tmp);
    if (d->comm) cudaStreamDestroy(d->comm);
    if (d->ev_packed) cudaEventDestroy(d->ev_packed);
    if (d->ev_halo) cudaEventDestroy(d->ev_halo);
    delete d;
    c->dist = nullptr;
}

namespace {

constexpr int DIST_THREADS = 256;

inline cudaStream_t S(void *stream) { return reinterpret_cast<cudaStream_t>(stream); }
inline unsigned blocks_for(int64_t n) { return (unsigned)((n + DIST_THREADS - 1) / DIST_THREADS); }

// own[i] = sum over this rank's copies of interface node i (ascending local index); the value goes to every
// neighbour that holds the node
__global__ void __launch_bounds__(DIST_THREADS)
dist_partial_kernel(const double *v, int64_t n_if, const int32_t *__restrict__ cp_off, const int32_t *__restrict__ cp_idx,
                    const int32_t *__restrict__ snd_off, const int32_t *__restrict__ snd_pos, double *__restrict__ own,
                    double *__restrict__ send)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_if) return;
    const int b = cp_off[i], e = cp_off[i + 1];
    double s = v[cp_idx[b]];
    for (int j = b + 1; j < e; ++j) s += v[cp_idx[j]];
    own[i] = s;
    for (int j = snd_off[i]; j < snd_off[i + 1]; ++j) send[snd_pos[j]] = s;
}

// total over the holders in ascending rank order -> every local copy (0 on Dirichlet nodes if asked)
__global__ void __launch_bounds__(DIST_THREADS)
dist_unpack_kernel(double *v, int64_t n_if, const int32_t *__restrict__ cp_off, const int32_t *__restrict__ cp_idx,
                   const int32_t *__restrict__ src_off, const int32_t *__restrict__ src, const double *own, const double *recv,
                   const uint8_t *__restrict__ code, int with_mask)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_if) return;
    double s = 0.0;
    for (int j = src_off[i]; j < src_off[i + 1]; ++j) {
        const int q = src[j];
        const double t = q < 0 ? own[i] : recv[q];
        s = (j == src_off[i]) ? t : s + t;
    }
    const int b = cp_off[i], e = cp_off[i + 1];
    if (with_mask && (code[cp_idx[b]] & NK_CODE_MASKED)) s = 0.0;
    for (int j = b; j < e; ++j) v[cp_idx[j]] = s;
}

// one thread: total over ranks in rank order, then the epilogue of nk_reduce.cuh
__global__ void dist_finish_kernel(int epi, const double *gath, int world, double *scal, double *out)
{
    double t = gath[0];
    for (int r = 1; r < world; ++r) t += gath[r];
    nk_epilogue(epi, t, scal, out);
}

__global__ void dist_add2_kernel(const double *a, const double *b, double *out) { out[0] = a[0] + b[0]; }

__global__ void __launch_bounds__(DIST_THREADS)
dist_set_mult_kernel(uint8_t *__restrict__ code, const double *__restrict__ mult, int64_t L, int *errflag)
{
    const int64_t l = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= L) return;
    const double m = mult[l];
    const int t = (int)m;
    if (!(m >= 1.0) || m >= (double)NK_CTAB || (double)t != m) { atomicExch(errflag, 1); return; }
    code[l] = (uint8_t)((code[l] & NK_CODE_MASKED) | (unsigned)t);
}

cudaError_t launch_partial(nk_ctx *c, const double *v, cudaStream_t st)
{
    nk_dist *d = c->dist;
    if (d->n_if == 0) return cudaSuccess;
    dist_partial_kernel<<<blocks_for(d->n_if), DIST_THREADS, 0, st>>>(v, d->n_if, d->cp_off, d->cp_idx, d->snd_off, d->snd_pos,
                                                                     d->own, d->send);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_unpack(nk_ctx *c, double *v, int with_mask, cudaStream_t st)
{
    nk_dist *d = c->dist;
    if (d->n_if == 0) return cudaSuccess;
    dist_unpack_kernel<<<blocks_for(d->n_if), DIST_THREADS, 0, st>>>(v, d->n_if, d->cp_off, d->cp_idx, d->src_off, d->src, d->own,
                                                                    d->recv, c->code, with_mask);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_finish(nk_ctx *c, int epi, double *out, cudaStream_t st)
{
    dist_finish_kernel<<<1, 1, 0, st>>>(epi, c->dist->sgath, c->dist->world, c->red.scal, out);
    c->launches++;
    return cudaGetLastError();
}

// runs `call` with the reducing kernel's rank-local total redirected to `raw` (instead of its epilogue)
template <typename F>
cudaError_t with_raw(nk_ctx *c, double *raw, F call)
{
    c->red.raw = raw;
    const cudaError_t e = call();
    c->red.raw = nullptr;
    return e;
}

inline bool ready(const nk_ctx *c) { return c && c->dist && c->dist->ssend && c->dist->sgath && (c->dist->n_send == 0 || (c->dist->send && c->dist->recv)); }

template <typename T>
cudaError_t upload(T **dev, const std::vector<T> &host)
{
    const size_t bytes = std::max<size_t>(host.size(), 1) * sizeof(T);
    cudaError_t e = cudaMalloc(reinterpret_cast<void **>(dev), bytes);
    if (e != cudaSuccess || host.empty()) return e;
    return cudaMemcpy(*dev, host.data(), host.size() * sizeof(T), cudaMemcpyHostToDevice);
}

// kind bits of the exchange callback
enum { XCH_HALO = 1, XCH_SCALAR = 2 };

int exchange(nk_ctx *c, nk_exchange_fn fn, void *user, int kind, cudaStream_t st)
{
    if (c->dist->world == 1) {                                  // nothing to move: the gathered scalar is the local one
        if (kind & XCH_SCALAR) NK_CUDA(cudaMemcpyAsync(c->dist->sgath, c->dist->ssend, sizeof(double), cudaMemcpyDeviceToDevice, st));
        return NK_OK;
    }
    if (!(kind & XCH_SCALAR) && c->dist->nbr_rank.empty()) return NK_OK;
    if (!fn) return NK_ERR_ARG;
    const int rc = fn(user, kind, reinterpret_cast<void *>(st));
    return rc == 0 ? NK_OK : NK_ERR_ARG;
}

// v <- Q Q^T v over all ranks (and the mask), no overlap: partial sums, exchange, local gs, totals
int dist_gs(nk_ctx *c, double *v, int with_mask, nk_exchange_fn fn, void *user, cudaStream_t st)
{
    NK_CUDA(launch_partial(c, v, st));
    const int rc = exchange(c, fn, user, XCH_HALO, st);
    if (rc != NK_OK) return rc;
    NK_CUDA(nk_launch_gs(c, v, with_mask, st));
    NK_CUDA(launch_unpack(c, v, with_mask, st));
    return NK_OK;
}

}  // namespace

extern "C" {

int nk_dist_candidates(int64_t E, int N, const int64_t *glo_num, int64_t *ids_out, int64_t *n_out)
{
    int64_t L;
    if (!nk_valid_EN(E, N, &L) || !glo_num || !ids_out || !n_out) return NK_ERR_ARG;
    const int n = N + 1;
    const int64_t P = (int64_t)n * n * n;
    std::vector<int64_t> ids;
    try {
        ids.reserve((size_t)(E * (P - (int64_t)(n - 2) * (n - 2) * (n - 2))));
        for (int64_t e = 0; e < E; ++e)
            for (int k = 0; k < n; ++k)
                for (int j = 0; j < n; ++j) {
                    const bool face = k == 0 || k == n - 1 || j == 0 || j == n - 1;
                    const int64_t base = e * P + (int64_t)n * (j + (int64_t)n * k);
                    if (face) {
                        for (int i = 0; i < n; ++i) ids.push_back(glo_num[base + i]);
                    } else {
                        ids.push_back(glo_num[base]);
                        if (n > 1) ids.push_back(glo_num[base + n - 1]);
                    }
                }
        std::sort(ids.begin(), ids.end());
        ids.erase(std::unique(ids.begin(), ids.end()), ids.end());
    } catch (const std::bad_alloc &) {
        return NK_ERR_ALLOC;
    }
    std::copy(ids.begin(), ids.end(), ids_out);
    *n_out = (int64_t)ids.size();
    return NK_OK;
}

int nk_dist_setup(nk_ctx *c, int rank, int world, const int64_t *glo_num, const int64_t *cand_ids, const int64_t *cand_counts,
                  void *stream)
{
    if (!c || world < 1 || rank < 0 || rank >= world || !glo_num || !cand_counts || (!cand_ids && world > 1)) return NK_ERR_ARG;
    (void)stream;
    nk_dist_release(c);
    nk_dist *d = new (std::nothrow) nk_dist();
    if (!d) return NK_ERR_ALLOC;
    c->dist = d;
    d->rank = rank; d->world = world;
    try {
        std::vector<int64_t> start((size_t)world + 1, 0);
        for (int r = 0; r < world; ++r) {
            if (cand_counts[r] < 0) return NK_ERR_ARG;
            start[(size_t)r + 1] = start[(size_t)r] + cand_counts[r];
        }
        const int64_t *mine = cand_ids + start[(size_t)rank];
        const int64_t n_mine = cand_counts[rank];
        // nodes shared with every other rank (both lists ascending): the neighbours and their segments
        std::vector<std::vector<int64_t>> shared((size_t)world);
        for (int r = 0; r < world; ++r) {
            if (r == rank) continue;
            const int64_t *theirs = cand_ids + start[(size_t)r];
            std::set_intersection(mine, mine + n_mine, theirs, theirs + cand_counts[r], std::back_inserter(shared[(size_t)r]));
        }
        std::vector<int64_t> iface;                                     // this rank's interface nodes, ascending id
        for (int r = 0; r < world; ++r) iface.insert(iface.end(), shared[(size_t)r].begin(), shared[(size_t)r].end());
        std::sort(iface.begin(), iface.end());
        iface.erase(std::unique(iface.begin(), iface.end()), iface.end());
        d->n_if = (int64_t)iface.size();
        auto node_of = [&](int64_t id) { return (int64_t)(std::lower_bound(iface.begin(), iface.end(), id) - iface.begin()); };
        // send layout: neighbours ascending, inside a segment ascending id
        std::vector<std::vector<int32_t>> snd((size_t)d->n_if);         // per node: its positions in the send buffer
        std::vector<std::vector<std::pair<int, int32_t>>> holders((size_t)d->n_if);   // (rank, recv position or -1)
        int64_t pos = 0;
        for (int r = 0; r < world; ++r) {
            const auto &sh = shared[(size_t)r];
            if (sh.empty()) continue;
            d->nbr_rank.push_back(r);
            d->nbr_off.push_back(pos);
            d->nbr_cnt.push_back((int64_t)sh.size());
            for (int64_t id : sh) {
                const int64_t i = node_of(id);
                snd[(size_t)i].push_back((int32_t)pos);
                holders[(size_t)i].push_back({r, (int32_t)pos});
                ++pos;
            }
        }
        d->n_send = pos;
        for (int64_t i = 0; i < d->n_if; ++i) {
            holders[(size_t)i].push_back({rank, -1});
            std::sort(holders[(size_t)i].begin(), holders[(size_t)i].end());
        }
        // local copies of the interface nodes (ascending local index), and how far the elements holding them reach
        std::vector<std::vector<int32_t>> copies((size_t)d->n_if);
        int64_t last = -1;
        if (d->n_if > 0) {
            for (int64_t l = 0; l < c->L; ++l) {
                const int64_t id = glo_num[l];
                const int64_t i = node_of(id);
                if (i < d->n_if && iface[(size_t)i] == id) { copies[(size_t)i].push_back((int32_t)l); last = l; }
            }
        }
        d->n_iface_elems = last < 0 ? 0 : last / c->P + 1;
        std::vector<int32_t> cp_off(1, 0), cp_idx, snd_off(1, 0), snd_pos, src_off(1, 0), src;
        for (int64_t i = 0; i < d->n_if; ++i) {
            if (copies[(size_t)i].empty()) return NK_ERR_ARG;            // a candidate id that is not in glo_num
            cp_idx.insert(cp_idx.end(), copies[(size_t)i].begin(), copies[(size_t)i].end());
            cp_off.push_back((int32_t)cp_idx.size());
            snd_pos.insert(snd_pos.end(), snd[(size_t)i].begin(), snd[(size_t)i].end());
            snd_off.push_back((int32_t)snd_pos.size());
            for (const auto &h : holders[(size_t)i]) src.push_back(h.second);
            src_off.push_back((int32_t)src.size());
        }
        d->n_copies = (int64_t)cp_idx.size();
        NK_CUDA(upload(&d->cp_off, cp_off));
        NK_CUDA(upload(&d->cp_idx, cp_idx));
        NK_CUDA(upload(&d->snd_off, snd_off));
        NK_CUDA(upload(&d->snd_pos, snd_pos));
        NK_CUDA(upload(&d->src_off, src_off));
        NK_CUDA(upload(&d->src, src));
        NK_CUDA(cudaMalloc(reinterpret_cast<void **>(&d->own), std::max<size_t>((size_t)d->n_if, 1) * sizeof(double)));
        NK_CUDA(cudaMalloc(reinterpret_cast<void **>(&d->tmp), 4 * sizeof(double)));
        NK_CUDA(cudaStreamCreateWithFlags(&d->comm, cudaStreamNonBlocking));
        NK_CUDA(cudaEventCreateWithFlags(&d->ev_packed, cudaEventDisableTiming));
        NK_CUDA(cudaEventCreateWithFlags(&d->ev_halo, cudaEventDisableTiming));
    } catch (const std::bad_alloc &) {
        return NK_ERR_ALLOC;
    }
    return NK_OK;
}

int nk_dist_info(nk_ctx *c, int *n_neighbors, int64_t *n_exchange, int64_t *n_interface_nodes, int64_t *n_interface_elements)
{
    if (!c || !c->dist) return NK_ERR_ARG;
    if (n_neighbors) *n_neighbors = (int)c->dist->nbr_rank.size();
    if (n_exchange) *n_exchange = c->dist->n_send;
    if (n_interface_nodes) *n_interface_nodes = c->dist->n_if;
    if (n_interface_elements) *n_interface_elements = c->dist->n_iface_elems;
    return NK_OK;
}

int nk_dist_neighbors(nk_ctx *c, int *ranks, int64_t *offsets, int64_t *counts)
{
    if (!c || !c->dist || !ranks || !offsets || !counts) return NK_ERR_ARG;
    for (size_t k = 0; k < c->dist->nbr_rank.size(); ++k) {
        ranks[k] = c->dist->nbr_rank[k];
        offsets[k] = c->dist->nbr_off[k];
        counts[k] = c->dist->nbr_cnt[k];
    }
    return NK_OK;
}

int nk_dist_set_buffers(nk_ctx *c, double *send_dev, double *recv_dev, double *scalar_send_dev, double *scalar_gathered_dev)
{
    if (!c || !c->dist || !scalar_send_dev || !scalar_gathered_dev) return NK_ERR_ARG;
    if (c->dist->n_send > 0 && (!send_dev || !recv_dev)) return NK_ERR_ARG;
    c->dist->send = send_dev; c->dist->recv = recv_dev;
    c->dist->ssend = scalar_send_dev; c->dist->sgath = scalar_gathered_dev;
    return NK_OK;
}

int nk_dist_set_mult(nk_ctx *c, const double *mult_dev, void *stream)
{
    if (!c || !mult_dev) return NK_ERR_ARG;
    if (c->dist && c->dist->world == 1) return NK_OK;   // one rank: the local multiplicities ARE the global ones
    cudaStream_t st = S(stream);
    // table by value: ctab[t] = 1/t, mtab[t] = t (the set-up's table lists the LOCAL multiplicities only)
    double tab[2 * NK_CTAB];
    tab[0] = 0.0; tab[NK_CTAB] = 0.0;
    for (int t = 1; t < NK_CTAB; ++t) { tab[t] = 1.0 / (double)t; tab[NK_CTAB + t] = (double)t; }
    NK_CUDA(cudaMemsetAsync(c->errflag, 0, sizeof(int), st));
    NK_CUDA(cudaMemcpyAsync(c->ctab, tab, sizeof(tab), cudaMemcpyHostToDevice, st));   // mtab follows ctab
    dist_set_mult_kernel<<<blocks_for(c->L), DIST_THREADS, 0, st>>>(c->code, mult_dev, c->L, c->errflag);
    NK_CUDA(cudaGetLastError());
    int flag = 0;
    NK_CUDA(cudaMemcpyAsync(&flag, c->errflag, sizeof(int), cudaMemcpyDeviceToHost, st));
    NK_CUDA(cudaStreamSynchronize(st));                 // set-up call: `tab` and `flag` live on this stack
    c->have_dinv = 0;
    c->dist_mult = 1;                                    // the weights are global now: the rank-local fused paths are off
    return flag ? NK_ERR_MULT : NK_OK;
}

int nk_dist_gs(nk_ctx *c, double *v, int with_mask, nk_exchange_fn fn, void *user, void *stream)
{
    if (!ready(c) || !v || !nk_aligned16(v)) return NK_ERR_ARG;
    return dist_gs(c, v, with_mask, fn, user, S(stream));
}

int nk_dist_dot(nk_ctx *c, const double *a, const double *b, double *out_dev, nk_exchange_fn fn, void *user, void *stream)
{
    if (!ready(c) || !a || !b || !out_dev || !nk_aligned16(a) || !nk_aligned16(b)) return NK_ERR_ARG;
    cudaStream_t st = S(stream);
    NK_CUDA(nk_launch_dot(c, a, b, c->dist->ssend, NK_EPI_STORE, st));
    const int rc = exchange(c, fn, user, XCH_SCALAR, st);
    if (rc != NK_OK) return rc;
    NK_CUDA(launch_finish(c, NK_EPI_STORE, out_dev, st));
    return NK_OK;
}

int nk_dist_cg(nk_ctx *c, const double *f, double *x, int niter, double *hist, nk_exchange_fn fn, void *user, void *stream)
{
    if (!ready(c) || !f || !x || !hist || niter < 0 || f == x || !nk_aligned16(f) || !nk_aligned16(x)) return NK_ERR_ARG;
    nk_dist *d = c->dist;
    cudaStream_t st = S(stream);
    if (d->world == 1) return nk_cg(c, f, x, niter, hist, stream);      // one rank: the single-GPU solver, all of it
    c->p_pending = 0;
    c->w_unsummed = 0;
    int rc;
    // r = mask o f, x = 0, p = r; rho = <r,r>_c over all ranks
    NK_CUDA(with_raw(c, d->ssend, [&] { return nk_launch_cg_init(c, f, x, c->res_dummy, st); }));
    if ((rc = exchange(c, fn, user, XCH_SCALAR, st)) != NK_OK) return rc;
    NK_CUDA(launch_finish(c, NK_EPI_RHO0, hist, st));
    const int64_t e_if = d->n_iface_elems, e_in = c->E - d->n_iface_elems;
    for (int k = 1; k <= niter; ++k) {
        // interface elements first; their partial sums go out while ax_e runs on the interior elements.
        // pap = sum over ALL ranks' elements of grad(p)^T G grad(p): element-local, so launch and rank totals just add
        NK_CUDA(with_raw(c, d->tmp, [&] { return nk_launch_ax_tma_range(c, nullptr, c->p, nullptr, c->w, 1, 0, e_if, st); }));
        NK_CUDA(launch_partial(c, c->w, st));
        NK_CUDA(cudaEventRecord(d->ev_packed, st));
        NK_CUDA(cudaStreamWaitEvent(d->comm, d->ev_packed, 0));
        if ((rc = exchange(c, fn, user, XCH_HALO, d->comm)) != NK_OK) return rc;
        NK_CUDA(cudaEventRecord(d->ev_halo, d->comm));
        if (e_in > 0) {
            NK_CUDA(with_raw(c, d->tmp + 1, [&] { return nk_launch_ax_tma_range(c, nullptr, c->p, nullptr, c->w, 1, e_if, e_in, st); }));
            dist_add2_kernel<<<1, 1, 0, st>>>(d->tmp, d->tmp + 1, d->ssend);
        } else {
            NK_CUDA(cudaMemcpyAsync(d->ssend, d->tmp, sizeof(double), cudaMemcpyDeviceToDevice, st));
        }
        if (e_if == 0) NK_CUDA(cudaMemcpyAsync(d->ssend, d->tmp + 1, sizeof(double), cudaMemcpyDeviceToDevice, st));
        NK_CUDA(cudaGetLastError());
        if ((rc = exchange(c, fn, user, XCH_SCALAR, st)) != NK_OK) return rc;
        NK_CUDA(launch_finish(c, NK_EPI_PAP, c->res_dummy, st));
        NK_CUDA(nk_launch_gs(c, c->w, 1, st));                                  // this rank's own sums (and the mask)
        NK_CUDA(cudaStreamWaitEvent(st, d->ev_halo, 0));
        NK_CUDA(launch_unpack(c, c->w, 1, st));                                 // the totals over all holders
        NK_CUDA(with_raw(c, d->ssend, [&] { return nk_launch_update_r(c, c->res_dummy, 0, st); }));
        if ((rc = exchange(c, fn, user, XCH_SCALAR, st)) != NK_OK) return rc;
        NK_CUDA(launch_finish(c, NK_EPI_RHO, hist + k, st));
        NK_CUDA(nk_launch_update_px(c, x, st));
    }
    return NK_OK;
}

}  // extern "C"
