// nk_dist.cu -- the CG iteration over an element partition: one rank per GPU (
// PAPER.md:336 "MPI ... future work").  ax_e and the vector updates are rank-local.  gs needs ONE exchange:
// every rank sums its own copies (nk_launch_gs), packs one value per INTERFACE node (a global id held by more
// than one rank) into a send buffer, the buffers of all ranks are all-gathered (the caller's collective: NCCL
// through torch.distributed on the same stream), and every rank adds the `world` partial sums IN RANK ORDER and
// writes the total to all its copies -- so all ranks hold bitwise the same value.  The two dot products travel
// the same way: the reducing kernel stores its rank-local total (nk_reduce_ws::raw) instead of running the
// epilogue, the totals are all-gathered (pap rides in the last slot of the gs buffer), and one thread adds them
// in rank order and runs the epilogue that the single-GPU kernels run in their last block.
//
// The library only enqueues kernels; between the calls marked [all-gather] the caller runs the collective on
// the same stream.  No call here synchronises.
#include "nk_internal.h"
#include "nk_host.h"
#include "nk_reduce.cuh"
#include "../../include/nk.h"

namespace {

constexpr int DIST_THREADS = 256;

inline cudaStream_t S(void *stream) { return reinterpret_cast<cudaStream_t>(stream); }

__global__ void __launch_bounds__(DIST_THREADS)
dist_pack_kernel(const double *__restrict__ v, const int32_t *__restrict__ pack, int64_t n_slots, double *__restrict__ send)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_slots) return;
    const int32_t l = pack[i];
    send[i] = l >= 0 ? v[l] : 0.0;                     // a node this rank does not hold contributes 0
}

__global__ void __launch_bounds__(DIST_THREADS)
dist_unpack_kernel(double *__restrict__ v, const int32_t *__restrict__ uloc, const int32_t *__restrict__ uslot,
                   int64_t n_unpack, const double *__restrict__ gath, int64_t stride, int world)
{
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_unpack) return;
    const int32_t slot = uslot[j];
    double s = 0.0;
    for (int r = 0; r < world; ++r) s += gath[(int64_t)r * stride + slot];    // rank order: same bits everywhere
    v[uloc[j]] = s;
}

// one thread: total over ranks in rank order, then the epilogue of nk_reduce.cuh
__global__ void dist_finish_kernel(int epi, const double *__restrict__ gath, int64_t stride, int world, double *scal,
                                   double *out)
{
    double t = 0.0;
    for (int r = 0; r < world; ++r) t += gath[(int64_t)r * stride];
    nk_epilogue(epi, t, scal, out);
}

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

inline unsigned blocks_for(int64_t n) { return (unsigned)((n + DIST_THREADS - 1) / DIST_THREADS); }

cudaError_t launch_pack(nk_ctx *c, const double *v, cudaStream_t st)
{
    if (c->dist_slots == 0) return cudaSuccess;
    dist_pack_kernel<<<blocks_for(c->dist_slots), DIST_THREADS, 0, st>>>(v, c->dist_pack, c->dist_slots, c->dist_send);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_unpack(nk_ctx *c, double *v, cudaStream_t st)
{
    if (c->dist_n_unpack == 0) return cudaSuccess;
    dist_unpack_kernel<<<blocks_for(c->dist_n_unpack), DIST_THREADS, 0, st>>>(v, c->dist_uloc, c->dist_uslot, c->dist_n_unpack,
                                                                             c->dist_gath, c->dist_slots + 1, c->dist_world);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_finish(nk_ctx *c, int epi, const double *gath, int64_t stride, double *out, cudaStream_t st)
{
    dist_finish_kernel<<<1, 1, 0, st>>>(epi, gath, stride, c->dist_world, c->red.scal, out);
    c->launches++;
    return cudaGetLastError();
}

// runs `call` with the reducing kernel's total redirected to `raw`
template <typename F>
cudaError_t with_raw(nk_ctx *c, double *raw, F call)
{
    c->red.raw = raw;
    const cudaError_t e = call();
    c->red.raw = nullptr;
    return e;
}

inline bool attached(const nk_ctx *c) { return c && c->dist_world > 0; }

}  // namespace

extern "C" {

int nk_dist_attach(nk_ctx *c, int rank, int world, int64_t n_slots, const int32_t *pack_dev, int64_t n_unpack,
                   const int32_t *unpack_loc_dev, const int32_t *unpack_slot_dev, double *send_dev, double *gathered_dev,
                   double *scalar_send_dev, double *scalar_gathered_dev)
{
    if (!c || world < 1 || rank < 0 || rank >= world || n_slots < 0 || n_unpack < 0) return NK_ERR_ARG;
    if (n_slots > 0 && !pack_dev) return NK_ERR_ARG;
    if (n_unpack > 0 && (!unpack_loc_dev || !unpack_slot_dev)) return NK_ERR_ARG;
    if (!send_dev || !gathered_dev || !scalar_send_dev || !scalar_gathered_dev) return NK_ERR_ARG;
    c->dist_rank = rank; c->dist_world = world;
    c->dist_slots = n_slots; c->dist_n_unpack = n_unpack;
    c->dist_pack = pack_dev; c->dist_uloc = unpack_loc_dev; c->dist_uslot = unpack_slot_dev;
    c->dist_send = send_dev; c->dist_gath = gathered_dev;
    c->dist_ssend = scalar_send_dev; c->dist_sgath = scalar_gathered_dev;
    return NK_OK;
}

int nk_dist_set_mult(nk_ctx *c, const double *mult_dev, void *stream)
{
    if (!c || !mult_dev) return NK_ERR_ARG;
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
    return flag ? NK_ERR_MULT : NK_OK;
}

int nk_dist_gs_begin(nk_ctx *c, double *v, int with_mask, void *stream)
{
    if (!attached(c) || !v) return NK_ERR_ARG;
    NK_CUDA(nk_launch_gs(c, v, with_mask, S(stream)));
    NK_CUDA(launch_pack(c, v, S(stream)));
    return NK_OK;
}

int nk_dist_gs_end(nk_ctx *c, double *v, void *stream)
{
    if (!attached(c) || !v) return NK_ERR_ARG;
    NK_CUDA(launch_unpack(c, v, S(stream)));
    return NK_OK;
}

int nk_dist_dot_begin(nk_ctx *c, const double *a, const double *b, void *stream)
{
    if (!attached(c) || !a || !b || !nk_aligned16(a) || !nk_aligned16(b)) return NK_ERR_ARG;
    NK_CUDA(nk_launch_dot(c, a, b, c->dist_ssend, NK_EPI_STORE, S(stream)));
    return NK_OK;
}

int nk_dist_dot_end(nk_ctx *c, double *out_dev, void *stream)
{
    if (!attached(c) || !out_dev) return NK_ERR_ARG;
    NK_CUDA(launch_finish(c, NK_EPI_STORE, c->dist_sgath, 1, out_dev, S(stream)));
    return NK_OK;
}

int nk_dist_cg_begin(nk_ctx *c, const double *f, double *x, void *stream)
{
    if (!attached(c) || !f || !x || f == x || !nk_aligned16(f) || !nk_aligned16(x)) return NK_ERR_ARG;
    c->p_pending = 0;
    cudaStream_t st = S(stream);
    NK_CUDA(with_raw(c, c->dist_ssend, [&] { return nk_launch_cg_init(c, f, x, c->res_dummy, st); }));
    return NK_OK;
}

int nk_dist_cg_begin_end(nk_ctx *c, double *hist0_dev, void *stream)
{
    if (!attached(c) || !hist0_dev) return NK_ERR_ARG;
    NK_CUDA(launch_finish(c, NK_EPI_RHO0, c->dist_sgath, 1, hist0_dev, S(stream)));
    return NK_OK;
}

int nk_dist_iter_a(nk_ctx *c, void *stream)
{
    if (!attached(c)) return NK_ERR_ARG;
    cudaStream_t st = S(stream);
    c->w_unsummed = 0;
    // pap = sum over ALL ranks' elements of grad(p)^T G grad(p): element-local, so the rank totals just add
    NK_CUDA(with_raw(c, c->dist_send + c->dist_slots,
                     [&] { return nk_launch_ax_tma(c, nullptr, c->p, nullptr, c->w, 1, st); }));
    NK_CUDA(nk_launch_gs(c, c->w, 1, st));
    NK_CUDA(launch_pack(c, c->w, st));
    return NK_OK;
}

int nk_dist_iter_b(nk_ctx *c, void *stream)
{
    if (!attached(c)) return NK_ERR_ARG;
    cudaStream_t st = S(stream);
    NK_CUDA(launch_unpack(c, c->w, st));
    NK_CUDA(launch_finish(c, NK_EPI_PAP, c->dist_gath + c->dist_slots, c->dist_slots + 1, c->res_dummy, st));
    NK_CUDA(with_raw(c, c->dist_ssend, [&] { return nk_launch_update_r(c, c->res_dummy, 0, st); }));
    return NK_OK;
}

int nk_dist_iter_c(nk_ctx *c, double *x, double *hist_k_dev, void *stream)
{
    if (!attached(c) || !x || !hist_k_dev || !nk_aligned16(x)) return NK_ERR_ARG;
    cudaStream_t st = S(stream);
    NK_CUDA(launch_finish(c, NK_EPI_RHO, c->dist_sgath, 1, hist_k_dev, st));
    NK_CUDA(nk_launch_update_px(c, x, st));
    return NK_OK;
}

}  // extern "C"
