// nk_gs.cu -- gather-scatter (direct-stiffness sum Q Q^T) fused with the Dirichlet mask
// (one work-item per unique shared node, its inner loops over the copies run in
// order; S 8(a) a2-a3; BJ north_star (2): CSR of sorted global ids, atomic-free segmented sum,
// then scatter, fused with the mask).
//
// Plan built by nk_setup: CSR rows over unique nodes that are shared and unmasked ("sum rows",
// [0, n_sum_rows)) followed by rows of masked nodes; inside a row the local indices ascend, so the
// sum order equals the ascending-local-index order of S 8(c) O4.  Rows are ordered by their first
// local index so that neighbouring threads touch neighbouring memory.
//   with_mask = 1:  sum rows are summed and scattered; every listed copy of a masked node gets 0
//                   (one thread per listed copy -- a flat, coalesced index stream);
//   with_mask = 0:  masked rows are summed like the others (rows of length 1 are a no-op).
#include "nk_internal.h"

namespace {

constexpr int GS_THREADS = 256;

__device__ __forceinline__ void gs_row(double *__restrict__ v, const int32_t *__restrict__ idx, int b, int e)
{
    // Rows are short (2, 4, 8 copies on a conforming hex mesh): issue the gathers first.
    const int len = e - b;
    if (len == 2) {
        const int i0 = idx[b], i1 = idx[b + 1];
        const double s = v[i0] + v[i1];
        v[i0] = s; v[i1] = s;
    } else if (len == 4) {
        const int i0 = idx[b], i1 = idx[b + 1], i2 = idx[b + 2], i3 = idx[b + 3];
        const double a0 = v[i0], a1 = v[i1], a2 = v[i2], a3 = v[i3];
        const double s = ((a0 + a1) + a2) + a3;
        v[i0] = s; v[i1] = s; v[i2] = s; v[i3] = s;
    } else if (len == 8) {
        int ii[8];
        double a[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) ii[j] = idx[b + j];
#pragma unroll
        for (int j = 0; j < 8; ++j) a[j] = v[ii[j]];
        double s = a[0];
#pragma unroll
        for (int j = 1; j < 8; ++j) s += a[j];
#pragma unroll
        for (int j = 0; j < 8; ++j) v[ii[j]] = s;
    } else {
        double s = 0.0;
        for (int j = b; j < e; ++j) s += v[idx[j]];
        for (int j = b; j < e; ++j) v[idx[j]] = s;
    }
}

__global__ void __launch_bounds__(GS_THREADS)
gs_kernel(double *__restrict__ v, const int32_t *__restrict__ off, const int32_t *__restrict__ idx,
          int n_sum_rows, int n_rows, int masked_begin, int n_listed, int with_mask)
{
    const int t = blockIdx.x * GS_THREADS + threadIdx.x;
    if (t < n_sum_rows) {
        gs_row(v, idx, off[t], off[t + 1]);
    } else if (with_mask) {
        const int q = masked_begin + (t - n_sum_rows);
        if (q < n_listed) v[idx[q]] = 0.0;
    } else {
        if (t < n_rows) {
            const int b = off[t], e = off[t + 1];
            if (e - b > 1) gs_row(v, idx, b, e);
        }
    }
}

}  // namespace

cudaError_t nk_launch_gs(nk_ctx *c, double *v, int with_mask, cudaStream_t st)
{
    const int64_t masked_listed = c->n_listed - c->n_sum_listed;
    const int64_t work = with_mask ? c->n_sum_rows + masked_listed : c->n_rows;
    if (work <= 0) return cudaSuccess;
    const int nb = (int)((work + GS_THREADS - 1) / GS_THREADS);
    gs_kernel<<<nb, GS_THREADS, 0, st>>>(v, c->row_off, c->row_idx, (int)c->n_sum_rows, (int)c->n_rows,
                                         (int)c->n_sum_listed, (int)c->n_listed, with_mask);
    c->launches++;
    return cudaGetLastError();
}
