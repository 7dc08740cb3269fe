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

struct gs_plan {
    const int32_t *pk2, *pk4, *pk8, *other, *off, *idx;
    int n2, n4, n8, n_other;          // summed rows by length class
    int n_sum_rows, n_rows;           // CSR: rows [0, n_sum_rows) summed, [n_sum_rows, n_rows) masked nodes
    int masked_begin, n_listed;       // the masked nodes' copies are idx[masked_begin, n_listed)
};

// Rows of 2, 4 and 8 copies (faces, edges, corners) come from the packed arrays: one vector load
// of the indices, no offset lookup -- one dependent memory round trip less than the CSR walk, on
// a kernel that is pure latency (ncu: 52 % of DRAM peak at 82 % occupancy, all long-scoreboard).
// Sums run in ascending local index, as in gs_row.
__global__ void __launch_bounds__(GS_THREADS)
gs_kernel(double *__restrict__ v, gs_plan pl, int with_mask)
{
    int t = blockIdx.x * GS_THREADS + threadIdx.x;
    if (t < pl.n2) {
        const int2 ii = reinterpret_cast<const int2 *>(pl.pk2)[t];
        const double s = v[ii.x] + v[ii.y];
        v[ii.x] = s; v[ii.y] = s;
        return;
    }
    t -= pl.n2;
    if (t < pl.n4) {
        const int4 ii = reinterpret_cast<const int4 *>(pl.pk4)[t];
        const double a0 = v[ii.x], a1 = v[ii.y], a2 = v[ii.z], a3 = v[ii.w];
        const double s = ((a0 + a1) + a2) + a3;
        v[ii.x] = s; v[ii.y] = s; v[ii.z] = s; v[ii.w] = s;
        return;
    }
    t -= pl.n4;
    if (t < pl.n8) {
        const int4 ia = reinterpret_cast<const int4 *>(pl.pk8)[2 * t], ib = reinterpret_cast<const int4 *>(pl.pk8)[2 * t + 1];
        const int ii[8] = {ia.x, ia.y, ia.z, ia.w, ib.x, ib.y, ib.z, ib.w};
        double a[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) a[j] = v[ii[j]];
        double s = a[0];
#pragma unroll
        for (int j = 1; j < 8; ++j) s += a[j];
#pragma unroll
        for (int j = 0; j < 8; ++j) v[ii[j]] = s;
        return;
    }
    t -= pl.n8;
    if (t < pl.n_other) {
        const int row = pl.other[t];
        gs_row(v, pl.idx, pl.off[row], pl.off[row + 1]);
        return;
    }
    t -= pl.n_other;
    if (with_mask) {
        const int q = pl.masked_begin + t;
        if (q < pl.n_listed) v[pl.idx[q]] = 0.0;
    } else {
        const int row = pl.n_sum_rows + t;
        if (row < pl.n_rows) {
            const int b = pl.off[row], e = pl.off[row + 1];
            if (e - b > 1) gs_row(v, pl.idx, b, e);
        }
    }
}

}  // namespace

cudaError_t nk_launch_gs(nk_ctx *c, double *v, int with_mask, cudaStream_t st)
{
    const int64_t masked_listed = c->n_listed - c->n_sum_listed;
    const int64_t tail = with_mask ? masked_listed : c->n_rows - c->n_sum_rows;
    const int64_t work = c->n_sum_rows + tail;
    if (work <= 0) return cudaSuccess;
    gs_plan pl;
    pl.pk2 = c->pk2; pl.pk4 = c->pk4; pl.pk8 = c->pk8; pl.other = c->other_rows;
    pl.off = c->row_off; pl.idx = c->row_idx;
    pl.n2 = (int)c->n2; pl.n4 = (int)c->n4; pl.n8 = (int)c->n8; pl.n_other = (int)c->n_other;
    pl.n_sum_rows = (int)c->n_sum_rows; pl.n_rows = (int)c->n_rows;
    pl.masked_begin = (int)c->n_sum_listed; pl.n_listed = (int)c->n_listed;
    const int nb = (int)((work + GS_THREADS - 1) / GS_THREADS);
    gs_kernel<<<nb, GS_THREADS, 0, st>>>(v, pl, with_mask);
    c->launches++;
    return cudaGetLastError();
}
