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
    const int32_t *pk, *desc, *off, *idx;
    int n_chunks;                     // chunks of NK_GS_CHUNK summed rows, BPC blocks each
    int n_sum_rows, n_rows;           // CSR: rows [0, n_sum_rows) summed, [n_sum_rows, n_rows) masked nodes
    int masked_begin, n_listed;       // the masked nodes' copies are idx[masked_begin, n_listed)
};

constexpr int BPC = NK_GS_CHUNK / GS_THREADS;     // blocks per chunk

// Rows of 2, 4 and 8 copies (faces, edges, corners) come from the packed arrays: one vector load
// of the indices, no offset lookup -- one dependent memory round trip less than the CSR walk, on
// a kernel that is pure latency (ncu: 52 % of DRAM peak at 82 % occupancy, all long-scoreboard).
// Packing is per chunk of consecutive rows, so that rows of different length that share 32-byte
// sectors are still worked on at about the same time (packing the whole mesh by length made
// DRAM traffic grow from 0.90 to 1.11 GB at config 5).  Sums run in ascending local index, as in gs_row.
__global__ void __launch_bounds__(GS_THREADS)
gs_kernel(double *__restrict__ v, gs_plan pl, int with_mask)
{
    nk_pdl_launch_dependents();            // the next kernel may queue up behind us (we are a dependent ourselves in pdl mode 2)
    const int chunk = blockIdx.x / BPC;
    if (chunk < pl.n_chunks) {
        const int4 d = reinterpret_cast<const int4 *>(pl.desc)[2 * chunk];       // offset, n2, n4, n8
        const int n_other = pl.desc[8 * chunk + 4];
        int t = (blockIdx.x - chunk * BPC) * GS_THREADS + threadIdx.x;
        const int32_t *pk2 = pl.pk + d.x;
        const int32_t *pk4 = pk2 + ((2 * d.y + 3) & ~3);
        const int32_t *pk8 = pk4 + 4 * d.z;
        const int32_t *oth = pk8 + 8 * d.w;
        nk_pdl_wait();                     // the plan is static; v is what the predecessor wrote
        if (t < d.y) {
            const int2 ii = reinterpret_cast<const int2 *>(pk2)[t];
            const double s = v[ii.x] + v[ii.y];
            v[ii.x] = s; v[ii.y] = s;
            return;
        }
        t -= d.y;
        if (t < d.z) {
            const int4 ii = reinterpret_cast<const int4 *>(pk4)[t];
            const double a0 = v[ii.x], a1 = v[ii.y], a2 = v[ii.z], a3 = v[ii.w];
            const double s = ((a0 + a1) + a2) + a3;
            v[ii.x] = s; v[ii.y] = s; v[ii.z] = s; v[ii.w] = s;
            return;
        }
        t -= d.z;
        if (t < d.w) {
            const int4 ia = reinterpret_cast<const int4 *>(pk8)[2 * t], ib = reinterpret_cast<const int4 *>(pk8)[2 * t + 1];
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
        t -= d.w;
        if (t < n_other) {
            const int row = oth[t];
            gs_row(v, pl.idx, pl.off[row], pl.off[row + 1]);
        }
        return;
    }
    const int t = (blockIdx.x - pl.n_chunks * BPC) * GS_THREADS + threadIdx.x;
    nk_pdl_wait();
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
    const int64_t nb = c->n_gs_chunks * BPC + (tail + GS_THREADS - 1) / GS_THREADS;
    if (nb <= 0) return cudaSuccess;
    gs_plan pl;
    pl.pk = c->pk; pl.desc = c->gs_desc; pl.off = c->row_off; pl.idx = c->row_idx;
    pl.n_chunks = (int)c->n_gs_chunks;
    pl.n_sum_rows = (int)c->n_sum_rows; pl.n_rows = (int)c->n_rows;
    pl.masked_begin = (int)c->n_sum_listed; pl.n_listed = (int)c->n_listed;
    // a programmatic dependent only in pdl mode 2 (the default up to 2^24 points, where the launch gap saved
    // matters more): on large meshes its blocks would land on SMs still carved out for ax_e's 227 KB of shared
    // memory (L1 of ~1 KB) and the gathers would miss it (measured: +95 us at config 5)
    cudaError_t e = nk_launch(gs_kernel, (unsigned)nb, GS_THREADS, 0, st, c->pdl_now == 2, v, pl, with_mask);
    c->launches++;
    return e != cudaSuccess ? e : cudaGetLastError();
}
