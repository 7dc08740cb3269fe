// nk_host.h -- host-side helpers shared by nk_api.cu and nk_setup.cu (product code only).
#pragma once
#include <cstdint>
#include <vector>

#include "nk_internal.h"

void nk_set_last_cuda(int e);

inline int nk_cuda_fail(cudaError_t e)
{
    nk_set_last_cuda((int)e);
    return NK_ERR_CUDA;
}
#define NK_CUDA(call)                                      \
    do {                                                   \
        cudaError_t e__ = (call);                          \
        if (e__ != cudaSuccess) return nk_cuda_fail(e__);  \
    } while (0)

inline size_t nk_align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline bool nk_aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

struct nk_carve {
    size_t g, vec, code, off, idx, nbr, gx, pk, tabs, partials, hist, scal, small, total;
};

// Worst case: every local point listed in the gs plan (n_listed <= L, n_rows <= L).
inline nk_carve nk_carve_sizes(int64_t L)
{
    nk_carve c;
    c.g = nk_align_up(3 * (size_t)L * sizeof(double2), 256);      // all six factors
    c.vec = nk_align_up((size_t)L * sizeof(double), 256);         // x9 (r, p, w, hf, hx, dinv, hf2, hx2, p2)
    c.code = nk_align_up((size_t)L, 256);
    c.off = nk_align_up(((size_t)L + 1) * sizeof(int32_t), 256);
    c.idx = nk_align_up((size_t)L * sizeof(int32_t), 256);
    c.nbr = nk_align_up((size_t)L * sizeof(int32_t), 256);         // per-point gather code of the fused gs (nk_ctx::nbr)
    // its side table: rows of 3 or more copies, at most 8 ints per 3 listed points (header + alignment),
    c.gx = nk_align_up((9 * ((size_t)L / 3 + 1) + 16 + 65536 + 8) * sizeof(int32_t), 256);   // + one int per such row (gx_rows)
                                                                                  // + the per-block cut of that list (gx_blk)
    // packed rows (<= L indices + 16 padding ints per chunk) and 8 ints of descriptor per chunk
    c.pk = nk_align_up(((size_t)L + 24 * ((size_t)L / (2 * NK_GS_CHUNK) + 2) + 256) * sizeof(int32_t), 256);
    c.tabs = nk_align_up(2 * NK_CTAB * sizeof(double) + (16 * 16 + 16) * sizeof(double), 256);
    c.partials = nk_align_up(NK_MAX_PARTIALS * sizeof(double), 256);
    c.hist = nk_align_up(NK_HIST_MAX * sizeof(double), 256);
    c.scal = 256;
    c.small = 256;                                                // counter, errflag, res_dummy
    c.total = c.g + 9 * c.vec + c.code + c.off + c.idx + c.nbr + c.gx + c.pk + c.tabs + c.partials + 2 * c.hist + c.scal + c.small;
    return c;
}

inline bool nk_valid_EN(int64_t E, int N, int64_t *L_out)
{
    if (E <= 0 || N < 1 || N > NK_MAX_ORDER) return false;
    const int64_t n = N + 1, P = n * n * n;
    if (E > ((int64_t)1 << 31) / P) return false;
    const int64_t L = E * P;
    if (L >= ((int64_t)1 << 31)) return false;
    *L_out = L;
    return true;
}
