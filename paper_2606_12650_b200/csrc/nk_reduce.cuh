// nk_reduce.cuh -- deterministic block reduction + ordered "last block" finish (S 8(a) a7;
// P:312 "tree reduction" in the group; BJ "warp-shuffle and block reductions and a deterministic
// two-pass finish").  No floating-point atomics: every block stores its partial, the block that
// draws the last ticket (integer atomicInc, self-resetting) re-reads ALL partials in index order
// and reduces them with the same fixed tree, so the total does not depend on which block is last.
#pragma once
#include "nk_internal.h"

__device__ __forceinline__ double nk_warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum over the block; result valid in thread 0.  `sm` needs >= 32 doubles.  blockDim.x <= 1024.
__device__ __forceinline__ double nk_block_sum(double v, double *sm)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int nw = (blockDim.x + 31) >> 5;
    v = nk_warp_sum(v);
    __syncthreads();                 // protect sm against a previous use
    if (lane == 0) sm[wid] = v;
    __syncthreads();
    double t = 0.0;
    if (wid == 0) {
        t = (lane < nw) ? sm[lane] : 0.0;
        t = nk_warp_sum(t);
    }
    return t;
}

__device__ __forceinline__ void nk_epilogue(int epi, double total, double *scal, double *out)
{
    if (epi == NK_EPI_STORE) {
        out[0] = total;
    } else if (epi == NK_EPI_RHO0) {
        scal[NK_S_RHO] = total;
        scal[NK_S_RHO_OLD] = total;
        scal[NK_S_BETA] = 0.0;
        scal[NK_S_ALPHA] = 0.0;
        scal[NK_S_PAP] = 0.0;
        scal[NK_S_RHO_NEW] = total;
        out[0] = sqrt(total);
    } else if (epi == NK_EPI_PAP) {
        const double rho = scal[NK_S_RHO];
        scal[NK_S_PAP] = total;
        scal[NK_S_ALPHA] = (rho == 0.0 || total == 0.0) ? 0.0 : rho / total;
    } else {   // NK_EPI_RHO
        const double rho = scal[NK_S_RHO], pap = scal[NK_S_PAP];
        scal[NK_S_RHO_NEW] = total;
        scal[NK_S_BETA] = (rho == 0.0 || pap == 0.0) ? 0.0 : total / rho;
        scal[NK_S_RHO_OLD] = rho;
        scal[NK_S_RHO] = total;
        out[0] = sqrt(total);
    }
}

// Called by ALL threads of every block with the block's contribution `v` (per thread).
// `sm` >= 33 doubles of shared memory.
__device__ __forceinline__ void nk_grid_reduce(double v, double *sm, nk_reduce_ws ws, int epi, double *out)
{
    const double bs = nk_block_sum(v, sm);
    __shared__ int s_last;
    const unsigned nb = gridDim.x;
    if (threadIdx.x == 0) {
        ws.partials[blockIdx.x] = bs;
        __threadfence();
        const unsigned ticket = atomicInc(ws.counter, nb - 1u);   // wraps to 0 after the last block
        s_last = (ticket == nb - 1u);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double t = 0.0;
    for (unsigned i = threadIdx.x; i < nb; i += blockDim.x) t += __ldcg(ws.partials + i);
    t = nk_block_sum(t, sm);
    if (threadIdx.x == 0) {
        if (ws.raw) ws.raw[0] = t;              // distributed: the epilogue runs after the all-gather (nk_dist.cu)
        else nk_epilogue(epi, t, ws.scal, out);
    }
}

// Two sums at once (preconditioned CG: <r,z>_c and <r,r>_c in one pass).  Partials of the second sum
// live in the upper half of the partials buffer.  Epilogue: rho' = t1 (beta = rho'/rho, guarded),
// out[0] = sqrt(t2); `first` marks the initial call (rho = t1, beta = 0).
__device__ __forceinline__ void nk_grid_reduce2(double v1, double v2, double *sm, nk_reduce_ws ws, int first, double *out)
{
    const double b1 = nk_block_sum(v1, sm);
    const double b2 = nk_block_sum(v2, sm);
    __shared__ int s_last2;
    const unsigned nb = gridDim.x;
    double *part2 = ws.partials + NK_MAX_PARTIALS / 2;
    if (threadIdx.x == 0) {
        ws.partials[blockIdx.x] = b1;
        part2[blockIdx.x] = b2;
        __threadfence();
        const unsigned ticket = atomicInc(ws.counter, nb - 1u);
        s_last2 = (ticket == nb - 1u);
    }
    __syncthreads();
    if (!s_last2) return;
    __threadfence();
    double t1 = 0.0, t2 = 0.0;
    for (unsigned i = threadIdx.x; i < nb; i += blockDim.x) { t1 += __ldcg(ws.partials + i); t2 += __ldcg(part2 + i); }
    t1 = nk_block_sum(t1, sm);
    t2 = nk_block_sum(t2, sm);
    if (threadIdx.x == 0) {
        double *scal = ws.scal;
        if (first) {
            scal[NK_S_RHO] = t1; scal[NK_S_RHO_OLD] = t1; scal[NK_S_RHO_NEW] = t1;
            scal[NK_S_BETA] = 0.0; scal[NK_S_ALPHA] = 0.0; scal[NK_S_PAP] = 0.0;
        } else {
            const double rho = scal[NK_S_RHO], pap = scal[NK_S_PAP];
            scal[NK_S_RHO_NEW] = t1;
            scal[NK_S_BETA] = (rho == 0.0 || pap == 0.0) ? 0.0 : t1 / rho;
            scal[NK_S_RHO_OLD] = rho;
            scal[NK_S_RHO] = t1;
        }
        out[0] = sqrt(t2);
    }
}
