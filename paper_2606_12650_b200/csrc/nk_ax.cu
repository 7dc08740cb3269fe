// nk_ax.cu -- ax_e, the round's FIRST kernel ("ax_variant" = 1; the default is nk_ax_tma.cu): one CTA
// per element batch, load -> compute -> store with nothing in flight while it computes (39 % of the
// copy peak at config 5).  Kept for A/B runs and as a second implementation under the parity tests.
//
// ax_e: w = A_L u, the element-local matrix-free Laplacian ("the action of the
// Poisson operator", the most expensive kernel; S 8(a) a1, S 8(c) O3; BJ north_star (1)).
//
//   u_r = D u along r, u_s = D u along s, u_t = D u along t            (3 x (N+1) fma per point)
//   (w_r, w_s, w_t) = G (u_r, u_s, u_t),  G symmetric 3x3 per point    (15 flops per point)
//   w = D^T w_r along r + D^T w_s along s + D^T w_t along t            (3 x (N+1) fma per point)
//
// HBM-bound by design: 64 B per point (u 8, G 48, w 8) against 12(N+1)+15 flops, so no tensor
// cores (BJ).  What limits a straightforward kernel on sm_100a is not HBM but shared-memory issue
// and the fp64 pipe (S 7 hard part 2), so the "line" kernel below arranges the work so that EVERY
// entry of D is a compile-time-indexed __constant__ operand folded into the DFMA itself:
//
//   One element = n^2 threads (n = N+1).  The same thread plays three roles on the element cube:
//     pencil (i,j): owns u(i,j,0..n-1) in registers   -> t-derivative and its transpose, G, load/store
//     row    (j,k): owns u(0..n-1,j,k) read from smem -> r-derivative and its transpose
//     column (i,k): owns u(i,0..n-1,k) read from smem -> s-derivative and its transpose
//   A thread that owns a whole grid line computes all n outputs of that line from n register
//   values: n^2 DFMAs whose D operand is c[bank][imm] -- no D registers, no D loads.  Per point
//   that leaves 16 shared-memory accesses (against 4(N+1)+3 for the 2-D-slab/k-loop scheme) and
//   6(N+1) DFMAs.  Rows are padded to an odd stride so row, column and pencil accesses are all
//   bank-conflict-free (or 2-way at worst for a few odd n).
//
// Fusions on the CG path (S 8(f) f-1):
//   dot   : sum_l u_l w_l is reduced in the same pass ("dot-fusion identity": for consistent,
//           masked p, <M QQ^T A_L p, p>_c = sum_l (A_L p)_l p_l), epilogue alpha = rho/pap;
//   r_in  : the direction update p = r + beta p is applied while loading (and p written back).
#include "nk_internal.h"
#include "nk_reduce.cuh"

namespace {

// D for every order N = 1..15 back to back: table of order n-1 starts at doff(n) = sum_{q=2}^{n-1} q^2.
__host__ __device__ constexpr int doff(int n) { int s = 0; for (int q = 2; q < n; ++q) s += q * q; return s; }
constexpr int D_TOTAL = doff(17);
__constant__ double c_D[D_TOTAL];

// elements per block for the line kernel (threads = EPB * n^2 rounded up to a warp multiple)
__host__ __device__ constexpr int line_epb(int n)
{
#ifdef NK_LINE_EPB
    return NK_LINE_EPB;
#else
    return n == 2 ? 32 : n == 3 ? 14 : n == 4 ? 8 : n == 5 ? 5 : n == 6 ? 7 : n == 7 ? 5 : n == 8 ? 2
         : n == 9 ? 3 : n == 10 ? 2 : n == 12 ? 2 : 1;
#endif
}
__host__ __device__ constexpr int round32(int x) { return (x + 31) / 32 * 32; }

template <int N>
struct LineCfg {
    static constexpr int n = N + 1, n2 = n * n, P = n2 * n;
    static constexpr int EPB = line_epb(n);
    static constexpr int THREADS = round32(EPB * n2);
    static constexpr int S1 = (n & 1) ? n : n + 1;     // odd row stride
    static constexpr int S2 = n * S1;                  // plane stride
    static constexpr int SE = n * S2;                  // one padded element cube
    static constexpr size_t SMEM = (size_t)EPB * 3 * SE * sizeof(double);
};

#define DM(i, m) c_D[DOFF + (i) * n + (m)]

template <int N>
__global__ void __launch_bounds__(LineCfg<N>::THREADS)
ax_line_kernel(double *__restrict__ u_rw, const double *__restrict__ u_ro, const double *__restrict__ r_in,
               double *__restrict__ w, const double2 *__restrict__ g, int64_t E, int dot, nk_reduce_ws red)
{
    using C = LineCfg<N>;
    constexpr int n = C::n, n2 = C::n2, S1 = C::S1, S2 = C::S2, SE = C::SE, EPB = C::EPB;
    constexpr int DOFF = doff(n);
    extern __shared__ double smem[];
    __shared__ double s_red[33];

    const int tid = threadIdx.x;
    const int slot = tid / n2;
    const int t2 = tid - slot * n2;
    const int a = t2 % n, b = t2 / n;
    const int64_t e = (int64_t)blockIdx.x * EPB + slot;
    const bool active = (slot < EPB) && (e < E);
    double *su = smem + (size_t)(slot < EPB ? slot : 0) * 3 * SE;
    double *sa = su + SE, *sb = sa + SE;
    const int64_t gbase = e * C::P + t2;            // pencil (i,j) = (a,b): + k*n2
    const int pbase = a + b * S1;                   // pencil in smem: + k*S2
    const int rbase = (a + n * b) * S1;             // row (j,k) = (a,b): + i        (S2 = n*S1)
    const int cbase = a + b * S2;                   // column (i,k) = (a,b): + j*S1

    double ru[n];
    if (active) {
        if (r_in != nullptr) {
            const double beta = red.scal[NK_S_BETA];
#pragma unroll
            for (int k = 0; k < n; ++k) {
                const double pv = u_rw[gbase + k * n2], rv = r_in[gbase + k * n2];
                ru[k] = fma(beta, pv, rv);
            }
#pragma unroll
            for (int k = 0; k < n; ++k) u_rw[gbase + k * n2] = ru[k];
        } else {
#pragma unroll
            for (int k = 0; k < n; ++k) ru[k] = u_ro[gbase + k * n2];
        }
#pragma unroll
        for (int k = 0; k < n; ++k) su[pbase + k * S2] = ru[k];
    }
    __syncthreads();
    if (active) {
        double ln[n];
#pragma unroll
        for (int m = 0; m < n; ++m) ln[m] = su[rbase + m];
#pragma unroll
        for (int i = 0; i < n; ++i) {
            double acc = DM(i, 0) * ln[0];
#pragma unroll
            for (int m = 1; m < n; ++m) acc = fma(DM(i, m), ln[m], acc);
            sa[rbase + i] = acc;
        }
#pragma unroll
        for (int m = 0; m < n; ++m) ln[m] = su[cbase + m * S1];
#pragma unroll
        for (int j = 0; j < n; ++j) {
            double acc = DM(j, 0) * ln[0];
#pragma unroll
            for (int m = 1; m < n; ++m) acc = fma(DM(j, m), ln[m], acc);
            sb[cbase + j * S1] = acc;
        }
    }
    __syncthreads();
    double rw[n];
    if (active) {
        double wt[n];
#pragma unroll
        for (int k = 0; k < n; ++k) {
            double acc = DM(k, 0) * ru[0];
#pragma unroll
            for (int m = 1; m < n; ++m) acc = fma(DM(k, m), ru[m], acc);
            wt[k] = acc;
        }
#pragma unroll
        for (int k = 0; k < n; ++k) {
            const double2 *gk = g + nk_g_index(e, k, 0, t2, n);
            const double2 ga = gk[0], gb = gk[n2], gc = gk[2 * n2];
            const double ur = sa[pbase + k * S2], us = sb[pbase + k * S2], ut = wt[k];
            sa[pbase + k * S2] = fma(ga.x, ur, fma(ga.y, us, gb.x * ut));   // w_r = rr ur + rs us + rt ut
            sb[pbase + k * S2] = fma(ga.y, ur, fma(gb.y, us, gc.x * ut));   // w_s = rs ur + ss us + st ut
            wt[k] = fma(gb.x, ur, fma(gc.x, us, gc.y * ut));                // w_t = rt ur + st us + tt ut
        }
#pragma unroll
        for (int m = 0; m < n; ++m) {
            double acc = DM(0, m) * wt[0];
#pragma unroll
            for (int k = 1; k < n; ++k) acc = fma(DM(k, m), wt[k], acc);
            rw[m] = acc;
        }
    }
    __syncthreads();
    if (active) {
        double ln[n];
#pragma unroll
        for (int m = 0; m < n; ++m) ln[m] = sa[rbase + m];
#pragma unroll
        for (int i = 0; i < n; ++i) {
            double acc = DM(0, i) * ln[0];
#pragma unroll
            for (int m = 1; m < n; ++m) acc = fma(DM(m, i), ln[m], acc);
            sa[rbase + i] = acc;
        }
#pragma unroll
        for (int m = 0; m < n; ++m) ln[m] = sb[cbase + m * S1];
#pragma unroll
        for (int j = 0; j < n; ++j) {
            double acc = DM(0, j) * ln[0];
#pragma unroll
            for (int m = 1; m < n; ++m) acc = fma(DM(m, j), ln[m], acc);
            sb[cbase + j * S1] = acc;
        }
    }
    __syncthreads();
    double dsum = 0.0;
    if (active) {
#pragma unroll
        for (int k = 0; k < n; ++k) {
            const double wv = rw[k] + (sa[pbase + k * S2] + sb[pbase + k * S2]);
            w[gbase + k * n2] = wv;
            dsum = fma(ru[k], wv, dsum);
        }
    }
    if (dot) nk_grid_reduce(dsum, s_red, red, NK_EPI_PAP, nullptr);
}

template <int N>
cudaError_t launch_line(nk_ctx *c, double *u_rw, const double *u_ro, const double *r_in, double *w, int dot,
                        cudaStream_t st)
{
    using C = LineCfg<N>;
    const int64_t nb = (c->E + C::EPB - 1) / C::EPB;
    if (dot && nb > NK_MAX_PARTIALS) return cudaErrorInvalidConfiguration;
    ax_line_kernel<N><<<(unsigned)nb, C::THREADS, C::SMEM, st>>>(u_rw, u_ro, r_in, w, c->g, c->E, dot, c->red);
    c->launches++;
    return cudaGetLastError();
}

template <int N>
cudaError_t prepare_line()
{
    return cudaFuncSetAttribute(ax_line_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)LineCfg<N>::SMEM);
}

}  // namespace

// Upload D for every order and opt every instantiation in to its dynamic shared memory size.
cudaError_t nk_upload_D_tables(void)
{
    static double h[D_TOTAL];
    double xi[16], wq[16];
    for (int N = 1; N <= NK_MAX_ORDER; ++N) nk_host_basis(N, xi, wq, h + doff(N + 1));
    cudaError_t e = cudaMemcpyToSymbol(c_D, h, sizeof(h));
    if (e != cudaSuccess) return e;
#define NK_CASE(NN) if ((e = prepare_line<NN>()) != cudaSuccess) return e;
    NK_CASE(1) NK_CASE(2) NK_CASE(3) NK_CASE(4) NK_CASE(5) NK_CASE(6) NK_CASE(7) NK_CASE(8)
    NK_CASE(9) NK_CASE(10) NK_CASE(11) NK_CASE(12) NK_CASE(13) NK_CASE(14) NK_CASE(15)
#undef NK_CASE
    return cudaSuccess;
}

cudaError_t nk_launch_ax_e(nk_ctx *c, double *u_rw, const double *u_ro, const double *r_in, double *w, int dot,
                           int variant, cudaStream_t st)
{
    if (variant != 1) return nk_launch_ax_tma(c, u_rw, u_ro, r_in, w, dot, st);
    switch (c->N) {
#define NK_CASE(NN) case NN: return launch_line<NN>(c, u_rw, u_ro, r_in, w, dot, st);
        NK_CASE(1) NK_CASE(2) NK_CASE(3) NK_CASE(4) NK_CASE(5) NK_CASE(6) NK_CASE(7) NK_CASE(8)
        NK_CASE(9) NK_CASE(10) NK_CASE(11) NK_CASE(12) NK_CASE(13) NK_CASE(14) NK_CASE(15)
#undef NK_CASE
    }
    return cudaErrorInvalidValue;
}
