// nk_ax_tma.cu -- ax_e: w = A_L u, TMA-pipelined persistent kernel for sm_100a (the default variant).
// ("the action of the Poisson operator", the most expensive kernel; S 8(a) a1, S 8(c) O3;
// BJ north_star (1).)
//
// Why this shape: ax_e moves 64 B per point (u 8, G 48, w 8) for 12(N+1)+15 flops and
// must run at HBM speed.  The first kernel of this round (nk_ax.cu, one CTA per element batch, load
// -> compute -> store, one CTA resident per SM) reached 39 % of the copy peak with the fp64 pipe
// 17 % busy: nothing was in flight while a CTA computed.  Here one persistent CTA per SM splits
// into
//   * a producer warp: one lane streams the geometric factors -- 75 % of the bytes -- into a
//     shared-memory ring with cp.async.bulk (TMA bulk copies, SASS UBLKCP) completing on mbarriers,
//     k-plane by k-plane, running up to a whole element batch ahead of the arithmetic;
//   * compute warps: the "line" scheme.  A thread owns the pencil (i,j) of u in registers, a whole
//     row (j,k) and a whole column (i,k) of the padded shared cube: 16 shared-memory accesses per
//     point.  Phases per batch: P1 pencil -> cube; P2 D along row, column and pencil in ONE pass over
//     the even-odd table (lines_apply: every entry fetched once through the uniform datapath, feeding
//     three DFMAs); P3 the 3x3 G per point from the ring (+ the fused pap); P4 D^T likewise; P5 sum
//     and store.  The next batch's u pencil is requested into registers while this one finishes.
// G never touches registers before it is used and u is read exactly once, so DRAM traffic equals
// the algorithmic bytes, and the bytes in flight per SM (ring of ~110-170 KB) exceed the ~30 KB
// that 5.6 TB/s x ~0.8 us of latency asks for.
//
//   u_r = D u along r, u_s = D u along s, u_t = D u along t            (3 x (N+1) fma per point)
//   (w_r, w_s, w_t) = G (u_r, u_s, u_t),  G symmetric 3x3 per point    (15 flops per point)
//   w = D^T w_r along r + D^T w_s along s + D^T w_t along t            (3 x (N+1) fma per point)
//
// Fusions on the CG path (S 8(f) f-1), as in nk_ax.cu:
//   dot   : sum_l u_l w_l reduced in the same pass (dot-fusion identity), epilogue alpha = rho/pap;
//   r_in  : p = r + beta p applied while loading (p written back).
#include "nk_internal.h"
#include "nk_reduce.cuh"

namespace {

// Even-odd tables.  D and D^T are centro-antisymmetric (M[n-1-i][n-1-m] = -M[i][m]: the GLL
// nodes are symmetric), so with e_m = v_m + v_{n-1-m}, o_m = v_m - v_{n-1-m}, h = floor(n/2), H = ceil(n/2):
//   S_i = sum_{m<h} Me[i][m] e_m (+ M[i][mid] v_mid, n odd),   Me[i][m] = (M[i][m] + M[i][n-1-m]) / 2
//   A_i = sum_{m<h} Mo[i][m] o_m,                               Mo[i][m] = (M[i][m] - M[i][n-1-m]) / 2
//   (M v)_i = A_i + S_i,   (M v)_{n-1-i} = A_i - S_i            for i < H
// -- n^2/2 DFMAs and 2n DADDs per grid line instead of n^2 DFMAs.  Per order n and per matrix (D, then
// D^T) the table holds H rows of [Mo[i][0..h) | Me[i][0..h) (, M[i][mid])].
__host__ __device__ constexpr int eo_row(int n) { return n / 2 + (n + 1) / 2; }
__host__ __device__ constexpr int eo_mat(int n) { return (n + 1) / 2 * eo_row(n); }
__host__ __device__ constexpr int eo_off(int n) { int s = 0; for (int q = 2; q < n; ++q) s += 2 * eo_mat(q); return s; }
constexpr int D_TOTAL = eo_off(17);
__constant__ double c_Dt[D_TOTAL];
// which row and which column of its sync group a compute thread takes: offsets (doubles) from the group's first
// cube, per order, [0] rows, [1] columns, indexed by the thread's index in the group (TmaCfg, line_tables)
constexpr int LUT_MAX = 384;
__constant__ uint16_t c_lut[NK_MAX_ORDER + 1][2][LUT_MAX];

constexpr int SMEM_CAP = 232448 - 1024;     // 227 KB opt-in limit minus this kernel's static shared memory
constexpr int BAR_BYTES = 1024;             // 2 x 64 mbarriers

// plane padding (doubles) that spreads the starts of rows, n j + S2 k, and of columns, i + S2 k, most evenly over
// the 16 eight-byte banks of a half-warp (0 .. 16 tried; ties go to the smaller cube)
__host__ __device__ constexpr int plane_pad(int n)
{
    const int n2 = n * n, groups = (n2 + 15) / 16;
    int best = 0, best_score = 1 << 30;
    for (int pad = 0; pad <= 16; ++pad) {
        const int S2 = n2 + pad;
        int hr[16] = {}, hc[16] = {};
        for (int k = 0; k < n; ++k)
            for (int a = 0; a < n; ++a) { ++hr[(n * a + S2 * k) & 15]; ++hc[(a + S2 * k) & 15]; }
        int mr = 0, mc = 0;
        for (int b = 0; b < 16; ++b) { mr = hr[b] > mr ? hr[b] : mr; mc = hc[b] > mc ? hc[b] : mc; }
        const int score = (mr > groups ? mr - groups : 0) + (mc > groups ? mc - groups : 0);
        if (score < best_score) { best_score = score; best = pad; }
    }
    return best;
}
// cube padding with nw (se0 + pad) = n2 (mod 16), 0 if there is none
__host__ __device__ constexpr int cube_pad(int nw, int se0, int n2)
{
    for (int pad = 0; pad < 16; ++pad)
        if (((nw * (se0 + pad)) & 15) == (n2 & 15)) return pad;
    return 0;
}

// elements per batch: ~256 compute threads, fewer where shared memory is the limit
__host__ __device__ constexpr int tma_epb(int n)
{
#ifdef NK_TMA_EPB
    return NK_TMA_EPB;
#else
#ifndef NK_EPB_8
#define NK_EPB_8 4
#endif
#ifndef NK_EPB_9
#define NK_EPB_9 4
#endif
#ifndef NK_EPB_10
#define NK_EPB_10 2
#endif
    return n <= 2 ? 32 : n == 3 ? 28 : n == 4 ? 16 : n == 5 ? 10 : n == 6 ? 7 : n == 7 ? 5 : n == 8 ? NK_EPB_8
         : n == 9 ? NK_EPB_9 : n == 10 ? NK_EPB_10 : n <= 12 ? 2 : 1;
#endif
}

template <int N>
struct TmaCfg {
    static constexpr int n = N + 1, n2 = n * n, P = n2 * n;
    static constexpr int EPB = tma_epb(n);
    // Sync groups: the element slots of a batch that share one named barrier.  From n^2 >= 64 on every
    // slot is its own group of whole warps, so the elements of a batch drift apart and the
    // shared-memory-bound phases of one overlap the DFMA-bound phases of the other.
    // (n = 9 with four slots of three warps each: 35.5 -> 34.0 us at 16^3, the one 4b point that was below 70 %)
    static constexpr int SG = (n == 8 || n == 9 || n == 10 || n == 11 || n == 12 || n == 16) ? 1 : EPB;   // slots per group
    // (only where a slot fills whole warps well; elsewhere per-slot groups cost a warp and registers)
    static constexpr int NG = EPB / SG;                       // groups
    static constexpr int GTH = (SG * n2 + 31) / 32 * 32;      // threads per group
    static constexpr int CT = NG * GTH;                       // compute threads
    static constexpr int CW = CT / 32;                        // compute warps
    // Warp-specialised register budget (n >= 15: eight full compute warps): the producer sits in a
    // warpgroup of its own, which gives its registers back (setmaxnreg.dec) so that the two compute
    // warpgroups can take 232 each (setmaxnreg.inc).  Without it nine warps cap every thread at 168
    // registers (the register file is split per scheduler) and the n = 15, 16 kernels spill to L2.
#ifdef NK_TMA_NO_SETMAXNREG
    static constexpr bool WGP = false;
#else
    static constexpr bool WGP = (n >= 15) && (CW % 4 == 0);
#endif
    static constexpr int THREADS = CT + (WGP ? 128 : 32);     // + producer warp (or warpgroup)
    static_assert(EPB % SG == 0 && NG <= 15, "sync groups");
    // Shared-memory cube: rows dense (stride n), planes padded by PADK doubles, cubes by PADE.  A thread's pencil
    // (i,j) then sits at its own thread index (+ k S2): consecutive lanes, consecutive doubles, never a bank
    // conflict.  Rows (j,k) start at n j + S2 k and columns (i,k) at i + S2 k; PADK is chosen so that these starts
    // spread evenly over the 16 eight-byte banks of a half-warp, and WHICH row / column a thread takes comes from a
    // table (c_lut, built on the host by line_tables below) that gives every half-warp 16 different banks.  (The
    // round-1 layout -- odd row stride, thread (a,b) takes row (a,b) -- had two-way conflicts on every pencil
    // access for even n and on every column access for odd n: 29 % of all shared-memory wavefronts at n = 12.)
    static constexpr int S1 = n;
    static constexpr int PADK = plane_pad(n);
    static constexpr int S2 = n2 + PADK;
    static constexpr int SE0 = n * S2;
    // a ring stage holds KP k-planes of every element of the batch: whole elements for small n
    // (one bulk copy per batch), single k-planes otherwise (one bulk copy per element and plane)
    static constexpr int KP = (n <= 6) ? n : 1;            // (2 or 3 planes per stage at n = 12: measured 1.5 % slower)
    static constexpr int STAGE_D2 = EPB * KP * 3 * n2;        // double2 per stage
    static constexpr int STAGE_BYTES = STAGE_D2 * 16;
    static constexpr int SPB = n / KP;                        // stages per batch
    static constexpr int work_bytes(int nw) { return nw * EPB * (SE0 + 15) * 8; }   // (bound: SE = SE0 + PADE <= SE0 + 15)
    static constexpr int ring_for(int nw) { return (SMEM_CAP - BAR_BYTES - work_bytes(nw)) / STAGE_BYTES; }
    // three work arrays (4 barriers per batch) if the ring then still holds 1.5 batches, else two (6
    // barriers).  (At N = 11 the alternative -- three arrays and a 9-plane ring -- is 2 % faster for a
    // lone ax_e but 4 % slower inside the CG iteration, measured A/B in one bench run: 723 vs 692 us.)
    static constexpr int NW = (ring_for(3) >= (3 * SPB + 1) / 2) ? 3 : 2;
    static constexpr int RMAX = ring_for(NW) < 3 * SPB ? ring_for(NW) : 3 * SPB;
#ifdef NK_TMA_RCAP
    static constexpr int R = RMAX > NK_TMA_RCAP ? NK_TMA_RCAP : RMAX;
#else
    static constexpr int R = RMAX > 64 ? 64 : RMAX;
#endif
    // several slots per sync group: thread indices run on from slot to slot, so the slot stride NW SE continues
    // the bank sequence where it can (NW SE = n^2 mod 16)
    static constexpr int PADE = (SG > 1) ? cube_pad(NW, SE0, n2) : 0;
    static constexpr int SE = SE0 + PADE;
    static constexpr int WORK_BYTES = NW * EPB * SE * 8;
    static constexpr int SMEM = R * STAGE_BYTES + WORK_BYTES + BAR_BYTES;
    static_assert(R >= 2, "ring too small");
#ifndef NK_TMA_IB
#define NK_TMA_IB 2
#endif
    static constexpr int IB = NK_TMA_IB;                      // table rows advanced together in lines_apply
    // where the next batch's u pencil is requested: 1 = after P3, 2 = after P4 (measured per order)
#ifdef NK_TMA_PF12
    static constexpr int PF = (n == 12) ? NK_TMA_PF12 : 1;
#else
    static constexpr int PF = (n == 12) ? 2 : 1;
#endif
};

// ---- mbarrier / bulk-copy PTX ---------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ uint32_t mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\n"
        "selp.u32 %0, 1, 0, P1;\n"
        "}\n" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    return done;
}
// Producer lane: plain spin.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) {}
}
// Compute warps: every lane probes (each needs the acquire), the loop branch is a warp vote.  A
// per-thread spin would leave ptxas unable to prove the warp converged afterwards, and all D
// operands behind it would fall off the uniform datapath (LDC into vector registers, not LDCU).
__device__ __forceinline__ void mbar_wait_warp(uint32_t bar, uint32_t parity)
{
    while (!__all_sync(0xffffffffu, mbar_try_wait(bar, parity))) {}
}
// global -> shared bulk copy (TMA, 1-D), completes `bytes` on the mbarrier; 16-byte aligned, size % 16 == 0
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
template <int COUNT>
__device__ __forceinline__ void group_sync(int grp)     // named barrier 1 + grp: one sync group's warps
{
    asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "n"(COUNT) : "memory");
}

// One grid line through M = D (MOFF = DOFF) or D^T (MOFF = TOFF): out_i = sum_m M[i][m] ln[m], by the
// even-odd splitting above.  IB rows advance together (2 IB independent DFMA chains per thread); every
// table entry is a compile-time-indexed __constant__ operand (uniform datapath: LDCU -> UR).
template <int n, int MOFF, class Store>
__device__ __forceinline__ void line_apply(const double (&ln)[n], Store store)
{
    constexpr int IB = 2, h = n / 2, H = (n + 1) / 2, ROW = eo_row(n);
    double ev[H], od[h > 0 ? h : 1];
#pragma unroll
    for (int m = 0; m < h; ++m) {
        ev[m] = ln[m] + ln[n - 1 - m];
        od[m] = ln[m] - ln[n - 1 - m];
    }
    if (n & 1) ev[H - 1] = ln[H - 1];
#pragma unroll
    for (int i0 = 0; i0 < H; i0 += IB) {
        double S[IB], A[IB];
#pragma unroll
        for (int j = 0; j < IB; ++j)
            if (i0 + j < H) {
                const double *row = c_Dt + MOFF + (i0 + j) * ROW;
                A[j] = row[0] * od[0];
                S[j] = row[h] * ev[0];
            }
#pragma unroll
        for (int m = 1; m < H; ++m) {
#pragma unroll
            for (int j = 0; j < IB; ++j)
                if (i0 + j < H) {
                    const double *row = c_Dt + MOFF + (i0 + j) * ROW;
                    if (m < h) A[j] = fma(row[m], od[m], A[j]);
                    S[j] = fma(row[h + m], ev[m], S[j]);
                }
        }
#pragma unroll
        for (int j = 0; j < IB; ++j)
            if (i0 + j < H) {
                const int i = i0 + j;
                if (n - 1 - i != i) {
                    store(i, A[j] + S[j]);
                    store(n - 1 - i, A[j] - S[j]);
                } else {
                    store(i, A[j]);          // middle row of an odd n: its even part vanishes
                }
            }
    }
}

// The same transform applied to NL grid lines at once (a thread's row, column and pencil): every table
// entry is fetched once per phase and feeds NL DFMAs, and 2 IB NL independent chains are in flight.
// (Three separate line_apply calls made ptxas keep the table of the first call alive for the next ones:
// uniform registers spilled to vector registers and back, ~1 extra instruction per DFMA.)
template <int n, int MOFF, int NL, int IB, class Store>
__device__ __forceinline__ void lines_apply(const double (&ln)[NL][n], Store store)
{
    constexpr int h = n / 2, H = (n + 1) / 2, ROW = eo_row(n);
    double ev[NL][H], od[NL][h > 0 ? h : 1];
#pragma unroll
    for (int q = 0; q < NL; ++q) {
#pragma unroll
        for (int m = 0; m < h; ++m) {
            ev[q][m] = ln[q][m] + ln[q][n - 1 - m];
            od[q][m] = ln[q][m] - ln[q][n - 1 - m];
        }
        if (n & 1) ev[q][H - 1] = ln[q][H - 1];
    }
#pragma unroll
    for (int i0 = 0; i0 < H; i0 += IB) {
        double S[IB][NL], A[IB][NL];
#pragma unroll
        for (int j = 0; j < IB; ++j)
            if (i0 + j < H) {
                const double *row = c_Dt + MOFF + (i0 + j) * ROW;
#pragma unroll
                for (int q = 0; q < NL; ++q) {
                    A[j][q] = (h > 0) ? row[0] * od[q][0] : 0.0;
                    S[j][q] = row[h] * ev[q][0];
                }
            }
#pragma unroll
        for (int m = 1; m < H; ++m) {
#pragma unroll
            for (int j = 0; j < IB; ++j)
                if (i0 + j < H) {
                    const double *row = c_Dt + MOFF + (i0 + j) * ROW;
#pragma unroll
                    for (int q = 0; q < NL; ++q) {
                        if (m < h) A[j][q] = fma(row[m], od[q][m], A[j][q]);
                        S[j][q] = fma(row[h + m], ev[q][m], S[j][q]);
                    }
                }
        }
#pragma unroll
        for (int j = 0; j < IB; ++j)
            if (i0 + j < H) {
                const int i = i0 + j;
#pragma unroll
                for (int q = 0; q < NL; ++q) {
                    if (n - 1 - i != i) {
                        store(q, i, A[j][q] + S[j][q]);
                        store(q, n - 1 - i, A[j][q] - S[j][q]);
                    } else {
                        store(q, i, A[j][q]);
                    }
                }
            }
    }
}

template <int N, bool FUSEP>
__global__ void __launch_bounds__(TmaCfg<N>::THREADS, 1)
ax_tma_kernel(double *__restrict__ u_rw, const double *__restrict__ u_ro, const double *__restrict__ r_in,
              double *__restrict__ w, const double2 *__restrict__ g, int64_t E, int dot, nk_reduce_ws red)
{
    using C = TmaCfg<N>;
    constexpr int n = C::n, n2 = C::n2, P = C::P, S1 = C::S1, S2 = C::S2, SE = C::SE, EPB = C::EPB;
    constexpr int R = C::R, KP = C::KP, NW = C::NW, CW = C::CW, CTHREADS = C::CT, GTH = C::GTH, SG = C::SG;
    constexpr int DOFF = eo_off(n), TOFF = DOFF + eo_mat(n);     // even-odd tables of D and D^T in c_Dt
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ double s_red[33];
    const double2 *ring = reinterpret_cast<const double2 *>(smem_raw);
    double *work = reinterpret_cast<double *>(smem_raw + (size_t)R * C::STAGE_BYTES);
    const uint32_t ring0 = smem_u32(smem_raw);
    const uint32_t full0 = ring0 + R * C::STAGE_BYTES + C::WORK_BYTES, empty0 = full0 + 8 * R;

    const int tid = threadIdx.x;
    if (tid == 0) {
        for (int s = 0; s < R; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, CW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // This CTA's elements: a contiguous range, equal over the CTAs to within one element (batches dealt round
    // robin left the last round 1/4 full on a 16^3 mesh at N = 9: one batch time of 10 lost).  The last batch of
    // a range may be partial.
    const int64_t elo = E * (int64_t)blockIdx.x / gridDim.x, ehi = E * ((int64_t)blockIdx.x + 1) / gridDim.x;
    const int nit = (int)((ehi - elo + EPB - 1) / EPB);
    double dsum = 0.0;

    if (C::WGP) {
        if (tid >= CTHREADS) asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
        else asm volatile("setmaxnreg.inc.sync.aligned.u32 240;");
    }
    if (tid >= CTHREADS) {
        // ---- producer warp: one lane streams G into the ring ----------------------------------------
        if (tid == CTHREADS) {
            int stage = 0;
            uint32_t phase = 0;
            for (int it = 0; it < nit; ++it) {
                const int64_t e0 = elo + (int64_t)it * EPB;
                const int ne = (int)((ehi - e0 < EPB) ? (ehi - e0) : EPB);
#pragma unroll 1
                for (int ks = 0; ks < C::SPB; ++ks) {
                    mbar_wait(empty0 + 8 * stage, phase ^ 1u);
                    const uint32_t fb = full0 + 8 * stage, dst = ring0 + stage * C::STAGE_BYTES;
                    if (KP == n) {       // whole elements: the batch is one contiguous chunk
                        mbar_expect_tx(fb, (uint32_t)ne * P * 48);
                        bulk_g2s(dst, g + nk_g_index(e0, 0, 0, 0, n), (uint32_t)ne * P * 48, fb);
                    } else {             // KP consecutive k-planes (contiguous in HBM) of every element of the batch
                        mbar_expect_tx(fb, (uint32_t)ne * KP * n2 * 48);
                        for (int q = 0; q < ne; ++q)
                            bulk_g2s(dst + q * KP * n2 * 48, g + nk_g_index(e0 + q, ks * KP, 0, 0, n), KP * n2 * 48, fb);
                    }
                    if (++stage == R) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else {
        // ---- compute warps ----------------------------------------------------------------------------
        // No arithmetic below sits under a thread-dependent branch: D reaches the DFMAs through the
        // uniform datapath (LDCU -> UR operand), which ptxas only uses in warp-uniform code.  Threads
        // without an element (ragged last warp, tail batch) compute on stale shared memory and only
        // their stores are predicated off.
        const int lane = tid & 31;
        const int grp = tid / GTH, lt = tid - grp * GTH;
        const int sl = lt / n2, t2 = lt - sl * n2;
        const int a = t2 % n, b = t2 / n;
        const bool mapped = sl < SG;
        const int slot = grp * SG + (mapped ? sl : 0);
        // work arrays of the sync group's first slot; slot s of the group sits s NW SE doubles further on
        double *sA = work + (size_t)(grp * SG) * NW * SE;              // u, then (NW = 2) the s direction
        double *sB = sA + SE;                                          // r direction
        double *sC = (NW == 3) ? sB + SE : sA;                         // s direction
        const int pbase = (mapped ? sl : 0) * NW * SE + t2;            // pencil (i,j) of the thread's slot: + k*S2
        const int rbase = c_lut[N][0][lt];                             // a row (j,k) of the group: + i
        const int cbase = c_lut[N][1][lt];                             // a column (i,k) of the group: + j*S1
        const double2 *gslot = ring + slot * KP * 3 * n2 + t2;
        nk_pdl_wait();                                  // u, r, beta come from the preceding kernels
        const double beta = FUSEP ? red.scal[NK_S_BETA] : 0.0;
        int stage = 0;
        uint32_t phase = 0;

        double nu[n], nr[FUSEP ? n : 1];               // next batch's pencil, in flight
        {
            const int64_t e = elo + slot;
            const bool act = mapped && e < ehi;
            const int64_t gb = act ? e * P + t2 : 0;
#pragma unroll
            for (int k = 0; k < n; ++k) {
                nu[k] = act ? (FUSEP ? u_rw[gb + k * n2] : u_ro[gb + k * n2]) : 0.0;
                if (FUSEP) nr[k] = act ? r_in[gb + k * n2] : 0.0;
            }
        }
        for (int it = 0; it < nit; ++it) {
            const int64_t e = elo + (int64_t)it * EPB + slot;
            const bool active = mapped && e < ehi;
            const int64_t gbase = e * P + t2;
            double ru[n];
            // P1: pencil -> padded cube (and p = r + beta p written back)
#pragma unroll
            for (int k = 0; k < n; ++k) ru[k] = FUSEP ? fma(beta, nu[k], nr[k]) : nu[k];
            if (mapped) {
#pragma unroll
                for (int k = 0; k < n; ++k) sA[pbase + k * S2] = ru[k];
            }
            if (FUSEP && active) {
#pragma unroll
                for (int k = 0; k < n; ++k) u_rw[gbase + k * n2] = ru[k];
            }
            group_sync<GTH>(grp);
            // P2: D along the thread's row (A -> B), column (A -> C) and pencil (registers -> wt), one pass
            double wt[n];
            {
                double ln[3][n], cres[NW == 2 ? n : 1];
#pragma unroll
                for (int m = 0; m < n; ++m) {
                    ln[0][m] = sA[rbase + m];
                    ln[1][m] = sA[cbase + m * S1];
                    ln[2][m] = ru[m];
                }
                lines_apply<n, DOFF, 3, C::IB>(ln, [&](int q, int i, double v) {
                    if (q == 0) { if (mapped) sB[rbase + i] = v; }
                    else if (q == 1) { if (NW == 2) cres[NW == 2 ? i : 0] = v; else if (mapped) sC[cbase + i * S1] = v; }
                    else wt[i] = v;
                });
                if (NW == 2) {                          // columns overwrite A in place: all reads of A are done
                    group_sync<GTH>(grp);
                    if (mapped) {
#pragma unroll
                        for (int j = 0; j < n; ++j) sC[cbase + j * S1] = cres[j];
                    }
                }
            }
            group_sync<GTH>(grp);
            // P3: the geometric factors from the ring, point by point along the pencil
            {
                // a stage (KP planes) is waited for when its first plane comes up and handed back after its
                // last one.  (Waiting for several stages at once was tried and is slower: the register
                // pressure of interleaved planes costs more than the waits.)
                double dloc = 0.0;
#pragma unroll
                for (int k = 0; k < n; ++k) {
                    if (k % KP == 0) mbar_wait_warp(full0 + 8 * stage, phase);
                    const double2 *gs = gslot + (size_t)stage * C::STAGE_D2 + (k % KP) * 3 * n2;
                    const double2 ga = gs[0], gb = gs[n2], gc = gs[2 * n2];
                    const double ur = sB[pbase + k * S2], us = sC[pbase + k * S2], ut = wt[k];
                    const double wr = fma(ga.x, ur, fma(ga.y, us, gb.x * ut));  // w_r = rr ur + rs us + rt ut
                    const double ws = fma(ga.y, ur, fma(gb.y, us, gc.x * ut));  // w_s = rs ur + ss us + st ut
                    const double wk = fma(gb.x, ur, fma(gc.x, us, gc.y * ut));  // w_t = rt ur + st us + tt ut
                    if (mapped) {
                        sB[pbase + k * S2] = wr;
                        sC[pbase + k * S2] = ws;
                    }
                    wt[k] = wk;
                    // <u, A_L u> = sum over points of grad(u)^T G grad(u): the fused pap needs no u later on
                    dloc += fma(ur, wr, fma(us, ws, ut * wk));
                    if (k % KP == KP - 1) {          // this warp is done with the stage: hand it back
                        __syncwarp();
                        if (lane == 0) mbar_arrive(empty0 + 8 * stage);
                        if (++stage == R) { stage = 0; phase ^= 1u; }
                    }
                }
                dsum += active ? dloc : 0.0;        // threads without an element computed on stale data
            }
            group_sync<GTH>(grp);
            auto prefetch = [&]() {
                // the next batch's pencil, in flight while this batch finishes (the register file is
                // split four ways, so > 8 warps means <= 168 registers: not before P3, where pressure peaks)
                const int64_t e1 = e + EPB;
                const bool act = mapped && e1 < ehi;
                const int64_t gb = act ? e1 * P + t2 : 0;
#pragma unroll
                for (int k = 0; k < n; ++k) {
                    nu[k] = act ? (FUSEP ? u_rw[gb + k * n2] : u_ro[gb + k * n2]) : 0.0;
                    if (FUSEP) nr[k] = act ? r_in[gb + k * n2] : 0.0;
                }
            };
            if (C::PF == 1) prefetch();
            // P4: D^T along the row (B in place), the column (C in place) and the pencil (wt -> rw), one pass
            double rw[n];
            {
                double ln[3][n];
#pragma unroll
                for (int m = 0; m < n; ++m) {
                    ln[0][m] = sB[rbase + m];
                    ln[1][m] = sC[cbase + m * S1];
                    ln[2][m] = wt[m];
                }
                lines_apply<n, TOFF, 3, C::IB>(ln, [&](int q, int i, double v) {
                    if (q == 0) { if (mapped) sB[rbase + i] = v; }
                    else if (q == 1) { if (mapped) sC[cbase + i * S1] = v; }
                    else rw[i] = v;
                });
            }
            group_sync<GTH>(grp);
            if (C::PF == 2) prefetch();
            // P5: sum the three directions, store
#pragma unroll
            for (int k = 0; k < n; ++k) {
                const double wv = rw[k] + (sB[pbase + k * S2] + sC[pbase + k * S2]);
                if (active) w[gbase + k * n2] = wv;
            }
            // (no barrier here even when C aliases A: P5 reads and the next P1 writes the same pencil
            //  positions, by the same thread)
            if (C::PF == 0) prefetch();
        }
    }
    if (dot) nk_grid_reduce(dsum, s_red, red, NK_EPI_PAP, nullptr);
}

template <int N>
cudaError_t launch_tma(nk_ctx *c, double *u_rw, const double *u_ro, const double *r_in, double *w, int dot,
                       cudaStream_t st)
{
    using C = TmaCfg<N>;
    const int64_t nb = (c->E + C::EPB - 1) / C::EPB;
    const unsigned grid = (unsigned)(nb < (int64_t)c->sm_count ? nb : (int64_t)c->sm_count);   // one CTA per SM
    cudaError_t e;
    if (r_in != nullptr)
        e = nk_launch(ax_tma_kernel<N, true>, grid, C::THREADS, C::SMEM, st, c->pdl_now, u_rw, (const double *)nullptr, r_in, w,
                      (const double2 *)c->g, c->E, dot, c->red);
    else
        e = nk_launch(ax_tma_kernel<N, false>, grid, C::THREADS, C::SMEM, st, c->pdl_now, (double *)nullptr, u_ro,
                      (const double *)nullptr, w, (const double2 *)c->g, c->E, dot, c->red);
    c->launches++;
    return e != cudaSuccess ? e : cudaGetLastError();
}

// Row and column assignment of one order (TmaCfg: the layout it serves).  The lines of a sync group -- rows at
// s NW SE + n j + S2 k, columns at s NW SE + i + S2 k, slot s of the group -- are dealt to the group's threads
// half-warp by half-warp, each half-warp taking lines from the 16-bank residue classes that have most lines left:
// 16 different banks as long as no class holds more lines than there are half-warps, which plane_pad arranges.
template <int N>
void line_tables(uint16_t (*lut)[LUT_MAX])
{
    using C = TmaCfg<N>;
    constexpr int n = C::n, n2 = C::n2, lines = C::SG * n2;
    static_assert(lines <= LUT_MAX && C::GTH <= LUT_MAX, "line table too small");
    static_assert((C::SG - 1) * C::NW * C::SE + n * C::S2 < 65536, "line offsets exceed 16 bits");
    for (int which = 0; which < 2; ++which) {
        int start[LUT_MAX];
        bool used[LUT_MAX] = {};
        for (int s = 0; s < C::SG; ++s)
            for (int k = 0; k < n; ++k)
                for (int a = 0; a < n; ++a)
                    start[(s * n + k) * n + a] = s * C::NW * C::SE + (which ? a : n * a) + C::S2 * k;
        for (int t = 0; t < LUT_MAX; ++t) lut[which][t] = 0;
        for (int h0 = 0; h0 < lines; h0 += 16) {
            const int want = lines - h0 < 16 ? lines - h0 : 16;
            bool bank_taken[16] = {};
            for (int got = 0; got < want; ++got) {
                int left[16] = {};
                for (int q = 0; q < lines; ++q)
                    if (!used[q]) ++left[start[q] & 15];
                int bank = -1;
                for (int b = 0; b < 16; ++b)
                    if (left[b] > 0 && !bank_taken[b] && (bank < 0 || left[b] > left[bank])) bank = b;
                if (bank < 0)                                   // every free bank is exhausted: accept a conflict
                    for (int b = 0; b < 16; ++b)
                        if (left[b] > 0 && (bank < 0 || left[b] > left[bank])) bank = b;
                int pick = -1;
                for (int q = 0; q < lines && pick < 0; ++q)
                    if (!used[q] && (start[q] & 15) == bank) pick = q;
                used[pick] = true;
                bank_taken[bank] = true;
                lut[which][h0 + got] = (uint16_t)start[pick];
            }
        }
    }
}

template <int N>
cudaError_t prepare_tma()
{
    cudaError_t e = cudaFuncSetAttribute(ax_tma_kernel<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         TmaCfg<N>::SMEM);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(ax_tma_kernel<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                TmaCfg<N>::SMEM);
}

}  // namespace

cudaError_t nk_upload_D_tables_tma(void)
{
    static double h[D_TOTAL];
    double xi[16], wq[16];
    for (int N = 1; N <= NK_MAX_ORDER; ++N) {
        const int n = N + 1, hh = n / 2, H = (n + 1) / 2, ROW = eo_row(n);
        double D[16 * 16];
        nk_host_basis(N, xi, wq, D);
        for (int t = 0; t < 2; ++t) {                  // t = 0: M = D, t = 1: M = D^T
            double *tab = h + eo_off(n) + t * eo_mat(n);
            for (int i = 0; i < H; ++i)
                for (int m = 0; m < H; ++m) {
                    const double a = t ? D[m * n + i] : D[i * n + m];
                    const double b = t ? D[(n - 1 - m) * n + i] : D[i * n + (n - 1 - m)];
                    if (m < hh) {
                        tab[i * ROW + m] = 0.5 * (a - b);
                        tab[i * ROW + hh + m] = 0.5 * (a + b);
                    } else {
                        tab[i * ROW + hh + m] = a;     // middle column of an odd n
                    }
                }
        }
    }
    cudaError_t e = cudaMemcpyToSymbol(c_Dt, h, sizeof(h));
    if (e != cudaSuccess) return e;
    static uint16_t lut[NK_MAX_ORDER + 1][2][LUT_MAX];
#define NK_CASE(NN) line_tables<NN>(lut[NN]);
    NK_CASE(1) NK_CASE(2) NK_CASE(3) NK_CASE(4) NK_CASE(5) NK_CASE(6) NK_CASE(7) NK_CASE(8)
    NK_CASE(9) NK_CASE(10) NK_CASE(11) NK_CASE(12) NK_CASE(13) NK_CASE(14) NK_CASE(15)
#undef NK_CASE
    if ((e = cudaMemcpyToSymbol(c_lut, lut, sizeof(lut))) != cudaSuccess) return e;
#define NK_CASE(NN) if ((e = prepare_tma<NN>()) != cudaSuccess) return e;
    NK_CASE(1) NK_CASE(2) NK_CASE(3) NK_CASE(4) NK_CASE(5) NK_CASE(6) NK_CASE(7) NK_CASE(8)
    NK_CASE(9) NK_CASE(10) NK_CASE(11) NK_CASE(12) NK_CASE(13) NK_CASE(14) NK_CASE(15)
#undef NK_CASE
    return cudaSuccess;
}

int nk_ax_tma_epb(int N)
{
    return (N >= 1 && N <= NK_MAX_ORDER) ? tma_epb(N + 1) : 0;
}

cudaError_t nk_launch_ax_tma(nk_ctx *c, double *u_rw, const double *u_ro, const double *r_in, double *w, int dot,
                             cudaStream_t st)
{
    switch (c->N) {
#define NK_CASE(NN) case NN: return launch_tma<NN>(c, u_rw, u_ro, r_in, w, dot, st);
        NK_CASE(1) NK_CASE(2) NK_CASE(3) NK_CASE(4) NK_CASE(5) NK_CASE(6) NK_CASE(7) NK_CASE(8)
        NK_CASE(9) NK_CASE(10) NK_CASE(11) NK_CASE(12) NK_CASE(13) NK_CASE(14) NK_CASE(15)
#undef NK_CASE
    }
    return cudaErrorInvalidValue;
}
