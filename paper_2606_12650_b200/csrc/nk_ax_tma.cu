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
#include <cstdio>

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
    // where the next batch's u pencil is requested: 1 = after P3, 2 = after P4, 0 = after P5.  1 nearly everywhere: since the
    // producer prefetches u into L2 (ax_produce) n = 12 is spill-free at 160 registers with it and gains 6 % over 2
    // (16^3: 77.5 -> 72.5 us; before that prefetch 1 cost 4 % there).
#if defined(NK_TMA_PF_N) && defined(NK_TMA_PF_VAL)
    static constexpr int PF = (n == NK_TMA_PF_N) ? NK_TMA_PF_VAL : (n == 15 ? 2 : 1);   // A/B knob: one order, another position
#else
    static constexpr int PF = (n == 15) ? 2 : 1;     // n = 15 spills 104 B with 1, 72 B with 2: 186 -> 176 us at 16^3
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
// the 16-byte-aligned part of [p, p + bytes) into L2, nothing else: no destination, no barrier, no register
__device__ __forceinline__ void bulk_prefetch_l2(const void *p, uint32_t bytes)
{
    const uintptr_t a = (reinterpret_cast<uintptr_t>(p) + 15u) & ~(uintptr_t)15u;
    const uintptr_t e = (reinterpret_cast<uintptr_t>(p) + bytes) & ~(uintptr_t)15u;
    if (e > a)
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(a), "r"((uint32_t)(e - a)) : "memory");
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

// ---- the two halves of one application of ax_e, as device functions ---------------------------------------
// (ax_tma_kernel below runs them once; cg_coop_kernel once per CG iteration with the ring state carried over)
struct RingState { int stage; uint32_t phase; };

template <int N>
struct AxSmem {                 // carve-up of the dynamic shared memory (the same in every kernel of this file)
    using C = TmaCfg<N>;
    const double2 *ring;
    double *work;
    uint32_t ring0, full0, empty0;
    __device__ __forceinline__ explicit AxSmem(unsigned char *raw)
    {
        ring = reinterpret_cast<const double2 *>(raw);
        work = reinterpret_cast<double *>(raw + (size_t)C::R * C::STAGE_BYTES);
        ring0 = smem_u32(raw);
        full0 = ring0 + C::R * C::STAGE_BYTES + C::WORK_BYTES;
        empty0 = full0 + 8 * C::R;
    }
    __device__ __forceinline__ void init_barriers() const      // one thread, before the CTA's first barrier
    {
        for (int s = 0; s < C::R; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, C::CW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
};

// Producer lane: the geometric factors of elements [elo, ehi) into the ring, batch by batch.
// pf0, pf1 (may be null): the vectors the compute warps read their pencils from.  When the producer starts on the
// factors of a batch it also asks for that batch's part of these vectors to be brought into L2 (bulk prefetch: no
// destination, no register), so that the compute warps' loads, issued a phase or two later, find them there instead
// of paying the DRAM latency at the head of every batch.  (Stale data is harmless: L2 is the point of coherence.)
#ifndef NK_TMA_UPF
#define NK_TMA_UPF 1
#endif
template <int N>
__device__ __forceinline__ void ax_produce(const AxSmem<N> &sm, const double2 *__restrict__ g, int64_t elo, int64_t ehi,
                                           RingState &rs, const double *pf0 = nullptr, const double *pf1 = nullptr)
{
    using C = TmaCfg<N>;
    constexpr int n = C::n, n2 = C::n2, P = C::P, EPB = C::EPB, R = C::R, KP = C::KP;
    const int nit = (int)((ehi - elo + EPB - 1) / EPB);
    for (int it = 0; it < nit; ++it) {
        const int64_t e0 = elo + (int64_t)it * EPB;
        const int ne = (int)((ehi - e0 < EPB) ? (ehi - e0) : EPB);
        if (NK_TMA_UPF && it > 0) {                  // (the first batch too: no gain, measured)
            if (pf0) bulk_prefetch_l2(pf0 + e0 * P, (uint32_t)ne * P * 8);
            if (pf1) bulk_prefetch_l2(pf1 + e0 * P, (uint32_t)ne * P * 8);
        }
#pragma unroll 1
        for (int ks = 0; ks < C::SPB; ++ks) {
            mbar_wait(sm.empty0 + 8 * rs.stage, rs.phase ^ 1u);
            const uint32_t fb = sm.full0 + 8 * rs.stage, dst = sm.ring0 + rs.stage * C::STAGE_BYTES;
            if (KP == n) {       // whole elements: the batch is one contiguous chunk
                mbar_expect_tx(fb, (uint32_t)ne * P * 48);
                bulk_g2s(dst, g + nk_g_index(e0, 0, 0, 0, n), (uint32_t)ne * P * 48, fb);
            } else {             // KP consecutive k-planes (contiguous in HBM) of every element of the batch
                mbar_expect_tx(fb, (uint32_t)ne * KP * n2 * 48);
                for (int q = 0; q < ne; ++q)
                    bulk_g2s(dst + q * KP * n2 * 48, g + nk_g_index(e0 + q, ks * KP, 0, 0, n), KP * n2 * 48, fb);
            }
            if (++rs.stage == R) { rs.stage = 0; rs.phase ^= 1u; }
        }
    }
}

// vectors other SMs wrote earlier in the SAME launch (cg_coop_kernel) are read past the L1
template <bool CG>
__device__ __forceinline__ double ld_vec(const double *p) { return CG ? __ldcg(p) : *p; }

// Compute warps: w = A_L u on elements [elo, ehi); returns the thread's share of sum_l u_l (A_L u)_l.
// (u_rw, u_ro, r_in are what a predecessor wrote: no `const __restrict__` pair, or their loads could be hoisted
//  above the caller's griddepcontrol.wait as invariant -- see nk_vec.cu.)
// FUSEP: u = r_in + beta u is applied while loading and written to u_rw; the old u is read from u_ro if that is given
// (out of place: the "defer_x" pairs keep the previous direction), else from u_rw.  CG: see ld_vec.
// No arithmetic below sits under a thread-dependent branch: D reaches the DFMAs through the uniform datapath
// (LDCU -> UR operand), which ptxas only uses in warp-uniform code.  Threads without an element (ragged last
// warp, tail batch) compute on stale shared memory and only their stores are predicated off.
template <int N, bool FUSEP, bool CG>
__device__ __forceinline__ double ax_compute(const AxSmem<N> &sm, double *u_rw, const double *u_ro,
                                             const double *r_in, double *__restrict__ w, double beta,
                                             int64_t elo, int64_t ehi, RingState &rs)
{
    using C = TmaCfg<N>;
    constexpr int n = C::n, n2 = C::n2, P = C::P, S1 = C::S1, S2 = C::S2, SE = C::SE, EPB = C::EPB;
    constexpr int R = C::R, KP = C::KP, NW = C::NW, GTH = C::GTH, SG = C::SG;
    constexpr int PF = (CG && n == 12) ? 2 : C::PF;   // the cooperative solve at n = 12 spills with 1 (its vectors sit in L2 anyway)
    constexpr int DOFF = eo_off(n), TOFF = DOFF + eo_mat(n);     // even-odd tables of D and D^T in c_Dt
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int grp = tid / GTH, lt = tid - grp * GTH;
    const int sl = lt / n2, t2 = lt - sl * n2;
    const bool mapped = sl < SG;
    const int slot = grp * SG + (mapped ? sl : 0);
    // work arrays of the sync group's first slot; slot s of the group sits s NW SE doubles further on
    double *sA = sm.work + (size_t)(grp * SG) * NW * SE;           // u, then (NW = 2) the s direction
    double *sB = sA + SE;                                          // r direction
    double *sC = (NW == 3) ? sB + SE : sA;                         // s direction
    const int pbase = (mapped ? sl : 0) * NW * SE + t2;            // pencil (i,j) of the thread's slot: + k*S2
    const int rbase = c_lut[N][0][lt];                             // a row (j,k) of the group: + i
    const int cbase = c_lut[N][1][lt];                             // a column (i,k) of the group: + j*S1
    const double2 *gslot = sm.ring + slot * KP * 3 * n2 + t2;
    const int nit = (int)((ehi - elo + EPB - 1) / EPB);
    double dsum = 0.0;
    const double *uin = FUSEP ? (u_ro ? u_ro : u_rw) : u_ro;

    double nu[n], nr[FUSEP ? n : 1];               // next batch's pencil, in flight
    {
        const int64_t e = elo + slot;
        const bool act = mapped && e < ehi;
        const int64_t gb = act ? e * P + t2 : 0;
#pragma unroll
        for (int k = 0; k < n; ++k) {
            nu[k] = act ? ld_vec<CG>(uin + gb + k * n2) : 0.0;
            if (FUSEP) nr[k] = act ? ld_vec<CG>(r_in + gb + k * n2) : 0.0;
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
                if (k % KP == 0) mbar_wait_warp(sm.full0 + 8 * rs.stage, rs.phase);
                const double2 *gs = gslot + (size_t)rs.stage * C::STAGE_D2 + (k % KP) * 3 * n2;
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
                    if (lane == 0) mbar_arrive(sm.empty0 + 8 * rs.stage);
                    if (++rs.stage == R) { rs.stage = 0; rs.phase ^= 1u; }
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
                nu[k] = act ? ld_vec<CG>(uin + gb + k * n2) : 0.0;
                if (FUSEP) nr[k] = act ? ld_vec<CG>(r_in + gb + k * n2) : 0.0;
            }
        };
        if (PF == 1) prefetch();
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
        if (PF == 2) prefetch();
        // P5: sum the three directions, store
#pragma unroll
        for (int k = 0; k < n; ++k) {
            const double wv = rw[k] + (sB[pbase + k * S2] + sC[pbase + k * S2]);
            if (active) w[gbase + k * n2] = wv;
        }
        // (no barrier here even when C aliases A: P5 reads and the next P1 writes the same pencil
        //  positions, by the same thread)
        if (PF == 0) prefetch();
    }
    return dsum;
}

template <int N, bool FUSEP>
__global__ void __launch_bounds__(TmaCfg<N>::THREADS, 1)
ax_tma_kernel(double *u_rw, const double *u_ro, const double *r_in,
              double *__restrict__ w, const double2 *__restrict__ g, int64_t e_begin, int64_t E, int dot, nk_reduce_ws red)
{
    using C = TmaCfg<N>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ double s_red[34];
    const AxSmem<N> sm(smem_raw);
    const int tid = threadIdx.x;
    if (tid == 0) sm.init_barriers();
    __syncthreads();

    // This CTA's elements: a contiguous range, equal over the CTAs to within one element (batches dealt round
    // robin left the last round 1/4 full on a 16^3 mesh at N = 9: one batch time of 10 lost).  The last batch of
    // a range may be partial.
    // (E elements starting at e_begin: the whole mesh, or the interface / interior part of a rank's share)
    const int64_t elo = e_begin + E * (int64_t)blockIdx.x / gridDim.x, ehi = e_begin + E * ((int64_t)blockIdx.x + 1) / gridDim.x;
    double dsum = 0.0;
    if (C::WGP) {
        if (tid >= C::CT) asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
        else asm volatile("setmaxnreg.inc.sync.aligned.u32 240;");
    }
    RingState rs{0, 0u};
    if (tid >= C::CT) {
        // ---- producer warp: one lane streams G into the ring (static data: no need to wait for the predecessor)
        if (tid == C::CT) ax_produce<N>(sm, g, elo, ehi, rs, FUSEP ? (u_ro ? u_ro : u_rw) : u_ro, FUSEP ? r_in : nullptr);
    } else {
        nk_pdl_wait();                                  // u, r, beta come from the preceding kernels
        const double beta = FUSEP ? red.scal[NK_S_BETA] : 0.0;
        dsum = ax_compute<N, FUSEP, false>(sm, u_rw, u_ro, r_in, w, beta, elo, ehi, rs);
    }
    if (dot) nk_grid_reduce(dsum, s_red, red, NK_EPI_PAP, nullptr);
}

// ---- the whole CG solve as ONE cooperative launch (small, L2-resident meshes) ------------------------------
// (S 8(f) f-1 "or a persistent cooperative kernel"; PAPER.md:320 performance only saturates from 4e6 DOFs on,
// PAPER.md:328 per-call overhead separates the implementations below that.)  On meshes that fit in L2 an
// iteration is a few microseconds of work; launched kernel by kernel -- even as a CUDA graph of programmatic
// dependents -- it costs 11-16 us.  Here one persistent CTA per SM runs all `niter` iterations: per iteration
//   phase A  ax_e on the CTA's elements with p = r + beta p folded into the load and pap as the quadratic form
//   -- grid barrier; every CTA adds the per-CTA pap partials in the same order: alpha --
//   phase B  on the CTA's share of the points: x += alpha p; r -= alpha (M Q Q^T w), the copies of shared nodes
//            gathered on the fly from the unsummed w (nk_ctx::nbr, gx); rho' partial
//   -- grid barrier; every CTA adds the rho' partials in the same order: beta, residual history --
// Two barriers per iteration (hand-written: one monotone counter in global memory, arrive = atomicAdd, wait =
// ld.acquire until the count reaches blocks x barriers passed; measured ~2 us each, as a grid.sync.  A variant
// that carried the partial sums in the flag words themselves, LL-protocol style, polled by a whole warp, was
// SLOWER: 4-5 us per exchange).  The producer warp never joins a barrier: the
// geometric factors are static, so it streams the NEXT iteration's first batches into the ring while the compute
// warps are in phase B -- the ring is full when phase A starts.  Vectors another SM may have written during the
// launch are read past the L1 (ld.global.cg).  Sums are deterministic (fixed ranges, fixed trees); the order
// differs from the launch-by-launch path, so the two agree to rounding, not bitwise.
struct nk_coop_args {
    const double *f;
    double *x, *r, *p, *w;
    const double2 *g;
    const uint8_t *code;
    const double *ctab;
    const int32_t *nbr, *gx, *gx_rows;   // nk_ctx: gather codes, index rows of nodes with >= 3 copies, their list
    int64_t n_gx_rows;
    double *hist, *part, *scal;        // part: 2 x gridDim partial sums (alternating); scal: nk_reduce_ws::scal
    unsigned *bar;                     // barrier counter, zeroed by the host before the launch
    int64_t E, L;
    int niter;
};

template <int CT>
__device__ __forceinline__ void coop_cta_sync() { asm volatile("bar.sync 15, %0;" ::"n"(CT) : "memory"); }

// all compute threads of all CTAs; `passed` counts the barriers this CTA has been through
template <int CT>
__device__ __forceinline__ void coop_grid_barrier(unsigned *bar, unsigned &passed)
{
    coop_cta_sync<CT>();
    if (threadIdx.x == 0) {
        const unsigned target = gridDim.x * (passed + 1u);
        __threadfence();
        atomicAdd(bar, 1u);
        unsigned seen;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(bar) : "memory");
        } while (seen < target);
        __threadfence();
    }
    coop_cta_sync<CT>();
    ++passed;
}

// Sum of v over all compute threads of all CTAs, the same bits in every thread of every CTA.  `s_red`: 34 doubles.
// Two CTA barriers per exchange: warp 0 alone talks to the other CTAs -- lane 0 stores the CTA's partial, arrives
// with a release reduction (which orders that store and, through the CTA barrier before it, everything the CTA wrote
// in the phase), polls the counter with acquire loads; then the warp adds all partials in index order.  The result
// slot alternates with the parity of the exchange, so no third barrier is needed before s_red is reused.
#ifndef NK_COOP_SUM_V2
#define NK_COOP_SUM_V2 1
#endif
template <int CT>
__device__ __forceinline__ double coop_grid_sum(double v, double *s_red, double *part, unsigned *bar, unsigned &passed)
{
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    constexpr int NWARP = CT / 32;
    v = nk_warp_sum(v);
    if (lane == 0) s_red[wid] = v;
    coop_cta_sync<CT>();
    double *mine = part + (size_t)(passed & 1u) * gridDim.x;
#if NK_COOP_SUM_V2
    const int slot = 32 + (int)(passed & 1u);
    if (wid == 0) {
        double t = (lane < NWARP) ? s_red[lane] : 0.0;
        t = nk_warp_sum(t);
        if (lane == 0) {
            __stcg(mine + blockIdx.x, t);
            const unsigned target = gridDim.x * (passed + 1u);
            asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
            unsigned seen;
            do {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(bar) : "memory");
            } while (seen < target);
        }
        __syncwarp();
        double sum = 0.0;
        for (unsigned i = lane; i < gridDim.x; i += 32) sum += __ldcg(mine + i);
        sum = nk_warp_sum(sum);
        if (lane == 0) s_red[slot] = sum;
    }
    coop_cta_sync<CT>();
    ++passed;
    return s_red[slot];
#else
    if (wid == 0) {
        double t = (lane < NWARP) ? s_red[lane] : 0.0;
        t = nk_warp_sum(t);
        if (lane == 0) __stcg(mine + blockIdx.x, t);
    }
    coop_grid_barrier<CT>(bar, passed);            // (`mine` was picked before `passed` moved on)
    if (wid == 0) {
        double t = 0.0;
        for (unsigned i = lane; i < gridDim.x; i += 32) t += __ldcg(mine + i);
        t = nk_warp_sum(t);
        if (lane == 0) s_red[32] = t;
    }
    coop_cta_sync<CT>();
    const double total = s_red[32];
    coop_cta_sync<CT>();                           // s_red is free again
    return total;
#endif
}

// The same for ONE THREAD-BLOCK CLUSTER of CS CTAs (meshes of a few thousand points: a handful of CTAs has all the
// parallelism there is, and a cluster exchange costs a fraction of a grid barrier).  Every CTA stores its partial sum
// into slot [rank] of EVERY CTA's shared memory (distributed shared memory) and arrives, with release semantics at
// cluster scope, on every CTA's mbarrier; each CTA waits on its own mbarrier (CS arrivals per phase) and adds the CS
// partials in rank order.  Two slot arrays alternate as in coop_grid_sum.  No all-thread cluster barrier is used:
// the producer lane never joins.
constexpr int COOP_CS = 16;

__device__ __forceinline__ uint32_t mapa_u32(uint32_t addr, uint32_t cta)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(cta));
    return r;
}

template <int CT>
__device__ __forceinline__ double coop_cluster_sum(double v, double *s_red, double *s_part, uint32_t cbar, unsigned &passed)
{
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    constexpr int NWARP = CT / 32;
    v = nk_warp_sum(v);
    if (lane == 0) s_red[wid] = v;
    const unsigned e = passed++;                       // exchange number, from 0
    double *mine = s_part + (e & 1u) * COOP_CS;
    coop_cta_sync<CT>();                               // the CTA's writes of this phase happen-before the release below
    if (wid == 0) {
        double t = (lane < NWARP) ? s_red[lane] : 0.0;
        t = nk_warp_sum(t);
        if (lane < (int)gridDim.x) {
            const uint32_t slot = mapa_u32(smem_u32(mine + blockIdx.x), (uint32_t)lane);
            const uint32_t rbar = mapa_u32(cbar, (uint32_t)lane);
            asm volatile("st.shared::cluster.f64 [%0], %1;" ::"r"(slot), "d"(t) : "memory");
            asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(rbar) : "memory");
        }
        uint32_t done;
        do {
            asm volatile("{\n.reg .pred P1;\n"
                         "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 P1, [%1], %2;\n"
                         "selp.u32 %0, 1, 0, P1;\n}\n" : "=r"(done) : "r"(cbar), "r"(e & 1u) : "memory");
        } while (!__all_sync(0xffffffffu, done));
        if (lane == 0) {
            double sum = mine[0];
            for (unsigned i = 1; i < gridDim.x; ++i) sum += mine[i];
            s_red[32] = sum;
        }
    }
    coop_cta_sync<CT>();
    return s_red[32];
}

// (M Q Q^T w)_l of a streamed point from the unsummed w: own value / face partner g / Dirichlet.  Points of nodes
// with three or more copies (v < -1) are left to coop_row_update: `skip`.
__device__ __forceinline__ double coop_gs_value(int l, int v, double wl, double g, bool &skip)
{
    skip = v < -1;
    const double sum = v > l ? wl + g : g + wl;              // ascending local index
    return (v == l) ? wl : (v >= 0 ? sum : 0.0);
}

// One node with three or more copies (edges, corners): gather w (past the L1) and r at all copies, sum in ascending
// local index, r -= alpha sum at every copy; returns the node's share of rho'.  One thread per node, so that the
// dependent loads of many nodes overlap (inlined per point they serialised behind each other: 10 us per phase).
// (len, ia: the row's length and first four indices -- static, so a thread keeps those of its first row in registers
//  for the whole solve and the phase pays one memory round trip for the row instead of three.)
__device__ __forceinline__ double coop_row_update(const double *w, double *r, const int32_t *__restrict__ gx, int p4,
                                                  int len, int4 ia, double alpha, const double (&cw_of_len)[9])
{
    const int32_t *ii = gx + 4 * (int64_t)p4;
    double acc = 0.0;
    if (len == 4) {
        const double a0 = __ldcg(w + ia.x), a1 = __ldcg(w + ia.y), a2 = __ldcg(w + ia.z), a3 = __ldcg(w + ia.w);
        double r0 = r[ia.x], r1 = r[ia.y], r2 = r[ia.z], r3 = r[ia.w];
        const double s = ((a0 + a1) + a2) + a3, cw = cw_of_len[4];
        r0 = fma(-alpha, s, r0); r1 = fma(-alpha, s, r1); r2 = fma(-alpha, s, r2); r3 = fma(-alpha, s, r3);
        r[ia.x] = r0; r[ia.y] = r1; r[ia.z] = r2; r[ia.w] = r3;
        acc = fma(cw * r0, r0, acc); acc = fma(cw * r1, r1, acc); acc = fma(cw * r2, r2, acc); acc = fma(cw * r3, r3, acc);
        return acc;
    }
    const int4 ib = *reinterpret_cast<const int4 *>(ii + 4);
    const int id[8] = {ia.x, ia.y, ia.z, ia.w, ib.x, ib.y, ib.z, ib.w};
    double av[8], rr[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) { av[j] = (j < len) ? __ldcg(w + id[j]) : 0.0; rr[j] = (j < len) ? r[id[j]] : 0.0; }
    double s = av[0];
#pragma unroll
    for (int j = 1; j < 8; ++j) s = (j < len) ? s + av[j] : s;
    for (int j = 8; j < len; ++j) s += __ldcg(w + ii[j]);
    double cw = 1.0 / (double)len;
#pragma unroll
    for (int j = 1; j < 9; ++j) cw = (len == j) ? cw_of_len[j] : cw;
#pragma unroll
    for (int j = 0; j < 8; ++j)
        if (j < len) { const double rn = fma(-alpha, s, rr[j]); r[id[j]] = rn; acc = fma(cw * rn, rn, acc); }
    for (int j = 8; j < len; ++j) { const double rn = fma(-alpha, s, r[ii[j]]); r[ii[j]] = rn; acc = fma(cw * rn, rn, acc); }
    return acc;
}

template <int N, bool CLUSTER>
__global__ void __launch_bounds__(TmaCfg<N>::THREADS, 1)
cg_coop_kernel(nk_coop_args a)
{
    using C = TmaCfg<N>;
    constexpr int CT = C::CT;
    __shared__ double s_part[2 * COOP_CS];
    __shared__ __align__(8) unsigned long long s_cbar;
    const uint32_t cbar = smem_u32(&s_cbar);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ double s_red[34];
    __shared__ double s_c[NK_CTAB];
    const AxSmem<N> sm(smem_raw);
    const int tid = threadIdx.x;
    if (tid == 0) {
        sm.init_barriers();
        if (CLUSTER) { mbar_init(cbar, gridDim.x); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
    }
    for (int t = tid; t < NK_CTAB; t += blockDim.x) s_c[t] = a.ctab[t];
    __syncthreads();
    if (CLUSTER) {                                     // every CTA's mbarrier exists before anybody arrives on it
        asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
        asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
    }
    auto grid_sum = [&](double v, unsigned &passed) {
        return CLUSTER ? coop_cluster_sum<CT>(v, s_red, s_part, cbar, passed) : coop_grid_sum<CT>(v, s_red, a.part, a.bar, passed);
    };
    const int64_t elo = a.E * (int64_t)blockIdx.x / gridDim.x, ehi = a.E * ((int64_t)blockIdx.x + 1) / gridDim.x;
    RingState rs{0, 0u};
    if (tid >= CT) {
        // producer: free-running over the iterations, held back only by the ring
        if (tid == CT)
            for (int k = 0; k < a.niter; ++k) ax_produce<N>(sm, a.g, elo, ehi, rs);
        return;
    }
    // this CTA's share of the vectors for the streaming phases: a contiguous range of pairs
    const int64_t pairs = a.L >> 1;
    const int64_t plo = pairs * (int64_t)blockIdx.x / gridDim.x, phi = pairs * ((int64_t)blockIdx.x + 1) / gridDim.x;
    const bool odd_tail = (a.L & 1) && blockIdx.x == gridDim.x - 1 && tid == 0;       // the last point of an odd L
    // ... and of the nodes with three or more copies (coop_row_update)
    const int64_t rlo = a.n_gx_rows * (int64_t)blockIdx.x / gridDim.x, rhi = a.n_gx_rows * ((int64_t)blockIdx.x + 1) / gridDim.x;
    double cw_of_len[9];
#pragma unroll
    for (int j = 0; j < 9; ++j) cw_of_len[j] = j ? 1.0 / (double)j : 0.0;      // = ctab of that multiplicity, bit for bit
    // the thread's first such node: where its row sits (static: kept in a register for the whole solve; its length and
    // first four copies are requested at the head of every phase B, ahead of the streaming loop)
    const int row0_p4 = (rlo + tid < rhi) ? a.gx_rows[rlo + tid] : -1;
    unsigned passed = 0;
    double *x2 = a.x, *r2 = a.r, *p2 = a.p;
    // ---- r = mask o f, x = 0, p = r, rho = <r,r>_c -------------------------------------------------------------
    double acc = 0.0;
    for (int64_t q = plo + tid; q < phi; q += CT) {
        double2 fv = reinterpret_cast<const double2 *>(a.f)[q];
        const uchar2 cd = reinterpret_cast<const uchar2 *>(a.code)[q];
        if (cd.x & NK_CODE_MASKED) fv.x = 0.0;
        if (cd.y & NK_CODE_MASKED) fv.y = 0.0;
        reinterpret_cast<double2 *>(r2)[q] = fv;
        reinterpret_cast<double2 *>(p2)[q] = fv;
        reinterpret_cast<double2 *>(x2)[q] = make_double2(0.0, 0.0);
        acc = fma(s_c[cd.x & 0x7f] * fv.x, fv.x, acc);
        acc = fma(s_c[cd.y & 0x7f] * fv.y, fv.y, acc);
    }
    if (odd_tail) {
        const int64_t l = a.L - 1;
        const uint8_t cd = a.code[l];
        const double fv = (cd & NK_CODE_MASKED) ? 0.0 : a.f[l];
        r2[l] = fv; p2[l] = fv; x2[l] = 0.0;
        acc = fma(s_c[cd & 0x7f] * fv, fv, acc);
    }
    double rho = grid_sum(acc, passed);
    if (blockIdx.x == 0 && tid == 0) a.hist[0] = sqrt(rho);
    double beta = 0.0, alpha = 0.0, pap = 0.0, rho_old = rho;
    for (int k = 1; k <= a.niter; ++k) {
        // ---- phase A: w = A_L p with p = r + beta p folded in; pap ------------------------------------------------
#ifdef NK_COOP_TIMING
        unsigned long long tt[5];
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tt[0]));
#endif
        const double dsum = ax_compute<N, true, true>(sm, p2, nullptr, r2, a.w, beta, elo, ehi, rs);
#ifdef NK_COOP_TIMING
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tt[1]));
#endif
        pap = grid_sum(dsum, passed);
#ifdef NK_COOP_TIMING
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tt[2]));
#endif
        alpha = (rho == 0.0 || pap == 0.0) ? 0.0 : rho / pap;
        // ---- phase B: x += alpha p; r -= alpha M Q Q^T w; rho' ----------------------------------------------------
        acc = 0.0;
        const int row0_len = row0_p4 >= 0 ? a.gx[4 * (int64_t)row0_p4 - 1] : 0;
        const int4 row0_ia = row0_p4 >= 0 ? *reinterpret_cast<const int4 *>(a.gx + 4 * (int64_t)row0_p4) : make_int4(0, 0, 0, 0);
        for (int64_t q0 = plo + tid; q0 < phi; q0 += 4 * CT) {          // four pairs per thread in flight
            double2 pv[4], wv[4], xv[4], rv[4], gv[4];
            int2 nv[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int64_t q = q0 + j * CT;
                const bool on = q < phi;
                nv[j] = on ? reinterpret_cast<const int2 *>(a.nbr)[q] : make_int2(0, 0);
                pv[j] = on ? __ldcg(reinterpret_cast<const double2 *>(p2) + q) : make_double2(0.0, 0.0);
                wv[j] = on ? __ldcg(reinterpret_cast<const double2 *>(a.w) + q) : make_double2(0.0, 0.0);
                xv[j] = on ? reinterpret_cast<const double2 *>(x2)[q] : make_double2(0.0, 0.0);
                rv[j] = on ? reinterpret_cast<const double2 *>(r2)[q] : make_double2(0.0, 0.0);
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {                                  // the face partners, all at once
                const int l = (int)(2 * (q0 + j * CT));
                gv[j].x = (q0 + j * CT < phi && nv[j].x >= 0 && nv[j].x != l) ? __ldcg(a.w + nv[j].x) : 0.0;
                gv[j].y = (q0 + j * CT < phi && nv[j].y >= 0 && nv[j].y != l + 1) ? __ldcg(a.w + nv[j].y) : 0.0;
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int64_t q = q0 + j * CT;
                if (q < phi) {
                    const int l = (int)(2 * q);
                    bool k0, k1;
                    const double s0 = coop_gs_value(l, nv[j].x, wv[j].x, gv[j].x, k0);
                    const double s1 = coop_gs_value(l + 1, nv[j].y, wv[j].y, gv[j].y, k1);
                    xv[j].x = fma(alpha, pv[j].x, xv[j].x);
                    xv[j].y = fma(alpha, pv[j].y, xv[j].y);
                    rv[j].x = fma(-alpha, s0, rv[j].x);
                    rv[j].y = fma(-alpha, s1, rv[j].y);
                    reinterpret_cast<double2 *>(x2)[q] = xv[j];
                    if (!(k0 || k1)) {
                        reinterpret_cast<double2 *>(r2)[q] = rv[j];
                    } else {                                           // coop_row_update owns the other entry
                        if (!k0) r2[l] = rv[j].x;
                        if (!k1) r2[l + 1] = rv[j].y;
                    }
                    // weight 1 / multiplicity from the gather code: own copy 1, face partner 1/2 (nk_vec.cu gs_stream_weight)
                    acc = fma((k0 ? 0.0 : (nv[j].x == l ? 1.0 : 0.5)) * rv[j].x, rv[j].x, acc);
                    acc = fma((k1 ? 0.0 : (nv[j].y == l + 1 ? 1.0 : 0.5)) * rv[j].y, rv[j].y, acc);
                }
            }
        }
        if (row0_p4 >= 0) acc += coop_row_update(a.w, r2, a.gx, row0_p4, row0_len, row0_ia, alpha, cw_of_len);
        for (int64_t kr = rlo + tid + CT; kr < rhi; kr += CT) {
            const int p4 = a.gx_rows[kr];
            acc += coop_row_update(a.w, r2, a.gx, p4, a.gx[4 * (int64_t)p4 - 1], *reinterpret_cast<const int4 *>(a.gx + 4 * (int64_t)p4),
                                   alpha, cw_of_len);
        }
        if (odd_tail) {
            const int l = (int)(a.L - 1);
            const int vt = a.nbr[l];
            bool k0;
            const double s0 = coop_gs_value(l, vt, __ldcg(a.w + l), (vt >= 0 && vt != l) ? __ldcg(a.w + vt) : 0.0, k0);
            x2[l] = fma(alpha, __ldcg(p2 + l), x2[l]);
            if (!k0) {
                const double rn = fma(-alpha, s0, r2[l]);
                r2[l] = rn;
                acc = fma((vt == l ? 1.0 : 0.5) * rn, rn, acc);
            }
        }
#ifdef NK_COOP_TIMING
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tt[3]));
#endif
        const double rho_new = grid_sum(acc, passed);
#ifdef NK_COOP_TIMING
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tt[4]));
        if ((blockIdx.x == 0 || blockIdx.x == 77) && tid == 0 && (k == 5 || k == 6))
            printf("cta %d it %d: A %llu  sum1 %llu  B %llu  sum2 %llu ns\n", blockIdx.x, k, tt[1] - tt[0], tt[2] - tt[1], tt[3] - tt[2], tt[4] - tt[3]);
#endif
        beta = (rho == 0.0 || pap == 0.0) ? 0.0 : rho_new / rho;
        rho_old = rho;
        rho = rho_new;
        if (blockIdx.x == 0 && tid == 0) a.hist[k] = sqrt(rho_new);
    }
    // ---- leave the context as the launch-by-launch path does: p = r + beta p applied, scalars of the last step ----
    if (a.niter > 0) {
        for (int64_t q = plo + tid; q < phi; q += CT) {
            const double2 rv = reinterpret_cast<const double2 *>(r2)[q];
            double2 pv = __ldcg(reinterpret_cast<const double2 *>(p2) + q);
            pv.x = fma(beta, pv.x, rv.x);
            pv.y = fma(beta, pv.y, rv.y);
            reinterpret_cast<double2 *>(p2)[q] = pv;
        }
        if (odd_tail) { const int64_t l = a.L - 1; p2[l] = fma(beta, __ldcg(p2 + l), r2[l]); }
    }
    if (blockIdx.x == 0 && tid == 0) {
        a.scal[NK_S_RHO] = rho; a.scal[NK_S_RHO_OLD] = rho_old; a.scal[NK_S_RHO_NEW] = rho;
        a.scal[NK_S_PAP] = pap; a.scal[NK_S_ALPHA] = alpha; a.scal[NK_S_BETA] = beta;
    }
}

template <int N>
cudaError_t launch_coop(nk_ctx *c, const double *f, double *x, int niter, double *hist, cudaStream_t st)
{
    using C = TmaCfg<N>;
    nk_coop_args a;
    a.f = f; a.x = x; a.r = c->r; a.p = c->p; a.w = c->w; a.g = c->g;
    a.code = c->code; a.ctab = c->ctab; a.nbr = c->nbr; a.gx = c->gx; a.gx_rows = c->gx_rows; a.n_gx_rows = c->n_gx_rows;
    a.hist = hist; a.part = c->red.partials; a.scal = c->red.scal; a.bar = c->coop_bar;
    a.E = c->E; a.L = c->L; a.niter = niter;
    cudaError_t e;
    cudaLaunchConfig_t cfg = {};
    if (c->L <= NK_CLUSTER_AUTO_MAX_L && c->cluster_ok) {
        // a few thousand points: ONE cluster of COOP_CS CTAs, exchanges through distributed shared memory
        cfg.gridDim = dim3(COOP_CS); cfg.blockDim = dim3(C::THREADS);
        cfg.dynamicSmemBytes = C::SMEM; cfg.stream = st;
        cudaLaunchAttribute ac[1];
        ac[0].id = cudaLaunchAttributeClusterDimension;
        ac[0].val.clusterDim.x = COOP_CS; ac[0].val.clusterDim.y = 1; ac[0].val.clusterDim.z = 1;
        cfg.attrs = ac; cfg.numAttrs = 1;
        e = cudaLaunchKernelEx(&cfg, cg_coop_kernel<N, true>, a);
        if (e == cudaSuccess) { c->launches++; return cudaGetLastError(); }
        (void)cudaGetLastError();
        c->cluster_ok = 0;                                     // this device cannot place such a cluster: the grid variant from now on
    }
    e = cudaMemsetAsync(c->coop_bar, 0, sizeof(unsigned), st);
    if (e != cudaSuccess) return e;
    cfg = cudaLaunchConfig_t{};
    cfg.gridDim = dim3((unsigned)c->sm_count); cfg.blockDim = dim3(C::THREADS);
    cfg.dynamicSmemBytes = C::SMEM; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeCooperative;                 // all CTAs co-resident, or the launch fails
    at[0].val.cooperative = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    e = cudaLaunchKernelEx(&cfg, cg_coop_kernel<N, false>, a);
    c->launches++;
    return e != cudaSuccess ? e : cudaGetLastError();
}

template <int N>
cudaError_t launch_tma(nk_ctx *c, double *u_rw, const double *u_ro, const double *r_in, double *w, int dot,
                       int64_t e_begin, int64_t e_count, cudaStream_t st)
{
    using C = TmaCfg<N>;
    if (e_count <= 0) return cudaSuccess;
    const int64_t nb = (e_count + C::EPB - 1) / C::EPB;
    const unsigned grid = (unsigned)(nb < (int64_t)c->sm_count ? nb : (int64_t)c->sm_count);   // one CTA per SM
    cudaError_t e;
    if (r_in != nullptr)
        e = nk_launch(ax_tma_kernel<N, true>, grid, C::THREADS, C::SMEM, st, c->pdl_now, u_rw, u_ro, r_in, w,
                      (const double2 *)c->g, e_begin, e_count, dot, c->red);
    else
        e = nk_launch(ax_tma_kernel<N, false>, grid, C::THREADS, C::SMEM, st, c->pdl_now, (double *)nullptr, u_ro,
                      (const double *)nullptr, w, (const double2 *)c->g, e_begin, e_count, dot, c->red);
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
    e = cudaFuncSetAttribute(ax_tma_kernel<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, TmaCfg<N>::SMEM);
    if (e != cudaSuccess) return e;
    if constexpr (N <= 13) {         // nk_coop_supported
        e = cudaFuncSetAttribute(cg_coop_kernel<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, TmaCfg<N>::SMEM);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(cg_coop_kernel<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, TmaCfg<N>::SMEM);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(cg_coop_kernel<N, true>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    }
    return e;
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

// the whole solve as one cooperative launch (orders whose ax_e needs no register re-balancing: N <= 13)
int nk_coop_supported(int N) { return N >= 1 && N <= 13; }

cudaError_t nk_launch_cg_coop(nk_ctx *c, const double *f, double *x, int niter, double *hist, cudaStream_t st)
{
    switch (c->N) {
#define NK_CASE(NN) case NN: return launch_coop<NN>(c, f, x, niter, hist, st);
        NK_CASE(1) NK_CASE(2) NK_CASE(3) NK_CASE(4) NK_CASE(5) NK_CASE(6) NK_CASE(7) NK_CASE(8)
        NK_CASE(9) NK_CASE(10) NK_CASE(11) NK_CASE(12) NK_CASE(13)
#undef NK_CASE
    }
    return cudaErrorInvalidValue;
}

int nk_ax_tma_epb(int N)
{
    return (N >= 1 && N <= NK_MAX_ORDER) ? tma_epb(N + 1) : 0;
}

cudaError_t nk_launch_ax_tma(nk_ctx *c, double *u_rw, const double *u_ro, const double *r_in, double *w, int dot,
                             cudaStream_t st)
{
    return nk_launch_ax_tma_range(c, u_rw, u_ro, r_in, w, dot, 0, c->E, st);
}

cudaError_t nk_launch_ax_tma_range(nk_ctx *c, double *u_rw, const double *u_ro, const double *r_in, double *w, int dot,
                                   int64_t e_begin, int64_t e_count, cudaStream_t st)
{
    switch (c->N) {
#define NK_CASE(NN) case NN: return launch_tma<NN>(c, u_rw, u_ro, r_in, w, dot, e_begin, e_count, st);
        NK_CASE(1) NK_CASE(2) NK_CASE(3) NK_CASE(4) NK_CASE(5) NK_CASE(6) NK_CASE(7) NK_CASE(8)
        NK_CASE(9) NK_CASE(10) NK_CASE(11) NK_CASE(12) NK_CASE(13) NK_CASE(14) NK_CASE(15)
#undef NK_CASE
    }
    return cudaErrorInvalidValue;
}
