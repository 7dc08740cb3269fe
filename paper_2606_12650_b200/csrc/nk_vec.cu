// nk_vec.cu -- CG "streaming" and "reduction" kernels (Table V; S 8(a) a4-a7).
// Each kernel makes ONE pass over its vectors with 16-byte accesses, folds the dot product it
// needs into that pass, and finishes the reduction on the device (nk_reduce.cuh).  The inverse
// multiplicity c_l comes from a 1-byte code per point through a 128-entry table in shared memory
// (multiplicities on a hex mesh are a handful of small integers), so <a,b>_c costs 1 B/pt, not 8.
#include "nk_internal.h"
#include "nk_reduce.cuh"

namespace {

// Pointer qualifiers in this file: a kernel launched as a PROGRAMMATIC DEPENDENT starts while its predecessor
// still runs and reads the predecessor's output only after griddepcontrol.wait (nk_pdl_wait).  Such inputs (w, r,
// p, the scalar block) are plain `const double *`, never `const ... __restrict__`: that pair lets the compiler use
// non-coherent loads (LDG.CONSTANT), which it treats as invariant and hoists ABOVE the wait -- round 1's update_p
// fetched beta before its predecessor had written it (found by the cooperative path's state comparison).  Static
// set-up data (code, ctab, nbr, gx, dinv) keeps the qualifiers: fetching it before the wait is the point.
//
// Fixed grid => fixed partial sums => run-to-run bitwise reproducible.
inline int vec_blocks(const nk_ctx *c, int64_t pairs) { return nk_vec_blocks(c->sm_count, pairs); }

__device__ __forceinline__ void load_ctab(double *s_c, const double *ctab)
{
    for (int t = threadIdx.x; t < NK_CTAB; t += blockDim.x) s_c[t] = ctab[t];
    __syncthreads();
}

// out = <a,b>_c
__global__ void __launch_bounds__(NK_VEC_THREADS)
dot_kernel(const double *__restrict__ a, const double *__restrict__ b, const uint8_t *__restrict__ code,
           const double *__restrict__ ctab, int64_t L, nk_reduce_ws ws, int epi, double *out)
{
    __shared__ double s_c[NK_CTAB];
    __shared__ double s_red[33];
    load_ctab(s_c, ctab);
    const int64_t pairs = L >> 1;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    double acc = 0.0;
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < pairs; q += stride) {
        const double2 av = reinterpret_cast<const double2 *>(a)[q];
        const double2 bv = reinterpret_cast<const double2 *>(b)[q];
        const uchar2 cd = reinterpret_cast<const uchar2 *>(code)[q];
        acc = fma(s_c[cd.x & 0x7f] * av.x, bv.x, acc);
        acc = fma(s_c[cd.y & 0x7f] * av.y, bv.y, acc);
    }
    if ((L & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        const int64_t l = L - 1;
        acc = fma(s_c[code[l] & 0x7f] * a[l], b[l], acc);
    }
    nk_grid_reduce(acc, s_red, ws, epi, out);
}

// r = mask o f, x = 0, p = r, rho0 = <r,r>_c       (S 8(c) O8 initialisation)
__global__ void __launch_bounds__(NK_VEC_THREADS)
cg_init_kernel(const double *__restrict__ f, double *__restrict__ x, double *__restrict__ r,
               double *__restrict__ p, const uint8_t *__restrict__ code, const double *__restrict__ ctab,
               int64_t L, nk_reduce_ws ws, double *hist0)
{
    __shared__ double s_c[NK_CTAB];
    __shared__ double s_red[33];
    load_ctab(s_c, ctab);
    const int64_t pairs = L >> 1;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    double acc = 0.0;
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < pairs; q += stride) {
        double2 fv = reinterpret_cast<const double2 *>(f)[q];
        const uchar2 cd = reinterpret_cast<const uchar2 *>(code)[q];
        if (cd.x & NK_CODE_MASKED) fv.x = 0.0;
        if (cd.y & NK_CODE_MASKED) fv.y = 0.0;
        reinterpret_cast<double2 *>(r)[q] = fv;
        reinterpret_cast<double2 *>(p)[q] = fv;
        reinterpret_cast<double2 *>(x)[q] = make_double2(0.0, 0.0);
        acc = fma(s_c[cd.x & 0x7f] * fv.x, fv.x, acc);
        acc = fma(s_c[cd.y & 0x7f] * fv.y, fv.y, acc);
    }
    if ((L & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        const int64_t l = L - 1;
        const uint8_t cd = code[l];
        const double fv = (cd & NK_CODE_MASKED) ? 0.0 : f[l];
        r[l] = fv; p[l] = fv; x[l] = 0.0;
        acc = fma(s_c[cd & 0x7f] * fv, fv, acc);
    }
    nk_grid_reduce(acc, s_red, ws, NK_EPI_RHO0, hist0);
}

// x += alpha p; r -= alpha w; rho' = <r,r>_c          (S 8(a) a5: axpy, axpy and dot in one pass)
__global__ void __launch_bounds__(NK_VEC_THREADS)
update_xr_kernel(double *__restrict__ x, double *__restrict__ r, const double *p,
                 const double *w, const uint8_t *__restrict__ code,
                 const double *__restrict__ ctab, int64_t L, nk_reduce_ws ws, double *hist_k)
{
    __shared__ double s_c[NK_CTAB];
    __shared__ double s_red[33];
    nk_pdl_launch_dependents();
    load_ctab(s_c, ctab);
    nk_pdl_wait();
    const double alpha = ws.scal[NK_S_ALPHA];
    const int64_t pairs = L >> 1;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    double acc = 0.0;
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < pairs; q += stride) {
        const double2 pv = reinterpret_cast<const double2 *>(p)[q];
        const double2 wv = reinterpret_cast<const double2 *>(w)[q];
        double2 xv = reinterpret_cast<double2 *>(x)[q];
        double2 rv = reinterpret_cast<double2 *>(r)[q];
        const uchar2 cd = reinterpret_cast<const uchar2 *>(code)[q];
        xv.x = fma(alpha, pv.x, xv.x);
        xv.y = fma(alpha, pv.y, xv.y);
        rv.x = fma(-alpha, wv.x, rv.x);
        rv.y = fma(-alpha, wv.y, rv.y);
        reinterpret_cast<double2 *>(x)[q] = xv;
        reinterpret_cast<double2 *>(r)[q] = rv;
        acc = fma(s_c[cd.x & 0x7f] * rv.x, rv.x, acc);
        acc = fma(s_c[cd.y & 0x7f] * rv.y, rv.y, acc);
    }
    if ((L & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        const int64_t l = L - 1;
        const double xv = fma(alpha, p[l], x[l]);
        const double rv = fma(-alpha, w[l], r[l]);
        x[l] = xv; r[l] = rv;
        acc = fma(s_c[code[l] & 0x7f] * rv, rv, acc);
    }
    nk_grid_reduce(acc, s_red, ws, NK_EPI_RHO, hist_k);
}

// ---- gs and the mask folded into the residual update ("fuse_gs"; SURVEY 8(a) a2 + a3 + a5 in one pass) -------
// Inside CG the summed w = M Q Q^T A_L p is read exactly once, by r -= alpha w (pap comes out of ax_e as a
// quadratic form).  So w need never be summed IN PLACE: this kernel streams the UNSUMMED ax_e output and sums
// the copies of shared nodes on the fly.  gs's write-back (8 B per listed copy, 32 B where the copy is alone in
// its sector: the stride-n r-faces), its re-read by the update and one launch per iteration are gone.
// Every block takes a contiguous chunk of the vectors and does two things:
//   * it streams the chunk.  A point whose node has no other copy keeps its value; a point of a multiplicity-2
//     node (faces: 82 % of the shared points of a brick) adds its ONE partner, whose index nbr[l] was fetched one
//     step ahead so that the gather is issued together with the streaming loads; a Dirichlet point takes 0; a
//     point of a node with three or more copies (edges, corners) is SKIPPED;
//   * it then handles the nodes with three or more copies whose first copy lies in the chunk, one thread each:
//     gathers w and r of all copies (indices by vector load from gx), sums in ascending local index as nk_gs.cu
//     does, and updates r at every copy.  (Inlined into the streaming loop this work cost two dependent memory
//     round trips in nearly every warp -- one edge point among 32 lanes is enough -- and tripled the time of the
//     pass; given to blocks of their own, far from where the chunk's data is in L2, it cost 0.3 GB of DRAM traffic.)
// Blocks run in index order, so the resident ones form a window of some tens of MB that moves through the
// vectors once: partners 14 KB (r-faces), 0.4 MB (s-faces) or 14 MB (t-faces, config 5) away are L2 hits.
// The per-point multiplicity code is NOT read here: the weight of a streamed point follows from its gather code
// (gs_stream_weight), that of a node with several copies from their number.  Dropping that 1-byte stream (a 2-byte
// load per thread and step, a table in shared memory) took the pass from 365 to 333 us at config 5 -- it is bound by
// load instructions in flight, not by bytes.
// r, x are the values of nk_gs followed by the plain update, entry by entry; rho' sums the same terms in another
// (fixed) order.  Run-to-run bitwise reproducible like every reduction here.
struct nk_gather {
    const int32_t *nbr, *gx, *rows;     // nk_internal.h nk_ctx::nbr, gx; rows[k] = p of the k-th node with >= 3 copies
    const int32_t *blk;                 // rows [blk[b], blk[b+1]) have their first copy in block b's chunk of the vector
};

__device__ __forceinline__ double gs_partner(const double *w, int l, int v)
{
    return (v >= 0 && v != l) ? w[v] : 0.0;
}
// value of (M Q Q^T w)_l for a streamed point: own / face partner / Dirichlet; `skip` for the row blocks' points
__device__ __forceinline__ double gs_stream_value(int l, int v, double wl, double g, bool &skip)
{
    skip = v < -1;
    const double sum = (v > l) ? wl + g : g + wl;            // ascending local index
    return (v == l) ? wl : (v >= 0 ? sum : 0.0);
}

// The weight c = 1 / multiplicity of a streamed point follows from its gather code: 1 for a node with one copy, 1/2
// for a face node (exactly the table entries nk_setup builds as 1.0 / multiplicity), so the streaming loop does not
// read the per-point code at all.  A Dirichlet point (v = -1) has r = 0 in every state CG produces (r0 = M f, and
// M Q Q^T w = 0 there): its term vanishes whatever the weight.
__device__ __forceinline__ double gs_stream_weight(int l, int v, bool skip)
{
    return skip ? 0.0 : (v == l ? 1.0 : 0.5);
}

// one node with three or more copies: r -= alpha sum at every copy; returns its share of rho'
// (weight 1 / len: the correctly rounded quotient nk_setup stores in its table)
__device__ __forceinline__ double gs_row_update(const double *w, double *r, const int32_t *__restrict__ gx, int p4,
                                                double alpha)
{
    const int4 ia = reinterpret_cast<const int4 *>(gx)[p4];
    const int len = gx[4 * p4 - 1];
    double acc = 0.0;
    if (len == 4) {                                       // an edge of a conforming hex mesh
        const double a0 = w[ia.x], a1 = w[ia.y], a2 = w[ia.z], a3 = w[ia.w];
        double r0 = r[ia.x], r1 = r[ia.y], r2 = r[ia.z], r3 = r[ia.w];
        const double cw = 0.25;
        const double s = ((a0 + a1) + a2) + a3;
        r0 = fma(-alpha, s, r0); r1 = fma(-alpha, s, r1); r2 = fma(-alpha, s, r2); r3 = fma(-alpha, s, r3);
        r[ia.x] = r0; r[ia.y] = r1; r[ia.z] = r2; r[ia.w] = r3;
        acc = fma(cw * r0, r0, acc); acc = fma(cw * r1, r1, acc);
        acc = fma(cw * r2, r2, acc); acc = fma(cw * r3, r3, acc);
        return acc;
    }
    const int32_t *ii = gx + 4 * (int64_t)p4;
    double s = w[ii[0]];
    for (int j = 1; j < len; ++j) s += w[ii[j]];
    const double cw = 1.0 / (double)len;
    for (int j = 0; j < len; ++j) {
        const double rn = fma(-alpha, s, r[ii[j]]);
        r[ii[j]] = rn;
        acc = fma(cw * rn, rn, acc);
    }
    return acc;
}

// 256-bit global accesses (sm_100: LDG.E.256 / STG.E.256): four doubles per instruction, 32-byte aligned
struct double4v { double a, b, c, d; };
__device__ __forceinline__ double4v ld256(const double *p)
{
    double4v v;
    asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v.a), "=d"(v.b), "=d"(v.c), "=d"(v.d) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st256(double *p, const double4v &v)
{
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(v.a), "d"(v.b), "d"(v.c), "d"(v.d) : "memory");
}
__device__ __forceinline__ bool aligned32(const void *a, const void *b, const void *c)
{
    return ((reinterpret_cast<uintptr_t>(a) | reinterpret_cast<uintptr_t>(b) | reinterpret_cast<uintptr_t>(c)) & 31u) == 0;
}
#ifndef NK_V256
#define NK_V256 1
#endif

#ifndef NK_GSU_U
#define NK_GSU_U 1
#endif
#ifndef NK_GSU_UX
#define NK_GSU_UX 1                                      // ... and of the variant that also updates x (mid-size meshes)
#endif
constexpr int GS_U = NK_GSU_U;                           // QUADS (four consecutive points) per thread and step

__device__ __forceinline__ double4v ld4(const double *p, bool a32)
{
    if (a32) return ld256(p);
    const double2 lo = reinterpret_cast<const double2 *>(p)[0], hi = reinterpret_cast<const double2 *>(p)[1];
    double4v v;
    v.a = lo.x; v.b = lo.y; v.c = hi.x; v.d = hi.y;
    return v;
}
__device__ __forceinline__ void st4(double *p, const double4v &v, bool a32)
{
    if (a32) { st256(p, v); return; }
    reinterpret_cast<double2 *>(p)[0] = make_double2(v.a, v.b);
    reinterpret_cast<double2 *>(p)[1] = make_double2(v.c, v.d);
}

// one streamed point: r -= alpha (M Q Q^T w)_l, its share of rho'; `skip`: the point belongs to gs_row_update
__device__ __forceinline__ void gs_point(int l, int v, double wl, double g, double alpha, double &rl, bool &skip, double &acc)
{
    const double s = gs_stream_value(l, v, wl, g, skip);
    rl = fma(-alpha, s, rl);
    acc = fma(gs_stream_weight(l, v, skip) * rl, rl, acc);
}

// XM: what happens to x in the same pass.  0: nothing; 1: x += alpha p; 2: the deferred update of two iterations,
// x = fma(alpha, pb, fma(alpha_prev, p, x)) (nk_api.cu "defer_x" on the "fuse_p" path: p, pb = the directions of the
// first and second iteration of the pair).  stash != 0 (first of a pair): alpha is kept in NK_S_ALPHA_PREV.
template <int XM>
__global__ void __launch_bounds__(NK_GSU_THREADS, NK_GSU_MINB)
gs_update_kernel(double *__restrict__ x, double *r, const double *p, const double *pb, const double *w, int64_t L,
                 nk_reduce_ws ws, double *hist_k, nk_gather gp, int stash)
{
    constexpr bool WITH_X = XM != 0;
    __shared__ double s_red[33];
    nk_pdl_launch_dependents();
    double acc = 0.0;
    // this block's CONTIGUOUS chunk of quads (blocks run in index order, so the resident blocks form one window
    // that moves through the vectors: a partner a few KB or MB away is in L2 when it is gathered).  Four points per
    // thread and step through 256-bit loads and stores: the pass is bound by the load instructions in flight, not by
    // bytes (r, p, w live in the workspace, 256-byte aligned; the caller's x may only be 16-byte aligned).
    const int64_t quads = L >> 2;
    const int64_t qlo = quads * (int64_t)blockIdx.x / gridDim.x, qhi = quads * ((int64_t)blockIdx.x + 1) / gridDim.x;
    const int64_t stride = blockDim.x;
    constexpr int U = WITH_X ? NK_GSU_UX : GS_U;              // quads per step, all loads before the stores
    const bool x32 = WITH_X && (reinterpret_cast<uintptr_t>(x) & 31u) == 0;
    int64_t q = qlo + threadIdx.x;
    int4 nv[U];
#pragma unroll
    for (int j = 0; j < U; ++j)                               // gather codes of the first step: static, before the wait
        nv[j] = (q + j * stride < qhi) ? reinterpret_cast<const int4 *>(gp.nbr)[q + j * stride] : make_int4(0, 0, 0, 0);
    nk_pdl_wait();
    const double alpha = ws.scal[NK_S_ALPHA];
    const double alpha_prev = XM == 2 ? ws.scal[NK_S_ALPHA_PREV] : 0.0;
    if (stash && blockIdx.x == 0 && threadIdx.x == 0) ws.scal[NK_S_ALPHA_PREV] = alpha;   // the next ax_e overwrites alpha
    // (Staging the streamed operands through shared memory with cp.async, four pairs per thread in flight instead of
    //  two, was measured SLOWER: 394 vs 369 us at config 5.)
    for (; q < qhi; q += U * stride) {
        double4v wv[U], rv[U], g[U], xv[WITH_X ? U : 1], pv[WITH_X ? U : 1], qv[XM == 2 ? U : 1];
        int4 nn[U];
        bool on[U];
#pragma unroll
        for (int j = 0; j < U; ++j) {
            const int64_t qj = q + j * stride;
            on[j] = qj < qhi;
            if (on[j]) {
                const int l = (int)(4 * qj);
                wv[j] = ld256(w + 4 * qj);
                rv[j] = ld256(r + 4 * qj);
                g[j].a = gs_partner(w, l, nv[j].x);
                g[j].b = gs_partner(w, l + 1, nv[j].y);
                g[j].c = gs_partner(w, l + 2, nv[j].z);
                g[j].d = gs_partner(w, l + 3, nv[j].w);
                if (WITH_X) {
                    xv[WITH_X ? j : 0] = ld4(x + 4 * qj, x32);
                    pv[WITH_X ? j : 0] = ld256(p + 4 * qj);
                    if (XM == 2) qv[XM == 2 ? j : 0] = ld256(pb + 4 * qj);
                }
            }
        }
#pragma unroll
        for (int j = 0; j < U; ++j) {                         // next step's gather codes
            const int64_t qn = q + (U + j) * stride;
            nn[j] = (qn < qhi) ? reinterpret_cast<const int4 *>(gp.nbr)[qn] : make_int4(0, 0, 0, 0);
        }
#pragma unroll
        for (int j = 0; j < U; ++j) {
            if (on[j]) {
                const int64_t qj = q + j * stride;
                const int l = (int)(4 * qj);
                bool k0, k1, k2, k3;
                gs_point(l, nv[j].x, wv[j].a, g[j].a, alpha, rv[j].a, k0, acc);
                gs_point(l + 1, nv[j].y, wv[j].b, g[j].b, alpha, rv[j].b, k1, acc);
                gs_point(l + 2, nv[j].z, wv[j].c, g[j].c, alpha, rv[j].c, k2, acc);
                gs_point(l + 3, nv[j].w, wv[j].d, g[j].d, alpha, rv[j].d, k3, acc);
                if (!(k0 || k1 || k2 || k3)) {
                    st256(r + 4 * qj, rv[j]);
                } else {                                      // gs_row_update owns the skipped entries
                    if (!k0) r[l] = rv[j].a;
                    if (!k1) r[l + 1] = rv[j].b;
                    if (!k2) r[l + 2] = rv[j].c;
                    if (!k3) r[l + 3] = rv[j].d;
                }
                if (WITH_X) {
                    double4v xn = xv[WITH_X ? j : 0];
                    const double4v pj = pv[WITH_X ? j : 0];
                    if (XM == 2) {
                        const double4v qj2 = qv[XM == 2 ? j : 0];
                        xn.a = fma(alpha, qj2.a, fma(alpha_prev, pj.a, xn.a)); xn.b = fma(alpha, qj2.b, fma(alpha_prev, pj.b, xn.b));
                        xn.c = fma(alpha, qj2.c, fma(alpha_prev, pj.c, xn.c)); xn.d = fma(alpha, qj2.d, fma(alpha_prev, pj.d, xn.d));
                    } else {
                        xn.a = fma(alpha, pj.a, xn.a); xn.b = fma(alpha, pj.b, xn.b);
                        xn.c = fma(alpha, pj.c, xn.c); xn.d = fma(alpha, pj.d, xn.d);
                    }
                    st4(x + 4 * qj, xn, x32);
                }
            }
            nv[j] = nn[j];
        }
    }
    if (blockIdx.x == gridDim.x - 1 && (int64_t)threadIdx.x < (L & 3)) {    // up to three points past the last quad
        const int l = (int)((quads << 2) + threadIdx.x);
        const int v = gp.nbr[l];
        bool k0;
        double rl = r[l];
        double a0 = 0.0;
        gs_point(l, v, w[l], gs_partner(w, l, v), alpha, rl, k0, a0);
        if (!k0) { r[l] = rl; acc += a0; }
        if (XM == 1) x[l] = fma(alpha, p[l], x[l]);
        if (XM == 2) x[l] = fma(alpha, pb[l], fma(alpha_prev, p[l], x[l]));
    }
    // the nodes with three or more copies whose FIRST copy lies in this block's chunk (their other copies sit in
    // neighbouring chunks: in L2, just streamed or about to be), one thread each
    for (int k = gp.blk[blockIdx.x] + (int)threadIdx.x; k < gp.blk[blockIdx.x + 1]; k += blockDim.x)
        acc += gs_row_update(w, r, gp.gx, gp.rows[k], alpha);
    nk_grid_reduce(acc, s_red, ws, NK_EPI_RHO, hist_k);
}

// p = r + beta p                                       (S 8(a) a6)
__global__ void __launch_bounds__(NK_VEC_THREADS)
update_p_kernel(double *p, const double *pin, const double *r, const double *scal, int64_t L)   // pin == p: in place
{
    nk_pdl_launch_dependents();
    nk_pdl_wait();
    const double beta = scal[NK_S_BETA];
    const int64_t pairs = L >> 1;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < pairs; q += stride) {
        const double2 rv = reinterpret_cast<const double2 *>(r)[q];
        double2 pv = reinterpret_cast<const double2 *>(pin)[q];
        pv.x = fma(beta, pv.x, rv.x);
        pv.y = fma(beta, pv.y, rv.y);
        reinterpret_cast<double2 *>(p)[q] = pv;
    }
    if ((L & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        const int64_t l = L - 1;
        p[l] = fma(beta, pin[l], r[l]);
    }
}

// r -= alpha w; rho' = <r,r>_c.  With update_px_kernel below this is the un-fused iteration's vector
// work in 65 B/pt instead of 73: p is read once per iteration (by update_px, which still has the old
// p in registers when x needs it) instead of twice.  Same arithmetic per entry as update_xr_kernel.
__global__ void __launch_bounds__(NK_VEC_THREADS)
update_r_kernel(double *__restrict__ r, const double *w, const uint8_t *__restrict__ code,
                const double *__restrict__ ctab, int64_t L, nk_reduce_ws ws, double *hist_k)
{
    __shared__ double s_c[NK_CTAB];
    __shared__ double s_red[33];
    nk_pdl_launch_dependents();
    load_ctab(s_c, ctab);
    nk_pdl_wait();
    const double alpha = ws.scal[NK_S_ALPHA];
    const int64_t pairs = L >> 1;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    double acc = 0.0;
    // four pairs per step, all loads before the stores (r is loaded and stored through one pointer, so
    // the compiler will not overlap the next step's loads with this step's store on its own)
    int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; q + 3 * stride < pairs; q += 4 * stride) {
        double2 wv[4], rv[4];
        uchar2 cd[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            wv[j] = reinterpret_cast<const double2 *>(w)[q + j * stride];
            rv[j] = reinterpret_cast<double2 *>(r)[q + j * stride];
            cd[j] = reinterpret_cast<const uchar2 *>(code)[q + j * stride];
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            rv[j].x = fma(-alpha, wv[j].x, rv[j].x);
            rv[j].y = fma(-alpha, wv[j].y, rv[j].y);
            reinterpret_cast<double2 *>(r)[q + j * stride] = rv[j];
            acc = fma(s_c[cd[j].x & 0x7f] * rv[j].x, rv[j].x, acc);
            acc = fma(s_c[cd[j].y & 0x7f] * rv[j].y, rv[j].y, acc);
        }
    }
    for (; q < pairs; q += stride) {
        const double2 wv = reinterpret_cast<const double2 *>(w)[q];
        double2 rv = reinterpret_cast<double2 *>(r)[q];
        const uchar2 cd = reinterpret_cast<const uchar2 *>(code)[q];
        rv.x = fma(-alpha, wv.x, rv.x);
        rv.y = fma(-alpha, wv.y, rv.y);
        reinterpret_cast<double2 *>(r)[q] = rv;
        acc = fma(s_c[cd.x & 0x7f] * rv.x, rv.x, acc);
        acc = fma(s_c[cd.y & 0x7f] * rv.y, rv.y, acc);
    }
    if ((L & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        const int64_t l = L - 1;
        const double rv = fma(-alpha, w[l], r[l]);
        r[l] = rv;
        acc = fma(s_c[code[l] & 0x7f] * rv, rv, acc);
    }
    nk_grid_reduce(acc, s_red, ws, NK_EPI_RHO, hist_k);
}

// ---- the x update deferred by one iteration ("defer_x"; large meshes, where the direction update is a kernel of its
// own).  x_k+1 = x_k + alpha_k p_k is not needed before the solve ends, so two iterations share one pass over x:
//   first of a pair   p2 = r + beta p                        (24 B/pt; alpha kept in NK_S_ALPHA_PREV)
//   second            x = fma(alpha', p2, fma(alpha, p, x)); p = r + beta' p2                  (48 B/pt)
// 72 B/pt per pair instead of 2 x 40, and x, entry by entry, is bit for bit what two separate updates give (the same
// two fused multiply-adds in the same order).  Costs one more vector in the workspace.
__global__ void __launch_bounds__(NK_VEC_THREADS)
update_p2_kernel(double *__restrict__ p2, const double *p, const double *r, double *scal, int64_t L)
{
    nk_pdl_launch_dependents();
    nk_pdl_wait();
    const double beta = scal[NK_S_BETA];
    if (blockIdx.x == 0 && threadIdx.x == 0) scal[NK_S_ALPHA_PREV] = scal[NK_S_ALPHA];   // the next ax_e overwrites alpha
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t quads = L >> 2;                            // p, p2, r live in the workspace: 256-byte aligned
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < quads; q += stride) {
        const double4v rv = ld256(r + 4 * q), pv = ld256(p + 4 * q);
        double4v o;
        o.a = fma(beta, pv.a, rv.a); o.b = fma(beta, pv.b, rv.b);
        o.c = fma(beta, pv.c, rv.c); o.d = fma(beta, pv.d, rv.d);
        st256(p2 + 4 * q, o);
    }
    if (blockIdx.x == 0 && (int64_t)threadIdx.x < (L & 3)) {
        const int64_t l = (quads << 2) + threadIdx.x;
        p2[l] = fma(beta, p[l], r[l]);
    }
}

__global__ void __launch_bounds__(NK_VEC_THREADS)
update_pxx_kernel(double *__restrict__ x, double *p, const double *p2, const double *r, const double *scal, int64_t L)
{
    nk_pdl_launch_dependents();
    nk_pdl_wait();
    const double alpha0 = scal[NK_S_ALPHA_PREV], alpha1 = scal[NK_S_ALPHA], beta = scal[NK_S_BETA];
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t quads = L >> 2;
    const bool x32 = (reinterpret_cast<uintptr_t>(x) & 31u) == 0;      // the caller's x may only be 16-byte aligned
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < quads; q += stride) {
        const double4v rv = ld256(r + 4 * q), pa = ld256(p + 4 * q), pb = ld256(p2 + 4 * q);
        double4v xv = ld4(x + 4 * q, x32), o;
        xv.a = fma(alpha1, pb.a, fma(alpha0, pa.a, xv.a)); xv.b = fma(alpha1, pb.b, fma(alpha0, pa.b, xv.b));
        xv.c = fma(alpha1, pb.c, fma(alpha0, pa.c, xv.c)); xv.d = fma(alpha1, pb.d, fma(alpha0, pa.d, xv.d));
        o.a = fma(beta, pb.a, rv.a); o.b = fma(beta, pb.b, rv.b);
        o.c = fma(beta, pb.c, rv.c); o.d = fma(beta, pb.d, rv.d);
        st4(x + 4 * q, xv, x32);
        st256(p + 4 * q, o);
    }
    if (blockIdx.x == 0 && (int64_t)threadIdx.x < (L & 3)) {
        const int64_t l = (quads << 2) + threadIdx.x;
        x[l] = fma(alpha1, p2[l], fma(alpha0, p[l], x[l]));
        p[l] = fma(beta, p2[l], r[l]);
    }
}

// x += alpha p (the OLD p); p = r + beta p
__global__ void __launch_bounds__(NK_VEC_THREADS)
update_px_kernel(double *__restrict__ x, double *__restrict__ p, const double *r,
                 const double *scal, int64_t L)
{
    nk_pdl_launch_dependents();
    nk_pdl_wait();
    const double alpha = scal[NK_S_ALPHA], beta = scal[NK_S_BETA];
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    int64_t done = 0;                                       // points handled four at a time
    if (NK_V256 && aligned32(x, p, r)) {
        const int64_t quads = L >> 2;
        for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < quads; q += stride) {
            const double4v rv = ld256(r + 4 * q);
            double4v pv = ld256(p + 4 * q), xv = ld256(x + 4 * q);
            xv.a = fma(alpha, pv.a, xv.a); xv.b = fma(alpha, pv.b, xv.b);
            xv.c = fma(alpha, pv.c, xv.c); xv.d = fma(alpha, pv.d, xv.d);
            pv.a = fma(beta, pv.a, rv.a); pv.b = fma(beta, pv.b, rv.b);
            pv.c = fma(beta, pv.c, rv.c); pv.d = fma(beta, pv.d, rv.d);
            st256(x + 4 * q, xv);
            st256(p + 4 * q, pv);
        }
        done = quads << 2;
    }
    const int64_t pairs = L >> 1;
    for (int64_t q = (done >> 1) + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < pairs; q += stride) {
        const double2 rv = reinterpret_cast<const double2 *>(r)[q];
        double2 pv = reinterpret_cast<double2 *>(p)[q];
        double2 xv = reinterpret_cast<double2 *>(x)[q];
        xv.x = fma(alpha, pv.x, xv.x);
        xv.y = fma(alpha, pv.y, xv.y);
        pv.x = fma(beta, pv.x, rv.x);
        pv.y = fma(beta, pv.y, rv.y);
        reinterpret_cast<double2 *>(x)[q] = xv;
        reinterpret_cast<double2 *>(p)[q] = pv;
    }
    if ((L & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        const int64_t l = L - 1;
        x[l] = fma(alpha, p[l], x[l]);
        p[l] = fma(beta, p[l], r[l]);
    }
}

__global__ void __launch_bounds__(NK_VEC_THREADS)
get_mult_kernel(double *__restrict__ mult, const uint8_t *__restrict__ code, const double *__restrict__ mtab, int64_t L)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t l = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; l < L; l += stride)
        mult[l] = mtab[code[l] & 0x7f];
}

// ---- Jacobi-preconditioned CG: z = dinv o r is never stored ---------------------
// r = mask o f, x = 0, p = z = dinv o r, rho = <r,z>_c, hist[0] = sqrt<r,r>_c
__global__ void __launch_bounds__(NK_VEC_THREADS)
pcg_init_kernel(const double *__restrict__ f, double *__restrict__ x, double *__restrict__ r,
                double *__restrict__ p, const double *__restrict__ dinv, const uint8_t *__restrict__ code,
                const double *__restrict__ ctab, int64_t L, nk_reduce_ws ws, double *hist0)
{
    __shared__ double s_c[NK_CTAB];
    __shared__ double s_red[33];
    load_ctab(s_c, ctab);
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    double a1 = 0.0, a2 = 0.0;
    for (int64_t l = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; l < L; l += stride) {
        const uint8_t cd = code[l];
        const double rv = (cd & NK_CODE_MASKED) ? 0.0 : f[l];
        const double zv = dinv[l] * rv;
        r[l] = rv; p[l] = zv; x[l] = 0.0;
        const double cw = s_c[cd & 0x7f] * rv;
        a1 = fma(cw, zv, a1);
        a2 = fma(cw, rv, a2);
    }
    nk_grid_reduce2(a1, a2, s_red, ws, 1, hist0);
}

// r -= alpha w; z = dinv o r; rho' = <r,z>_c; hist = sqrt<r,r>_c   (x rides with the p update below)
__global__ void __launch_bounds__(NK_VEC_THREADS)
update_rz_kernel(double *__restrict__ r, const double *w, const double *__restrict__ dinv,
                  const uint8_t *__restrict__ code, const double *__restrict__ ctab, int64_t L,
                  nk_reduce_ws ws, double *hist_k)
{
    __shared__ double s_c[NK_CTAB];
    __shared__ double s_red[33];
    nk_pdl_launch_dependents();
    load_ctab(s_c, ctab);
    nk_pdl_wait();
    const double alpha = ws.scal[NK_S_ALPHA];
    const int64_t pairs = L >> 1;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    double a1 = 0.0, a2 = 0.0;
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < pairs; q += stride) {
        const double2 wv = reinterpret_cast<const double2 *>(w)[q];
        const double2 dv = reinterpret_cast<const double2 *>(dinv)[q];
        double2 rv = reinterpret_cast<double2 *>(r)[q];
        const uchar2 cd = reinterpret_cast<const uchar2 *>(code)[q];
        rv.x = fma(-alpha, wv.x, rv.x);
        rv.y = fma(-alpha, wv.y, rv.y);
        reinterpret_cast<double2 *>(r)[q] = rv;
        const double c0 = s_c[cd.x & 0x7f] * rv.x, c1 = s_c[cd.y & 0x7f] * rv.y;
        a1 = fma(c0, dv.x * rv.x, a1);
        a1 = fma(c1, dv.y * rv.y, a1);
        a2 = fma(c0, rv.x, a2);
        a2 = fma(c1, rv.y, a2);
    }
    if ((L & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        const int64_t l = L - 1;
        const double rv = fma(-alpha, w[l], r[l]);
        r[l] = rv;
        const double c0 = s_c[code[l] & 0x7f] * rv;
        a1 = fma(c0, dinv[l] * rv, a1);
        a2 = fma(c0, rv, a2);
    }
    nk_grid_reduce2(a1, a2, s_red, ws, 0, hist_k);
}

// x += alpha p (the OLD p); p = dinv o r + beta p
__global__ void __launch_bounds__(NK_VEC_THREADS)
update_pxz_kernel(double *__restrict__ x, double *__restrict__ p, const double *r,
                  const double *__restrict__ dinv, const double *scal, int64_t L)
{
    nk_pdl_launch_dependents();
    nk_pdl_wait();
    const double alpha = scal[NK_S_ALPHA], beta = scal[NK_S_BETA];
    const int64_t pairs = L >> 1;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < pairs; q += stride) {
        const double2 rv = reinterpret_cast<const double2 *>(r)[q];
        const double2 dv = reinterpret_cast<const double2 *>(dinv)[q];
        double2 pv = reinterpret_cast<double2 *>(p)[q];
        double2 xv = reinterpret_cast<double2 *>(x)[q];
        xv.x = fma(alpha, pv.x, xv.x);
        xv.y = fma(alpha, pv.y, xv.y);
        pv.x = fma(beta, pv.x, dv.x * rv.x);
        pv.y = fma(beta, pv.y, dv.y * rv.y);
        reinterpret_cast<double2 *>(x)[q] = xv;
        reinterpret_cast<double2 *>(p)[q] = pv;
    }
    if ((L & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        const int64_t l = L - 1;
        x[l] = fma(alpha, p[l], x[l]);
        p[l] = fma(beta, p[l], dinv[l] * r[l]);
    }
}

}  // namespace

cudaError_t nk_launch_dot(nk_ctx *c, const double *a, const double *b, double *out, int epi, cudaStream_t st)
{
    const int nb = vec_blocks(c, c->L >> 1);
    dot_kernel<<<nb, NK_VEC_THREADS, 0, st>>>(a, b, c->code, c->ctab, c->L, c->red, epi, out);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t nk_launch_cg_init(nk_ctx *c, const double *f, double *x, double *hist, cudaStream_t st)
{
    const int nb = vec_blocks(c, c->L >> 1);
    cg_init_kernel<<<nb, NK_VEC_THREADS, 0, st>>>(f, x, c->r, c->p, c->code, c->ctab, c->L, c->red, hist);
    c->launches++;
    return cudaGetLastError();
}

namespace {
// gs != 0: the fused kernel (gs_update_kernel).  It is a programmatic dependent only where gs itself would be
// (nk_pdl_mode: its gathers want the L1 that ax_e's shared-memory carve-out takes away on large meshes).
template <int XM>
cudaError_t launch_gs_update(nk_ctx *c, double *x, const double *pa, const double *pb, double *hist_k, int stash, cudaStream_t st)
{
    nk_gather gp;
    gp.nbr = c->nbr; gp.gx = c->gx; gp.rows = c->gx_rows; gp.blk = c->gx_blk;
    const int nb = nk_gsu_blocks(c->sm_count, c->L >> 1);         // the grid nk_setup cut the row list for (gx_blk)
    const cudaError_t e = nk_launch(gs_update_kernel<XM>, nb, NK_GSU_THREADS, 0, st, c->pdl_now == 2, x, c->r, pa, pb,
                                    (const double *)c->w, c->L, c->red, hist_k, gp, stash);
    if (e != cudaSuccess) return e;
    c->launches++;
    return cudaGetLastError();
}
}  // namespace

cudaError_t nk_launch_update_xr(nk_ctx *c, double *x, double *hist_k, int gs, cudaStream_t st)
{
    if (gs) return launch_gs_update<1>(c, x, c->pc, nullptr, hist_k, 0, st);
    const int nb = vec_blocks(c, c->L >> 1);
    const cudaError_t e = nk_launch(update_xr_kernel, nb, NK_VEC_THREADS, 0, st, c->pdl_now, x, c->r, c->pc, c->w, c->code,
                                    c->ctab, c->L, c->red, hist_k);
    if (e != cudaSuccess) return e;
    c->launches++;
    return cudaGetLastError();
}

cudaError_t nk_launch_update_p(nk_ctx *c, cudaStream_t st)
{
    const int nb = vec_blocks(c, c->L >> 1);
    const cudaError_t e = nk_launch(update_p_kernel, nb, NK_VEC_THREADS, 0, st, c->pdl_now, c->p, (const double *)c->pc, (const double *)c->r,
                                    (const double *)c->red.scal, c->L);   // c->pc != c->p: the pending update lands in c->p
    if (e != cudaSuccess) return e;
    c->launches++;
    return cudaGetLastError();
}

cudaError_t nk_launch_get_mult(nk_ctx *c, double *mult, cudaStream_t st)
{
    const int nb = vec_blocks(c, c->L);
    get_mult_kernel<<<nb, NK_VEC_THREADS, 0, st>>>(mult, c->code, c->mtab, c->L);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t nk_launch_pcg_init(nk_ctx *c, const double *f, double *x, double *hist, cudaStream_t st)
{
    const int nb = vec_blocks(c, c->L >> 1);
    pcg_init_kernel<<<nb, NK_VEC_THREADS, 0, st>>>(f, x, c->r, c->p, c->dinv, c->code, c->ctab, c->L, c->red, hist);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t nk_launch_update_xrz(nk_ctx *c, double *x, double *hist_k, cudaStream_t st)
{
    const int nb = vec_blocks(c, c->L >> 1);
    (void)x;
    const cudaError_t e = nk_launch(update_rz_kernel, nb, NK_VEC_THREADS, 0, st, c->pdl_now, c->r, c->w, c->dinv, c->code,
                                    c->ctab, c->L, c->red, hist_k);
    if (e != cudaSuccess) return e;
    c->launches++;
    return cudaGetLastError();
}

cudaError_t nk_launch_update_pz(nk_ctx *c, double *x, cudaStream_t st)
{
    const int nb = vec_blocks(c, c->L >> 1);
    const cudaError_t e = nk_launch(update_pxz_kernel, nb, NK_VEC_THREADS, 0, st, c->pdl_now, x, c->p, c->r, c->dinv,
                                    c->red.scal, c->L);
    if (e != cudaSuccess) return e;
    c->launches++;
    return cudaGetLastError();
}

cudaError_t nk_launch_update_r(nk_ctx *c, double *hist_k, int gs, cudaStream_t st)
{
    if (gs) return launch_gs_update<0>(c, nullptr, nullptr, nullptr, hist_k, 0, st);
    const int nb = vec_blocks(c, c->L >> 1);
    const cudaError_t e = nk_launch(update_r_kernel, nb, NK_VEC_THREADS, 0, st, c->pdl_now, c->r, c->w, c->code, c->ctab,
                                    c->L, c->red, hist_k);
    if (e != cudaSuccess) return e;
    c->launches++;
    return cudaGetLastError();
}

cudaError_t nk_launch_update_p2(nk_ctx *c, cudaStream_t st)
{
    const int nb = vec_blocks(c, c->L >> 1);
    const cudaError_t e = nk_launch(update_p2_kernel, nb, NK_VEC_THREADS, 0, st, c->pdl_now, c->p2, (const double *)c->p,
                                    (const double *)c->r, c->red.scal, c->L);
    if (e != cudaSuccess) return e;
    c->launches++;
    return cudaGetLastError();
}

cudaError_t nk_launch_update_pxx(nk_ctx *c, double *x, cudaStream_t st)
{
    const int nb = vec_blocks(c, c->L >> 1);
    const cudaError_t e = nk_launch(update_pxx_kernel, nb, NK_VEC_THREADS, 0, st, c->pdl_now, x, c->p, (const double *)c->p2,
                                    (const double *)c->r, (const double *)c->red.scal, c->L);
    if (e != cudaSuccess) return e;
    c->launches++;
    return cudaGetLastError();
}

cudaError_t nk_launch_update_px(nk_ctx *c, double *x, cudaStream_t st)
{
    const int nb = vec_blocks(c, c->L >> 1);
    const cudaError_t e = nk_launch(update_px_kernel, nb, NK_VEC_THREADS, 0, st, c->pdl_now, x, c->p, c->r, c->red.scal, c->L);
    if (e != cudaSuccess) return e;
    c->launches++;
    return cudaGetLastError();
}

// "defer_x" on the "fuse_p" path: the fused gs update of the first iteration of a pair (no x, alpha kept) and of the
// second (x takes both steps: pa, pb = the directions of the first and second iteration)
cudaError_t nk_launch_update_r_first(nk_ctx *c, double *hist_k, cudaStream_t st)
{
    return launch_gs_update<0>(c, nullptr, nullptr, nullptr, hist_k, 1, st);
}
cudaError_t nk_launch_update_xxr(nk_ctx *c, double *x, const double *pa, const double *pb, double *hist_k, cudaStream_t st)
{
    return launch_gs_update<2>(c, x, pa, pb, hist_k, 0, st);
}
