// nk_plan.cu -- the gather-scatter plan of nk_setup built ON THE DEVICE (S 8(a) row a0; north_star: the host is
// there for memory and streams).  Same arrays, bit for bit, as the host builder in nk_setup.cu
// (tests/test_gpu_operators.py::test_device_plan_equals_host_plan):
//   ids, mask uploaded -> validate -> stable LSD radix sort of (global id, local index), 8 bits per pass, only the
//   passes the largest id needs -> heads of the groups of equal ids (scan over the sorted list) -> per group:
//   length, Dirichlet flag, first local index -> rows in ascending first local index (a scan over LOCAL indices of
//   "this point is the first copy of a summed / masked node": no second sort) -> CSR (row_off, row_idx), per-point
//   multiplicity code, gather codes of the fused update (nbr, gx, gx_rows, gx_blk), packed rows of nk_gs.cu (pk, desc).
// Hand-written kernels only (no CUB / Thrust).  Two host synchronisations: after validation (number of sort passes)
// and after the scans (the distinct multiplicities, at most NK_CTAB, become the ctab / mtab tables on the host).
// Scratch: the workspace regions nothing uses before the geometry kernel (G, hf, hx, dinv, the partial-sum block).
#include <algorithm>
#include <cstring>
#include <vector>

#include "nk_host.h"

namespace {

constexpr int PT = 256;                  // threads per block of the plan kernels
constexpr int MULT_DIRECT = 4096;        // multiplicities up to here are recorded in a byte map, larger ones in a list
constexpr int MULT_OVF_CAP = 8192;       // entries of that list (duplicates included); beyond: the host builder takes over

// ---- packed counters: NC 64-bit words, each two 32-bit counters (no carry between them: every count < 2^31) -------
template <int NC>
struct Vec { unsigned long long v[NC]; };

template <int NC>
__device__ __forceinline__ Vec<NC> vzero()
{
    Vec<NC> z;
#pragma unroll
    for (int c = 0; c < NC; ++c) z.v[c] = 0ull;
    return z;
}
template <int NC>
__device__ __forceinline__ Vec<NC> vadd(const Vec<NC> &a, const Vec<NC> &b)
{
    Vec<NC> s;
#pragma unroll
    for (int c = 0; c < NC; ++c) s.v[c] = a.v[c] + b.v[c];
    return s;
}
__device__ __forceinline__ unsigned lo32(unsigned long long x) { return (unsigned)(x & 0xffffffffull); }
__device__ __forceinline__ unsigned hi32(unsigned long long x) { return (unsigned)(x >> 32); }

// exclusive scan over the PT threads of a block; `sm` holds PT / 32 entries; `total` is valid in every thread
template <int NC>
__device__ __forceinline__ void block_excl_scan(const Vec<NC> &x, Vec<NC> &excl, Vec<NC> &total, Vec<NC> *sm)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    Vec<NC> inc = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const unsigned long long t = __shfl_up_sync(0xffffffffu, inc.v[c], o);
            if (lane >= o) inc.v[c] += t;
        }
    }
    __syncthreads();                                   // sm may still be read from a previous call
    if (lane == 31) sm[wid] = inc;
    __syncthreads();
    Vec<NC> base = vzero<NC>();
    total = vzero<NC>();
#pragma unroll
    for (int w = 0; w < PT / 32; ++w) {
        if (w < wid) base = vadd(base, sm[w]);
        total = vadd(total, sm[w]);
    }
#pragma unroll
    for (int c = 0; c < NC; ++c) excl.v[c] = base.v[c] + inc.v[c] - x.v[c];
}

// ---- a scan over n items in three launches: per-block sums, their exclusive scan, per-block scan + emit -----------
// F: static NC; Vec<NC> value(int64 i); void emit(int64 i, const Vec<NC> &excl, const Vec<NC> &val, const Vec<NC> &total)
template <class F>
__global__ void __launch_bounds__(PT) scan_reduce_kernel(F f, int64_t n, Vec<F::NC> *bsum)
{
    __shared__ Vec<F::NC> sm[PT / 32];
    const int64_t lo = n * (int64_t)blockIdx.x / gridDim.x, hi = n * ((int64_t)blockIdx.x + 1) / gridDim.x;
    Vec<F::NC> acc = vzero<F::NC>();
    for (int64_t i = lo + threadIdx.x; i < hi; i += PT) acc = vadd(acc, f.value(i));
    Vec<F::NC> excl, total;
    block_excl_scan(acc, excl, total, sm);
    if (threadIdx.x == 0) bsum[blockIdx.x] = total;
}

template <int NC>
__global__ void scan_blocks_kernel(Vec<NC> *bsum, int nb, Vec<NC> *total)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    Vec<NC> run = vzero<NC>();
    for (int b = 0; b < nb; ++b) {
        const Vec<NC> t = bsum[b];
        bsum[b] = run;
        run = vadd(run, t);
    }
    *total = run;
}

template <class F>
__global__ void __launch_bounds__(PT) scan_emit_kernel(F f, int64_t n, const Vec<F::NC> *bsum, const Vec<F::NC> *total)
{
    __shared__ Vec<F::NC> sm[PT / 32];
    const int64_t lo = n * (int64_t)blockIdx.x / gridDim.x, hi = n * ((int64_t)blockIdx.x + 1) / gridDim.x;
    Vec<F::NC> carry = bsum[blockIdx.x];
    const Vec<F::NC> tot = *total;
    for (int64_t base = lo; base < hi; base += PT) {
        const int64_t i = base + threadIdx.x;
        const Vec<F::NC> val = i < hi ? f.value(i) : vzero<F::NC>();
        Vec<F::NC> excl, sum;
        block_excl_scan(val, excl, sum, sm);
        if (i < hi) f.emit(i, vadd(carry, excl), val, tot);
        carry = vadd(carry, sum);
    }
}

inline int scan_grid(int sm_count, int64_t n)
{
    const int64_t want = (n + PT - 1) / PT, cap = (int64_t)sm_count * 8;
    return (int)std::max<int64_t>(1, std::min(want, cap));
}

// ---- what the kernels report back (one small block, read twice by the host) --------------------------------------
struct PlanInfo {
    unsigned long long max_id;
    int bad_id, bad_mask, mask_clash, ovf_n;
    unsigned long long n_shared, n_masked;
    Vec<1> heads;                         // lo: groups = unique nodes
    Vec<3> rows;                          // [0] lo summed rows, hi masked rows; [1] lo / hi their listed copies;
                                          // [2] lo rows with >= 3 copies, hi their quads in gx
    long long pk_size;
    unsigned char present[MULT_DIRECT + 1];
    int ovf[MULT_OVF_CAP];
};

__global__ void __launch_bounds__(PT) validate_kernel(const long long *glo, const double *mask, int64_t L, PlanInfo *info)
{
    unsigned long long mx = 0;
    int bi = 0, bm = 0;
    for (int64_t l = (int64_t)blockIdx.x * PT + threadIdx.x; l < L; l += (int64_t)gridDim.x * PT) {
        const long long g = glo[l];
        if (g < 0) bi = 1;
        else if ((unsigned long long)g > mx) mx = (unsigned long long)g;
        const double m = mask[l];
        if (!(m == 0.0 || m == 1.0)) bm = 1;
    }
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long t = __shfl_xor_sync(0xffffffffu, mx, o);
        mx = t > mx ? t : mx;
    }
    bi = __any_sync(0xffffffffu, bi);
    bm = __any_sync(0xffffffffu, bm);
    if ((threadIdx.x & 31) == 0) {
        atomicMax(&info->max_id, mx);
        if (bi) atomicOr(&info->bad_id, 1);
        if (bm) atomicOr(&info->bad_mask, 1);
    }
}

// ---- stable LSD radix sort, 8 bits per pass ----------------------------------------------------------------------
// A block owns a contiguous run of tiles of RS_TILE keys; inside a tile warp w owns keys [512 w, 512 w + 512) and
// takes them 32 at a time, so (block, tile, warp, round, lane) is the input order and ranks handed out in that order
// keep the sort stable.  count: per-block digit histogram -> table[digit][block]; scan: exclusive over the table in
// that order; scatter: per round the lanes with equal digits find each other (match.any), rank = the warp's running
// count of the digit + the number of lower lanes with it.
constexpr int RS_ROUNDS = 16, RS_TILE = PT * RS_ROUNDS, RS_MAX_BLOCKS = 448;

__device__ __forceinline__ void rs_block_range(int64_t n, int64_t &lo, int64_t &hi)
{
    const int64_t tiles = (n + RS_TILE - 1) / RS_TILE;
    lo = tiles * (int64_t)blockIdx.x / gridDim.x * RS_TILE;
    hi = tiles * ((int64_t)blockIdx.x + 1) / gridDim.x * RS_TILE;
    if (hi > n) hi = n;
    if (lo > n) lo = n;
}

__global__ void __launch_bounds__(PT) radix_count_kernel(const unsigned long long *key, int64_t n, int shift, unsigned *table)
{
    __shared__ unsigned hist[256];
    hist[threadIdx.x] = 0;
    __syncthreads();
    int64_t lo, hi;
    rs_block_range(n, lo, hi);
    for (int64_t i = lo + threadIdx.x; i < hi; i += PT) atomicAdd(&hist[(unsigned)(key[i] >> shift) & 255u], 1u);
    __syncthreads();
    table[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = hist[threadIdx.x];
}

__global__ void __launch_bounds__(1024) radix_scan_kernel(unsigned *table, int m)
{
    __shared__ unsigned long long sm[32];
    const int per = (m + 1023) / 1024;
    const int lo = min(m, (int)threadIdx.x * per), hi = min(m, lo + per);
    unsigned long long s = 0;
    for (int i = lo; i < hi; ++i) s += table[i];
    // exclusive scan of s over 1024 threads
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    unsigned long long inc = s;
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) sm[wid] = inc;
    __syncthreads();
    unsigned long long base = 0;
    for (int w = 0; w < wid; ++w) base += sm[w];
    unsigned long long run = base + inc - s;
    for (int i = lo; i < hi; ++i) {
        const unsigned c = table[i];
        table[i] = (unsigned)run;                       // positions < 2^31
        run += c;
    }
}

template <bool FIRST>
__global__ void __launch_bounds__(PT) radix_scatter_kernel(const unsigned long long *key, const unsigned *val,
                                                           unsigned long long *key_out, unsigned *val_out, int64_t n,
                                                           int shift, const unsigned *table)
{
    __shared__ unsigned base[256];
    __shared__ unsigned wh[PT / 32][256];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    base[threadIdx.x] = table[(size_t)threadIdx.x * gridDim.x + blockIdx.x];
    int64_t lo, hi;
    rs_block_range(n, lo, hi);
    for (int64_t t0 = lo; t0 < hi; t0 += RS_TILE) {
#pragma unroll
        for (int w = 0; w < PT / 32; ++w) wh[w][threadIdx.x] = 0;
        __syncthreads();
        unsigned long long k[RS_ROUNDS];
        unsigned v[RS_ROUNDS];
        unsigned short rk[RS_ROUNDS];
#pragma unroll
        for (int r = 0; r < RS_ROUNDS; ++r) {
            const int64_t i = t0 + wid * (32 * RS_ROUNDS) + r * 32 + lane;
            const bool on = i < hi;
            k[r] = on ? key[i] : 0ull;
            v[r] = on ? (FIRST ? (unsigned)i : val[i]) : 0u;
            const unsigned d = on ? ((unsigned)(k[r] >> shift) & 255u) : (256u + (unsigned)lane);
            const unsigned peers = __match_any_sync(0xffffffffu, d);
            const unsigned before = __popc(peers & ((1u << lane) - 1u));
            unsigned prev = 0;
            if (on) prev = wh[wid][d];
            __syncwarp();
            if (on && before == 0) wh[wid][d] = prev + __popc(peers);
            __syncwarp();
            rk[r] = (unsigned short)(prev + before);
        }
        __syncthreads();
        {
            unsigned run = base[threadIdx.x];
#pragma unroll
            for (int w = 0; w < PT / 32; ++w) {
                const unsigned c = wh[w][threadIdx.x];
                wh[w][threadIdx.x] = run;
                run += c;
            }
            base[threadIdx.x] = run;
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < RS_ROUNDS; ++r) {
            const int64_t i = t0 + wid * (32 * RS_ROUNDS) + r * 32 + lane;
            if (i < hi) {
                const unsigned dst = wh[wid][(unsigned)(k[r] >> shift) & 255u] + rk[r];
                key_out[dst] = k[r];
                val_out[dst] = v[r];
            }
        }
        __syncthreads();
    }
}

// ---- groups of equal ids in the sorted list ----------------------------------------------------------------------
struct HeadScan {                         // over sorted positions i: gid[i] = index of i's group, pos[g] = where it starts
    static constexpr int NC = 1;
    const unsigned long long *key;
    unsigned *gid, *pos;
    __device__ Vec<1> value(int64_t i) const
    {
        Vec<1> v;
        v.v[0] = (i == 0 || key[i] != key[i - 1]) ? 1ull : 0ull;
        return v;
    }
    __device__ void emit(int64_t i, const Vec<1> &excl, const Vec<1> &val, const Vec<1> &) const
    {
        const unsigned g = (unsigned)(excl.v[0] + val.v[0]) - 1u;
        gid[i] = g;
        if (val.v[0]) pos[g] = (unsigned)i;
    }
};

// one thread per group: length | Dirichlet flag, "first copy" marker at its first local index, the statistics
__global__ void __launch_bounds__(PT) group_kernel(const unsigned *pos, const unsigned *loc, const double *mask, int64_t L,
                                                   unsigned *glen, unsigned *gl, PlanInfo *info)
{
    const int64_t G = (int64_t)lo32(info->heads.v[0]);
    unsigned shared = 0, masked = 0;
    for (int64_t g = (int64_t)blockIdx.x * PT + threadIdx.x; g < G; g += (int64_t)gridDim.x * PT) {
        const unsigned b = pos[g], e = g + 1 < G ? pos[g + 1] : (unsigned)L;
        const unsigned len = e - b, first = loc[b];
        const unsigned m0 = mask[first] == 0.0 ? 1u : 0u;
        glen[g] = len | (m0 << 31);
        gl[first] = (unsigned)g + 1u;
        shared += len > 1u;
        masked += m0;
        if (len <= (unsigned)MULT_DIRECT) {
            info->present[len] = 1;
        } else {
            const int k = atomicAdd(&info->ovf_n, 1);
            if (k < MULT_OVF_CAP) info->ovf[k] = (int)len;
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        shared += __shfl_xor_sync(0xffffffffu, shared, o);
        masked += __shfl_xor_sync(0xffffffffu, masked, o);
    }
    if ((threadIdx.x & 31) == 0) {
        if (shared) atomicAdd(&info->n_shared, (unsigned long long)shared);
        if (masked) atomicAdd(&info->n_masked, (unsigned long long)masked);
    }
}

// ---- rows in ascending FIRST local index: a scan over local indices ------------------------------------------------
struct PlanOut {                          // final arrays (workspace) and what the row scan leaves for the later kernels
    int32_t *off, *idx, *nbr, *gx, *pk;
    uint8_t *code;
    unsigned *doff, *gp4, *rbeg, *rlen;   // per group: position of its copies in idx, its p4 in gx; per summed row: start in
};                                        // the sorted list, length

struct RowScan {
    static constexpr int NC = 3;
    const unsigned *gl, *glen, *pos;
    PlanOut o;
    __device__ Vec<3> value(int64_t l) const
    {
        Vec<3> v = vzero<3>();
        const unsigned g1 = gl[l];
        if (g1 == 0u) return v;
        const unsigned lm = glen[g1 - 1u], len = lm & 0x7fffffffu;
        if (lm >> 31) {
            v.v[0] = 1ull << 32;
            v.v[1] = (unsigned long long)len << 32;
        } else if (len > 1u) {
            v.v[0] = 1ull;
            v.v[1] = len;
            if (len >= 3u) v.v[2] = 1ull | ((unsigned long long)(len / 4u + 1u) << 32);
        }
        return v;
    }
    __device__ void emit(int64_t l, const Vec<3> &ex, const Vec<3> &val, const Vec<3> &tot) const
    {
        if (l == 0) o.off[lo32(tot.v[0]) + hi32(tot.v[0])] = (int32_t)(lo32(tot.v[1]) + hi32(tot.v[1]));
        if ((val.v[0] | val.v[1]) == 0ull) return;
        const unsigned g = gl[l] - 1u;
        const unsigned len = glen[g] & 0x7fffffffu;
        if (val.v[0] >> 32) {                                  // a masked node
            const unsigned row = lo32(tot.v[0]) + hi32(ex.v[0]), at = lo32(tot.v[1]) + hi32(ex.v[1]);
            o.off[row] = (int32_t)at;
            o.doff[g] = at;
            return;
        }
        const unsigned row = lo32(ex.v[0]), at = lo32(ex.v[1]);
        o.off[row] = (int32_t)at;
        o.doff[g] = at;
        o.rbeg[row] = pos[g];
        o.rlen[row] = len;
        if (len >= 3u) {
            const unsigned p4 = 1u + hi32(ex.v[2]);
            int32_t *gx_rows = o.gx + 4 * ((size_t)hi32(tot.v[2]) + 4);      // gx holds 4 (Q + 3) ints, Q = 1 + quads
            gx_rows[lo32(ex.v[2])] = (int32_t)p4;
            o.gx[4 * (size_t)p4 - 1] = (int32_t)len;
            o.gp4[g] = p4;
        }
    }
};

// one thread per sorted position: multiplicity code, CSR entry, gather code, gx entry, mask consistency
__global__ void __launch_bounds__(PT) fill_kernel(const unsigned *gid, const unsigned *pos, const unsigned *glen,
                                                  const unsigned *loc, const double *mask, int64_t L, PlanOut o,
                                                  const int *mult, int n_mult, PlanInfo *info)
{
    __shared__ int s_mult[NK_CTAB];
    if (threadIdx.x < NK_CTAB) s_mult[threadIdx.x] = threadIdx.x < n_mult ? mult[threadIdx.x] : 0x7fffffff;
    __syncthreads();
    int clash = 0;
    for (int64_t i = (int64_t)blockIdx.x * PT + threadIdx.x; i < L; i += (int64_t)gridDim.x * PT) {
        const unsigned g = gid[i], b = pos[g], lm = glen[g], l = loc[i];
        const unsigned len = lm & 0x7fffffffu, m0 = lm >> 31, q = (unsigned)i - b;
        if ((mask[l] == 0.0 ? 1u : 0u) != m0) clash = 1;
        int t0 = 0, t1 = n_mult - 1;                           // lower bound of len in the ascending table
        while (t0 < t1) {
            const int mid = (t0 + t1) >> 1;
            if (s_mult[mid] < (int)len) t0 = mid + 1; else t1 = mid;
        }
        o.code[l] = (uint8_t)((unsigned)t0 | (m0 ? NK_CODE_MASKED : 0u));
        if (m0 || len > 1u) o.idx[o.doff[g] + q] = (int32_t)l;
        int32_t nb;
        if (m0) nb = -1;
        else if (len == 1u) nb = (int32_t)l;
        else if (len == 2u) nb = (int32_t)loc[b + 1u - q];
        else {
            const unsigned p4 = o.gp4[g];
            nb = -(int32_t)p4 - 2;
            o.gx[4 * (size_t)p4 + q] = (int32_t)l;
        }
        o.nbr[l] = nb;
    }
    if (__any_sync(0xffffffffu, clash) && (threadIdx.x & 31) == 0) atomicOr(&info->mask_clash, 1);
}

// gx_blk[b] = number of rows with >= 3 copies whose first copy lies before block b's chunk of the fused update
__global__ void gx_blk_kernel(const int32_t *gx, const int32_t *gx_rows, int n_gx_rows, int64_t L, int nvb, int32_t *gx_blk)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b > nvb) return;
    const int64_t pairs = L >> 1;
    const int64_t first_point = b == nvb ? L + 1 : 4 * ((L >> 2) * (int64_t)b / nvb);
    int lo = 0, hi = n_gx_rows;                               // smallest k with first(k) >= first_point
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if ((int64_t)gx[4 * (size_t)gx_rows[mid]] < first_point) lo = mid + 1; else hi = mid;
    }
    gx_blk[b] = b == 0 ? 0 : lo;
}

// ---- the packed rows of nk_gs.cu: chunks of NK_GS_CHUNK rows, inside a chunk by length (2, 4, 8, other) ------------
__device__ __forceinline__ int len_class(unsigned len) { return len == 2u ? 0 : len == 4u ? 1 : len == 8u ? 2 : 3; }
__device__ __forceinline__ long long pad4ll(long long v) { return (v + 3) / 4 * 4; }

__global__ void __launch_bounds__(PT) pack_count_kernel(const unsigned *rlen, const PlanInfo *info, int32_t *desc)
{
    __shared__ int cnt[4];
    const int64_t n_sum_rows = lo32(info->rows.v[0]);
    const int64_t r0 = (int64_t)blockIdx.x * NK_GS_CHUNK, r1 = min(r0 + (int64_t)NK_GS_CHUNK, n_sum_rows);
    if (threadIdx.x < 4) cnt[threadIdx.x] = 0;
    __syncthreads();
    int c[4] = {0, 0, 0, 0};
    for (int64_t r = r0 + threadIdx.x; r < r1; r += PT) ++c[len_class(rlen[r])];
    for (int k = 0; k < 4; ++k)
        if (c[k]) atomicAdd(&cnt[k], c[k]);
    __syncthreads();
    if (threadIdx.x < 8) desc[(size_t)blockIdx.x * 8 + threadIdx.x] = (threadIdx.x >= 1 && threadIdx.x <= 4) ? cnt[threadIdx.x - 1] : 0;
}

__global__ void pack_offsets_kernel(int32_t *desc, PlanInfo *info)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const int64_t n_chunks = ((int64_t)lo32(info->rows.v[0]) + NK_GS_CHUNK - 1) / NK_GS_CHUNK;
    long long run = 0;
    for (int64_t ch = 0; ch < n_chunks; ++ch) {
        int32_t *d = desc + ch * 8;
        d[0] = (int32_t)run;
        run += pad4ll(2ll * d[1]) + pad4ll(4ll * d[2]) + pad4ll(8ll * d[3]) + pad4ll(d[4]);
    }
    info->pk_size = run;
}

__global__ void __launch_bounds__(PT) pack_fill_kernel(const unsigned *rbeg, const unsigned *rlen, const unsigned *loc,
                                                       const int32_t *desc, int64_t n_sum_rows, int32_t *pk)
{
    __shared__ Vec<1> sm[PT / 32];
    const int64_t r0 = (int64_t)blockIdx.x * NK_GS_CHUNK, r1 = min(r0 + (int64_t)NK_GS_CHUNK, n_sum_rows);
    const int32_t *d = desc + (size_t)blockIdx.x * 8;
    int32_t *sec[4];
    sec[0] = pk + d[0];
    sec[1] = sec[0] + pad4ll(2ll * d[1]);
    sec[2] = sec[1] + pad4ll(4ll * d[2]);
    sec[3] = sec[2] + pad4ll(8ll * d[3]);
    unsigned done[4] = {0, 0, 0, 0};                           // rows of each class in the tiles before this one
    for (int64_t base = r0; base < r1; base += PT) {
        const int64_t r = base + threadIdx.x;
        const bool on = r < r1;
        const unsigned len = on ? rlen[r] : 0u;
        const int cls = on ? len_class(len) : 0;
        Vec<1> val, ex, tot;
        val.v[0] = on ? (1ull << (16 * cls)) : 0ull;
        block_excl_scan(val, ex, tot, sm);
        if (on) {
            const unsigned k = done[cls] + (unsigned)((ex.v[0] >> (16 * cls)) & 0xffffull);
            if (cls < 3) {
                int32_t *dst = sec[cls] + (size_t)k * len;
                const unsigned b = rbeg[r];
                for (unsigned q = 0; q < len; ++q) dst[q] = (int32_t)loc[b + q];
            } else {
                sec[3][k] = (int32_t)r;
            }
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) done[k] += (unsigned)((tot.v[0] >> (16 * k)) & 0xffffull);   // <= PT per tile: 16 bits do
    }
    if (threadIdx.x == 0) {                                    // zero padding at the end of every section
        const long long used[4] = {2ll * d[1], 4ll * d[2], 8ll * d[3], (long long)d[4]};
        for (int k = 0; k < 4; ++k)
            for (long long q = used[k]; q < pad4ll(used[k]); ++q) sec[k][q] = 0;
    }
}

template <class F>
cudaError_t run_scan(const F &f, int64_t n, int sm_count, Vec<F::NC> *bsum, Vec<F::NC> *total, cudaStream_t st)
{
    const int nb = scan_grid(sm_count, n);
    scan_reduce_kernel<F><<<nb, PT, 0, st>>>(f, n, bsum);
    scan_blocks_kernel<F::NC><<<1, 32, 0, st>>>(bsum, nb, total);
    scan_emit_kernel<F><<<nb, PT, 0, st>>>(f, n, bsum, total);
    return cudaGetLastError();
}

inline unsigned lo32h(unsigned long long x) { return (unsigned)(x & 0xffffffffull); }
inline unsigned hi32h(unsigned long long x) { return (unsigned)(x >> 32); }

}  // namespace

// Small scratch inside the partial-sum block (NK_MAX_PARTIALS doubles = 512 KB, idle during set-up)
constexpr size_t PS_INFO = 0, PS_MULT = 37888, PS_BSUM = 40960, PS_TABLE = 73728, PS_DESC = 376832, PS_END = 524288;
static_assert(sizeof(PlanInfo) <= PS_MULT && PS_MULT + NK_CTAB * sizeof(int) <= PS_BSUM, "plan scratch layout");
static_assert(PS_TABLE + 256u * 296u * sizeof(unsigned) <= PS_DESC && PS_END == NK_MAX_PARTIALS * sizeof(double), "plan scratch layout");

int nk_plan_device(nk_ctx *c, const int64_t *glo_num, const double *mask, double *ctab, double *mtab, cudaStream_t st)
{
    const int64_t L = c->L;
    const nk_carve cv = nk_carve_sizes(L);
    char *gb = reinterpret_cast<char *>(c->g);
    unsigned long long *keyA = reinterpret_cast<unsigned long long *>(gb), *keyB = keyA + L;
    unsigned *locA = reinterpret_cast<unsigned *>(keyB + L), *locB = locA + L;
    unsigned *gid = locB + L, *pos = gid + L, *glen = pos + L, *gl = glen + L;         // 40 L bytes of the 48 L of G
    double *maskd = c->hf;
    PlanOut o;
    o.off = c->row_off; o.idx = c->row_idx; o.nbr = c->nbr; o.gx = c->gx; o.pk = c->pk; o.code = c->code;
    o.doff = reinterpret_cast<unsigned *>(c->hx); o.gp4 = o.doff + L;
    o.rbeg = reinterpret_cast<unsigned *>(c->dinv); o.rlen = o.rbeg + (L / 2 + 1);
    char *ps = reinterpret_cast<char *>(c->red.partials);
    PlanInfo *info = reinterpret_cast<PlanInfo *>(ps + PS_INFO);
    int *mult_dev = reinterpret_cast<int *>(ps + PS_MULT);
    void *bsum = ps + PS_BSUM;
    unsigned *table = reinterpret_cast<unsigned *>(ps + PS_TABLE);
    const int64_t max_chunks = (L / 2 + NK_GS_CHUNK - 1) / NK_GS_CHUNK + 1;
    int32_t *desc_tmp = (size_t)max_chunks * 32 <= PS_END - PS_DESC ? reinterpret_cast<int32_t *>(ps + PS_DESC)
                                                                   : reinterpret_cast<int32_t *>(o.rlen + (L / 2 + 1));
    const int grid = scan_grid(c->sm_count, L);

    // ---- upload, validate -------------------------------------------------------------------------------------
    NK_CUDA(cudaMemcpyAsync(keyA, glo_num, (size_t)L * 8, cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemcpyAsync(maskd, mask, (size_t)L * 8, cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemsetAsync(info, 0, sizeof(PlanInfo), st));
    validate_kernel<<<grid, PT, 0, st>>>(reinterpret_cast<const long long *>(keyA), maskd, L, info);
    PlanInfo head;                                                  // only its leading fields are read here
    NK_CUDA(cudaMemcpyAsync(&head, info, offsetof(PlanInfo, present), cudaMemcpyDeviceToHost, st));
    NK_CUDA(cudaStreamSynchronize(st));
    if (head.bad_id) return NK_ERR_ID;
    if (head.bad_mask) return NK_ERR_MASK;
    // ---- sort (global id, local index) ------------------------------------------------------------------------
    int passes = 1;
    while (passes < 8 && (head.max_id >> (8 * passes)) != 0) ++passes;
    const int64_t tiles = (L + RS_TILE - 1) / RS_TILE;
    const int rs_nb = (int)std::max<int64_t>(1, std::min<int64_t>(tiles, std::min(2 * c->sm_count, 296)));
    unsigned long long *ks = keyA, *kd = keyB;
    unsigned *vs = locA, *vd = locB;
    for (int p = 0; p < passes; ++p) {
        radix_count_kernel<<<rs_nb, PT, 0, st>>>(ks, L, 8 * p, table);
        radix_scan_kernel<<<1, 1024, 0, st>>>(table, 256 * rs_nb);
        if (p == 0) radix_scatter_kernel<true><<<rs_nb, PT, 0, st>>>(ks, vs, kd, vd, L, 8 * p, table);
        else radix_scatter_kernel<false><<<rs_nb, PT, 0, st>>>(ks, vs, kd, vd, L, 8 * p, table);
        std::swap(ks, kd);
        std::swap(vs, vd);
    }
    NK_CUDA(cudaGetLastError());
    const unsigned long long *key = ks;
    const unsigned *loc = vs;
    // ---- groups, rows -----------------------------------------------------------------------------------------
    NK_CUDA(cudaMemsetAsync(gl, 0, (size_t)L * 4, st));
    NK_CUDA(cudaMemsetAsync(c->gx, 0, cv.gx, st));
    NK_CUDA(cudaMemsetAsync(c->pk, 0, 256, st));
    HeadScan hs;
    hs.key = key; hs.gid = gid; hs.pos = pos;
    NK_CUDA(run_scan(hs, L, c->sm_count, reinterpret_cast<Vec<1> *>(bsum), &info->heads, st));
    group_kernel<<<grid, PT, 0, st>>>(pos, loc, maskd, L, glen, gl, info);
    RowScan rs;
    rs.gl = gl; rs.glen = glen; rs.pos = pos; rs.o = o;
    NK_CUDA(run_scan(rs, L, c->sm_count, reinterpret_cast<Vec<3> *>(bsum), &info->rows, st));
    pack_count_kernel<<<(unsigned)max_chunks, PT, 0, st>>>(o.rlen, info, desc_tmp);
    pack_offsets_kernel<<<1, 32, 0, st>>>(desc_tmp, info);
    NK_CUDA(cudaGetLastError());
    std::vector<unsigned char> raw(sizeof(PlanInfo));
    NK_CUDA(cudaMemcpyAsync(raw.data(), info, sizeof(PlanInfo), cudaMemcpyDeviceToHost, st));
    NK_CUDA(cudaStreamSynchronize(st));
    const PlanInfo &pi = *reinterpret_cast<const PlanInfo *>(raw.data());
    if (pi.ovf_n > MULT_OVF_CAP) return NK_PLAN_FALLBACK;
    // ---- the distinct multiplicities -> tables (host: at most NK_CTAB numbers) ----------------------------------
    std::vector<int> mult_values;
    for (int v = 1; v <= MULT_DIRECT; ++v)
        if (pi.present[v]) mult_values.push_back(v);
    {
        std::vector<int> big(pi.ovf, pi.ovf + pi.ovf_n);
        std::sort(big.begin(), big.end());
        big.erase(std::unique(big.begin(), big.end()), big.end());
        mult_values.insert(mult_values.end(), big.begin(), big.end());      // all > MULT_DIRECT: still ascending
    }
    if (mult_values.size() > NK_CTAB) return NK_ERR_MULT;
    for (int t = 0; t < NK_CTAB; ++t) { ctab[t] = 0.0; mtab[t] = 0.0; }
    for (size_t t = 0; t < mult_values.size(); ++t) {
        mtab[t] = (double)mult_values[t];
        ctab[t] = 1.0 / (double)mult_values[t];
    }
    NK_CUDA(cudaMemcpyAsync(mult_dev, mult_values.data(), mult_values.size() * sizeof(int), cudaMemcpyHostToDevice, st));
    // ---- sizes and the places of the variable-length arrays -----------------------------------------------------
    const int64_t n_sum_rows = lo32h(pi.rows.v[0]), n_msk_rows = hi32h(pi.rows.v[0]);
    const int64_t n_sum_listed = lo32h(pi.rows.v[1]), n_msk_listed = hi32h(pi.rows.v[1]);
    const int64_t n_gx_rows = lo32h(pi.rows.v[2]), quads = hi32h(pi.rows.v[2]);
    c->n_unique = (int64_t)lo32h(pi.heads.v[0]);
    c->n_shared_unique = (int64_t)pi.n_shared;
    c->n_masked_unique = (int64_t)pi.n_masked;
    c->n_sum_rows = n_sum_rows; c->n_rows = n_sum_rows + n_msk_rows;
    c->n_sum_listed = n_sum_listed; c->n_listed = n_sum_listed + n_msk_listed;
    c->n_gx_rows = n_gx_rows;
    c->gx_rows = c->gx + 4 * (quads + 4);
    c->gx_blk = c->gx_rows + (n_gx_rows + 3) / 4 * 4;
    const int64_t n_chunks = (n_sum_rows + NK_GS_CHUNK - 1) / NK_GS_CHUNK;
    c->n_gs_chunks = n_chunks;
    c->n_pk = (int64_t)std::max<long long>(pi.pk_size, 1);
    c->gs_desc = c->pk + nk_align_up((size_t)c->n_pk, 64);
    // ---- per-point arrays, gx_blk, packed rows ------------------------------------------------------------------
    fill_kernel<<<grid, PT, 0, st>>>(gid, pos, glen, loc, maskd, L, o, mult_dev, (int)mult_values.size(), info);
    const int nvb = nk_gsu_blocks(c->sm_count, L >> 1);
    gx_blk_kernel<<<(nvb + 1 + PT - 1) / PT, PT, 0, st>>>(c->gx, c->gx_rows, (int)n_gx_rows, L, nvb, c->gx_blk);
    if (n_chunks > 0) {
        pack_fill_kernel<<<(unsigned)n_chunks, PT, 0, st>>>(o.rbeg, o.rlen, loc, desc_tmp, n_sum_rows, c->pk);
        NK_CUDA(cudaMemcpyAsync(c->gs_desc, desc_tmp, (size_t)n_chunks * 32, cudaMemcpyDeviceToDevice, st));
    } else {
        NK_CUDA(cudaMemsetAsync(c->gs_desc, 0, 32, st));
    }
    NK_CUDA(cudaGetLastError());
    int clash = 0;
    NK_CUDA(cudaMemcpyAsync(&clash, &info->mask_clash, sizeof(int), cudaMemcpyDeviceToHost, st));
    NK_CUDA(cudaStreamSynchronize(st));
    if (clash) return NK_ERR_MASK;
    return NK_OK;
}
