// nk_setup.cu -- nk_setup (S 8(a) row a0, S 3 call stack (4)): validate, GLL basis, carve the
// caller's workspace, build the gather-scatter plan (sort (global id, local index) pairs -> CSR of nodes that are
// shared or masked -> multiplicity codes, gather codes, packed rows), run the geometry kernel.  One-time cost; the
// paper discards set-up and warm-up from its timings too.
// The plan is built on the DEVICE by default (nk_plan.cu).  This file keeps the host builder (nk_set_plan_builder(1),
// and the fallback for degenerate inputs): all cores via OpenMP (parallel radix sort, group walk cut at group
// boundaries, chunked packing); every array it builds is independent of the thread count and equal, bit for bit, to
// the device builder's (tests/test_gpu_operators.py).
#include <algorithm>
#include <chrono>
#include <cmath>
#ifdef _OPENMP
#include <omp.h>
#endif
#include <cstdlib>
#include <cstring>
#include <new>

#include "nk_host.h"

namespace {

int g_host_threads = 0;          // nk_set_host_threads; 0 = all cores

inline int host_threads()
{
#ifdef _OPENMP
    return g_host_threads > 0 ? g_host_threads : omp_get_num_procs();
#else
    return 1;
#endif
}

// The big host arrays: uninitialised (a std::vector would zero 1.8 GB on ONE thread at config 5 before the parallel
// loops that fill them ever run; first touch then happens in those loops, spread over the cores).
template <class T>
struct raw_buf {
    T *p;
    size_t n;
    explicit raw_buf(size_t count) : p(static_cast<T *>(std::malloc(std::max<size_t>(count, 1) * sizeof(T)))), n(count)
    {
        if (!p) throw std::bad_alloc();
    }
    ~raw_buf() { std::free(p); }
    raw_buf(const raw_buf &) = delete;
    raw_buf &operator=(const raw_buf &) = delete;
    T &operator[](size_t i) { return p[i]; }
    const T &operator[](size_t i) const { return p[i]; }
    T *data() { return p; }
    size_t size() const { return n; }
    void swap(raw_buf &o) { std::swap(p, o.p); std::swap(n, o.n); }
    void release() { std::free(p); p = nullptr; n = 0; }
};

// Stable LSD radix sort of (key, payload) by key, 8 bits per pass (256 write streams per thread stay in cache and
// TLB; 2048 did not: 0.64 s for config 5's 56.6 M pairs), only the passes max_key needs; every pass is parallel over
// contiguous chunks (per-thread histograms, bucket-major prefix, in-order scatter: stable).
template <class KeyBuf, class ValBuf>
void radix_sort_pairs(KeyBuf &key, ValBuf &val, uint64_t max_key)
{
    const int64_t n = (int64_t)key.size();
    KeyBuf key2((size_t)n);
    ValBuf val2((size_t)n);
    constexpr int BITS = 8, BUCKETS = 1 << BITS;
    const int T = host_threads();
    std::vector<int64_t> count((size_t)T * BUCKETS);
    for (int shift = 0; shift < 64 && (max_key >> shift) != 0; shift += BITS) {
#pragma omp parallel num_threads(T)
        {
#ifdef _OPENMP
            const int t = omp_get_thread_num(), TT = omp_get_num_threads();      // TT <= T: what the runtime gave us
#else
            const int t = 0, TT = 1;
#endif
            const int64_t lo = n * t / TT, hi = n * (t + 1) / TT;
            int64_t *cnt = &count[(size_t)t * BUCKETS];
            for (int b = 0; b < BUCKETS; ++b) cnt[b] = 0;
            for (int64_t i = lo; i < hi; ++i) cnt[(key[(size_t)i] >> shift) & (BUCKETS - 1)]++;
#pragma omp barrier
#pragma omp single
            {
                int64_t run = 0;
                for (int b = 0; b < BUCKETS; ++b)
                    for (int u = 0; u < TT; ++u) { const int64_t c = count[(size_t)u * BUCKETS + b]; count[(size_t)u * BUCKETS + b] = run; run += c; }
            }
            for (int64_t i = lo; i < hi; ++i) {
                const int64_t d = cnt[(key[(size_t)i] >> shift) & (BUCKETS - 1)]++;
                key2[(size_t)d] = key[(size_t)i];
                val2[(size_t)d] = val[(size_t)i];
            }
        }
        key.swap(key2);
        val.swap(val2);
    }
}

struct Row { uint32_t first, begin, len; };   // first local index, position in the sorted list, copies

int g_plan_builder = 0;          // nk_set_plan_builder: 0 = device (nk_plan.cu), 1 = host (below)

// The plan built on the host cores; the device builder (nk_plan.cu) produces the same arrays bit for bit.
int plan_host(nk_ctx *c, const int64_t *glo_num, const double *mask, double *ctab, double *mtab, cudaStream_t st)
{
    const int64_t L = c->L;
    const int T = host_threads();
    // ---- validate ids and mask ------------------------------------------------------------------
    uint64_t max_id = 0;
    int bad_id = 0, bad_mask = 0;
#pragma omp parallel for schedule(static) num_threads(T) reduction(max : max_id) reduction(| : bad_id, bad_mask)
    for (int64_t l = 0; l < L; ++l) {
        if (glo_num[l] < 0) { bad_id = 1; continue; }
        if ((uint64_t)glo_num[l] > max_id) max_id = (uint64_t)glo_num[l];
        if (!(mask[l] == 0.0 || mask[l] == 1.0)) bad_mask = 1;
    }
    if (bad_id) return NK_ERR_ID;
    if (bad_mask) return NK_ERR_MASK;
    // ---- group local indices by global id (stable: ascending local index inside a group) ---------
    raw_buf<uint64_t> key((size_t)L);
    raw_buf<uint32_t> loc((size_t)L);
#pragma omp parallel for schedule(static) num_threads(T)
    for (int64_t l = 0; l < L; ++l) { key[(size_t)l] = (uint64_t)glo_num[l]; loc[(size_t)l] = (uint32_t)l; }
    radix_sort_pairs(key, loc, max_id);

    // ---- walk the groups, in parallel over chunks of the sorted list cut at group boundaries ------------------
    raw_buf<uint8_t> code((size_t)L);
    std::vector<std::vector<Row>> sum_t((size_t)T), msk_t((size_t)T);
    std::vector<std::vector<int64_t>> mult_t((size_t)T);
    std::vector<int64_t> cut((size_t)T + 1);
    for (int t = 0; t <= T; ++t) {
        int64_t p = L * t / T;
        while (p > 0 && p < L && key[(size_t)p] == key[(size_t)p - 1]) ++p;       // forward to the next group start
        cut[(size_t)t] = p;
    }
    int64_t n_unique = 0, n_shared = 0, n_masked = 0;
    int mask_clash = 0;
#pragma omp parallel for schedule(static, 1) num_threads(T) reduction(+ : n_unique, n_shared, n_masked) reduction(| : mask_clash)
    for (int t = 0; t < T; ++t) {
        std::vector<Row> &sr = sum_t[(size_t)t], &mr = msk_t[(size_t)t];
        std::vector<int64_t> &mv = mult_t[(size_t)t];
        for (int64_t b = cut[(size_t)t]; b < cut[(size_t)t + 1];) {
            int64_t e = b + 1;
            while (e < L && key[(size_t)e] == key[(size_t)b]) ++e;
            const int64_t len = e - b;
            const double m0 = mask[loc[(size_t)b]];
            for (int64_t q = b + 1; q < e; ++q)
                if (mask[loc[(size_t)q]] != m0) mask_clash = 1;
            ++n_unique;
            if (len > 1) ++n_shared;
            if (m0 == 0.0) ++n_masked;
            if (std::find(mv.begin(), mv.end(), len) == mv.end()) mv.push_back(len);
            Row r{loc[(size_t)b], (uint32_t)b, (uint32_t)len};
            if (m0 == 0.0) mr.push_back(r);
            else if (len > 1) sr.push_back(r);
            b = e;
        }
    }
    if (mask_clash) return NK_ERR_MASK;
    std::vector<int64_t> mult_values;                 // distinct multiplicities, ascending
    for (const auto &mv : mult_t)
        for (int64_t v : mv)
            if (std::find(mult_values.begin(), mult_values.end(), v) == mult_values.end()) mult_values.push_back(v);
    if (mult_values.size() > NK_CTAB) return NK_ERR_MULT;
    std::sort(mult_values.begin(), mult_values.end());
    for (int t = 0; t < NK_CTAB; ++t) { ctab[t] = 0.0; mtab[t] = 0.0; }
    for (size_t t = 0; t < mult_values.size(); ++t) {
        mtab[t] = (double)mult_values[t];
        ctab[t] = 1.0 / (double)mult_values[t];
    }
    // second pass: per-point codes
#pragma omp parallel for schedule(static, 1) num_threads(T)
    for (int t = 0; t < T; ++t)
        for (int64_t b = cut[(size_t)t]; b < cut[(size_t)t + 1];) {
            int64_t e = b + 1;
            while (e < L && key[(size_t)e] == key[(size_t)b]) ++e;
            const int64_t len = e - b;
            const int ti = (int)(std::lower_bound(mult_values.begin(), mult_values.end(), len) - mult_values.begin());
            const uint8_t cd = (uint8_t)(ti | (mask[loc[(size_t)b]] == 0.0 ? NK_CODE_MASKED : 0u));
            for (int64_t q = b; q < e; ++q) code[loc[(size_t)q]] = cd;
            b = e;
        }
    key.release();
    // ---- order rows by first local index so neighbouring threads touch neighbouring memory (first indices are
    // distinct, so the order does not depend on how the walk was cut) -------------------------------------------
    auto gather_sorted = [&](std::vector<std::vector<Row>> &parts) {
        size_t total = 0;
        for (const auto &v : parts) total += v.size();
        std::vector<Row> all;
        all.reserve(total);
        for (auto &v : parts) { all.insert(all.end(), v.begin(), v.end()); std::vector<Row>().swap(v); }
        std::vector<uint64_t> k(total);
        std::vector<uint32_t> id(total);
#pragma omp parallel for schedule(static) num_threads(T)
        for (int64_t i = 0; i < (int64_t)total; ++i) { k[(size_t)i] = all[(size_t)i].first; id[(size_t)i] = (uint32_t)i; }
        radix_sort_pairs(k, id, (uint64_t)(L > 0 ? L - 1 : 0));
        std::vector<Row> out(total);
#pragma omp parallel for schedule(static) num_threads(T)
        for (int64_t i = 0; i < (int64_t)total; ++i) out[(size_t)i] = all[id[(size_t)i]];
        return out;
    };
    std::vector<Row> sum_rows = gather_sorted(sum_t), msk_rows = gather_sorted(msk_t);
    const int64_t n_sum_rows = (int64_t)sum_rows.size(), n_rows = n_sum_rows + (int64_t)msk_rows.size();
    std::vector<int32_t> off((size_t)n_rows + 1);
    int64_t n_listed = 0, n_sum_listed = 0;
    {
        int64_t pos = 0, row = 0;
        for (const Row &r : sum_rows) { off[(size_t)row++] = (int32_t)pos; pos += r.len; }
        n_sum_listed = pos;
        for (const Row &r : msk_rows) { off[(size_t)row++] = (int32_t)pos; pos += r.len; }
        off[(size_t)row] = (int32_t)pos;
        n_listed = pos;
    }
    raw_buf<int32_t> idx((size_t)std::max<int64_t>(n_listed, 1));
#pragma omp parallel for schedule(static) num_threads(T)
    for (int64_t row = 0; row < n_rows; ++row) {
        const Row &r = row < n_sum_rows ? sum_rows[(size_t)row] : msk_rows[(size_t)(row - n_sum_rows)];
        int32_t *dst = &idx[(size_t)off[(size_t)row]];
        for (uint32_t q = 0; q < r.len; ++q) dst[q] = (int32_t)loc[r.begin + q];
    }
    // packed copy of the summed rows: chunks of NK_GS_CHUNK consecutive rows (ascending first local index,
    // so a chunk works on one neighbourhood of memory), inside a chunk the rows of 2, 4 and 8 copies
    // packed by length, rows of any other length as row ids into the CSR.  Descriptor per chunk:
    // {offset into pk, n2, n4, n8, n_other, 0, 0, 0}.  Sizes first, then offsets, then the chunks in parallel.
    const int64_t n_chunks = (n_sum_rows + NK_GS_CHUNK - 1) / NK_GS_CHUNK;
    std::vector<int32_t> desc((size_t)std::max<int64_t>(n_chunks, 1) * 8, 0);
    auto pad4 = [](int64_t v) { return (v + 3) / 4 * 4; };
#pragma omp parallel for schedule(static) num_threads(T)
    for (int64_t ch = 0; ch < n_chunks; ++ch) {
        const int64_t r0 = ch * NK_GS_CHUNK, r1 = std::min<int64_t>(r0 + NK_GS_CHUNK, n_sum_rows);
        int32_t cnt[4] = {0, 0, 0, 0};
        for (int64_t r = r0; r < r1; ++r) {
            const uint32_t len = sum_rows[(size_t)r].len;
            ++cnt[len == 2 ? 0 : len == 4 ? 1 : len == 8 ? 2 : 3];
        }
        int32_t *d = &desc[(size_t)ch * 8];
        d[1] = cnt[0]; d[2] = cnt[1]; d[3] = cnt[2]; d[4] = cnt[3];
    }
    int64_t pk_size = 0;
    for (int64_t ch = 0; ch < n_chunks; ++ch) {
        int32_t *d = &desc[(size_t)ch * 8];
        d[0] = (int32_t)pk_size;
        pk_size += pad4(2 * (int64_t)d[1]) + pad4(4 * (int64_t)d[2]) + pad4(8 * (int64_t)d[3]) + pad4(d[4]);
    }
    std::vector<int32_t> pk((size_t)std::max<int64_t>(pk_size, 1), 0);
#pragma omp parallel for schedule(static) num_threads(T)
    for (int64_t ch = 0; ch < n_chunks; ++ch) {
        const int64_t r0 = ch * NK_GS_CHUNK, r1 = std::min<int64_t>(r0 + NK_GS_CHUNK, n_sum_rows);
        const int32_t *d = &desc[(size_t)ch * 8];
        int32_t *p2 = &pk[(size_t)d[0]], *p4 = p2 + pad4(2 * (int64_t)d[1]), *p8 = p4 + pad4(4 * (int64_t)d[2]);
        int32_t *po = p8 + pad4(8 * (int64_t)d[3]);
        for (int64_t r = r0; r < r1; ++r) {
            const Row &row = sum_rows[(size_t)r];
            if (row.len == 2 || row.len == 4 || row.len == 8) {
                int32_t *&dst = row.len == 2 ? p2 : row.len == 4 ? p4 : p8;
                for (uint32_t q = 0; q < row.len; ++q) *dst++ = (int32_t)loc[row.begin + q];
            } else {
                *po++ = (int32_t)r;
            }
        }
    }
    // per-point gather codes of the fused gs (nk_internal.h nk_ctx::nbr)
    raw_buf<int32_t> nbr((size_t)L);
    std::vector<int32_t> gx, gx_rows;
#pragma omp parallel for schedule(static) num_threads(T)
    for (int64_t l = 0; l < L; ++l) nbr[(size_t)l] = (int32_t)l;
#pragma omp parallel for schedule(static) num_threads(T)
    for (int64_t r = 0; r < n_sum_rows; ++r) {
        const Row &row = sum_rows[(size_t)r];
        if (row.len == 2) {
            const uint32_t a = loc[row.begin], b = loc[row.begin + 1];
            nbr[a] = (int32_t)b;
            nbr[b] = (int32_t)a;
        }
    }
    for (int64_t r = 0; r < n_sum_rows; ++r) {
        const Row &row = sum_rows[(size_t)r];
        if (row.len == 2) continue;
        while ((gx.size() + 1) % 4) gx.push_back(0);
        gx.push_back((int32_t)row.len);
        const int32_t p4 = (int32_t)(gx.size() / 4);
        gx_rows.push_back(p4);
        for (uint32_t q = 0; q < row.len; ++q) {
            gx.push_back((int32_t)loc[row.begin + q]);
            nbr[loc[row.begin + q]] = -p4 - 2;
        }
    }
    {   // 4 (Q + 3) ints, Q = the quad the next row would start at: vector loads of the last row stay in bounds
        const size_t Q = gx_rows.empty() ? 1 : (size_t)gx_rows.back() + (size_t)gx[4 * (size_t)gx_rows.back() - 1] / 4 + 1;
        gx.resize(4 * (Q + 3), 0);
    }
    c->n_gx_rows = (int64_t)gx_rows.size();
    c->gx_rows = c->gx + gx.size();
    // the list cut by the chunks of the fused kernel's blocks: a node goes to the block whose chunk holds its first copy
    const int nvb = nk_gsu_blocks(c->sm_count, L >> 1);
    std::vector<int32_t> gx_blk((size_t)nvb + 1);
    {
        const int64_t pairs = L >> 1;
        size_t k = 0;
        for (int b = 0; b <= nvb; ++b) {
            const int64_t first_point = b == nvb ? L + 1 : 4 * ((L >> 2) * (int64_t)b / nvb);
            while (k < gx_rows.size() && (int64_t)gx[4 * (size_t)gx_rows[k]] < first_point) ++k;
            gx_blk[(size_t)b] = (int32_t)k;
        }
        gx_blk[0] = 0;
    }
    c->gx_blk = c->gx_rows + ((gx_rows.size() + 3) / 4 * 4);
#pragma omp parallel for schedule(static) num_threads(T)
    for (int64_t r = 0; r < (int64_t)msk_rows.size(); ++r) {
        const Row &row = msk_rows[(size_t)r];
        for (uint32_t q = 0; q < row.len; ++q) nbr[loc[row.begin + q]] = -1;
    }
    c->n_gs_chunks = n_chunks;
    c->n_pk = (int64_t)pk.size();
    c->gs_desc = c->pk + nk_align_up(pk.size(), 64);
    c->n_unique = n_unique; c->n_shared_unique = n_shared; c->n_masked_unique = n_masked;
    c->n_rows = n_rows; c->n_listed = n_listed; c->n_sum_rows = n_sum_rows; c->n_sum_listed = n_sum_listed;

    // ---- upload the plan ------------------------------------------------------------------------------------
    NK_CUDA(cudaMemcpyAsync(c->code, code.data(), (size_t)L, cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemcpyAsync(c->row_off, off.data(), off.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    if (n_listed > 0)
        NK_CUDA(cudaMemcpyAsync(c->row_idx, idx.data(), (size_t)n_listed * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemcpyAsync(c->pk, pk.data(), pk.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemcpyAsync(c->nbr, nbr.data(), (size_t)L * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemcpyAsync(c->gx, gx.data(), gx.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    if (!gx_rows.empty())
        NK_CUDA(cudaMemcpyAsync(c->gx_rows, gx_rows.data(), gx_rows.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemcpyAsync(c->gx_blk, gx_blk.data(), gx_blk.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemcpyAsync(c->gs_desc, desc.data(), desc.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaStreamSynchronize(st));                          // the host arrays go out of scope here
    return NK_OK;
}

int setup_impl(nk_ctx *c, const double *coords, const int64_t *glo_num, const double *mask, cudaStream_t st)
{
    const int64_t L = c->L;
    double ctab[NK_CTAB], mtab[NK_CTAB];
    const auto t0 = std::chrono::steady_clock::now();
    int rc = g_plan_builder == 0 ? nk_plan_device(c, glo_num, mask, ctab, mtab, st) : NK_PLAN_FALLBACK;
    c->plan_builder = 0;
    if (rc == NK_PLAN_FALLBACK) {
        rc = plan_host(c, glo_num, mask, ctab, mtab, st);
        c->plan_builder = 1;
    }
    if (rc != NK_OK) return rc;
    c->setup_plan_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    // ---- tables, coordinates; geometry kernel ------------------------------------------------------------------
    double *D_dev = c->ctab + 2 * NK_CTAB;
    double *wq_dev = D_dev + 16 * 16;
    NK_CUDA(cudaMemcpyAsync(c->ctab, ctab, sizeof(ctab), cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemcpyAsync(c->mtab, mtab, sizeof(mtab), cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemcpyAsync(D_dev, c->D, sizeof(double) * c->n * c->n, cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemcpyAsync(wq_dev, c->wq, sizeof(double) * c->n, cudaMemcpyHostToDevice, st));
    // low parts of D (set-up only): staged in the residual-history scratch
    double Dhi[16 * 16], Dlo[16 * 16], xi_t[16], wq_t[16];
    nk_host_basis_dd(c->N, xi_t, wq_t, Dhi, Dlo);
    double *Dlo_dev = c->hist;
    NK_CUDA(cudaMemcpyAsync(Dlo_dev, Dlo, sizeof(double) * c->n * c->n, cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemsetAsync(c->red.scal, 0, 256, st));
    NK_CUDA(cudaMemsetAsync(c->red.counter, 0, 256, st));       // counter, errflag, res_dummy
    // coordinates (x|y|z planes at stride L) are staged in the r|p|w block, which is >= 3L doubles
    double *coords_dev = c->r;
    NK_CUDA(cudaMemcpyAsync(coords_dev, coords, 3 * (size_t)L * sizeof(double), cudaMemcpyHostToDevice, st));
    NK_CUDA(nk_upload_D_tables_tma());
    NK_CUDA(nk_launch_geom(c, coords_dev, D_dev, Dlo_dev, wq_dev, st));
    int err = 0;
    NK_CUDA(cudaMemcpyAsync(&err, c->errflag, sizeof(int), cudaMemcpyDeviceToHost, st));
    NK_CUDA(cudaStreamSynchronize(st));
    if (err) return NK_ERR_GEOM;
    c->setup_total_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    return NK_OK;
}

}  // namespace

extern "C" int nk_set_host_threads(int n)
{
    g_host_threads = n > 0 ? n : 0;
    return NK_OK;
}

extern "C" int nk_set_plan_builder(int which)
{
    if (which != 0 && which != 1) return NK_ERR_ARG;
    g_plan_builder = which;
    return NK_OK;
}

extern "C" int nk_setup(nk_ctx **ctx, int64_t E, int N, const double *coords, const int64_t *glo_num,
                        const double *mask, void *workspace, size_t workspace_bytes, void *stream)
{
    if (!ctx) return NK_ERR_ARG;
    *ctx = nullptr;
    int64_t L;
    if (!nk_valid_EN(E, N, &L) || !coords || !glo_num || !mask) return NK_ERR_ARG;
    const nk_carve cv = nk_carve_sizes(L);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) != 0 || workspace_bytes < cv.total)
        return NK_ERR_WORKSPACE;
    int dev = 0, sms = 0;
    NK_CUDA(cudaGetDevice(&dev));
    NK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    nk_ctx *c = new (std::nothrow) nk_ctx();
    if (!c) return NK_ERR_ALLOC;
    std::memset(c, 0, sizeof(*c));
    c->E = E; c->N = N; c->n = N + 1; c->P = (int64_t)c->n * c->n * c->n; c->L = L;
    c->device = dev; c->sm_count = sms;
    c->ws = workspace; c->ws_bytes = workspace_bytes;
    c->opt_fuse_pap = 1; c->opt_fuse_p = 2; c->opt_fuse_gs = 2; c->opt_coop = 2; c->opt_graph = 2; c->opt_pdl = 3; c->opt_defer_x = 1; c->pdl_now = 0;
    nk_host_basis(N, c->xi, c->wq, c->D);
    char *q = static_cast<char *>(workspace);
    c->g = reinterpret_cast<double2 *>(q); q += cv.g;
    c->r = reinterpret_cast<double *>(q); q += cv.vec;
    c->p = reinterpret_cast<double *>(q); q += cv.vec;
    c->pc = c->p;
    c->w = reinterpret_cast<double *>(q); q += cv.vec;
    c->hf = reinterpret_cast<double *>(q); q += cv.vec;
    c->hx = reinterpret_cast<double *>(q); q += cv.vec;
    c->dinv = reinterpret_cast<double *>(q); q += cv.vec;
    c->hf2 = reinterpret_cast<double *>(q); q += cv.vec;
    c->hx2 = reinterpret_cast<double *>(q); q += cv.vec;
    c->p2 = reinterpret_cast<double *>(q); q += cv.vec;
    c->code = reinterpret_cast<uint8_t *>(q); q += cv.code;
    c->row_off = reinterpret_cast<int32_t *>(q); q += cv.off;
    c->row_idx = reinterpret_cast<int32_t *>(q); q += cv.idx;
    c->nbr = reinterpret_cast<int32_t *>(q); q += cv.nbr;
    c->gx = reinterpret_cast<int32_t *>(q); q += cv.gx;
    c->pk = reinterpret_cast<int32_t *>(q); q += cv.pk;
    c->ctab = reinterpret_cast<double *>(q); c->mtab = c->ctab + NK_CTAB; q += cv.tabs;
    c->red.partials = reinterpret_cast<double *>(q); q += cv.partials;
    c->hist = reinterpret_cast<double *>(q); q += cv.hist;
    c->hist2 = reinterpret_cast<double *>(q); q += cv.hist;
    c->red.scal = reinterpret_cast<double *>(q); q += cv.scal;
    c->red.counter = reinterpret_cast<unsigned *>(q);
    c->red.raw = nullptr;
    c->errflag = reinterpret_cast<int *>(q + 64);
    c->res_dummy = reinterpret_cast<double *>(q + 128);
    c->coop_bar = reinterpret_cast<unsigned *>(q + 192);
    {
        int coop = 0;
        NK_CUDA(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
        c->coop_ok = coop;
        c->cluster_ok = 1;
    }
    int rc;
    try {
        rc = setup_impl(c, coords, glo_num, mask, static_cast<cudaStream_t>(stream));
    } catch (const std::bad_alloc &) {
        rc = NK_ERR_ALLOC;
    }
    if (rc != NK_OK) { delete c; return rc; }
    *ctx = c;
    return NK_OK;
}
