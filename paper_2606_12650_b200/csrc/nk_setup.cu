// nk_setup.cu -- nk_setup (S 8(a) row a0, S 3 call stack (4)): validate, GLL basis, carve the
// caller's workspace, build the gather-scatter plan on the host (sort (global id, local index)
// pairs -> CSR of nodes that are shared or masked -> multiplicity codes), upload, run the geometry
// kernel.  One-time cost; the paper discards set-up and warm-up from its timings too.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>

#include "nk_host.h"

namespace {

// Stable LSD radix sort of (key, payload) by key, 11 bits per pass, only the passes max_key needs.
void radix_sort_pairs(std::vector<uint64_t> &key, std::vector<uint32_t> &val, uint64_t max_key)
{
    const size_t n = key.size();
    std::vector<uint64_t> key2(n);
    std::vector<uint32_t> val2(n);
    constexpr int BITS = 11, BUCKETS = 1 << BITS;
    std::vector<size_t> count(BUCKETS);
    for (int shift = 0; shift < 64 && (max_key >> shift) != 0; shift += BITS) {
        std::fill(count.begin(), count.end(), 0);
        for (size_t i = 0; i < n; ++i) count[(key[i] >> shift) & (BUCKETS - 1)]++;
        size_t run = 0;
        for (int b = 0; b < BUCKETS; ++b) { const size_t c = count[b]; count[b] = run; run += c; }
        for (size_t i = 0; i < n; ++i) {
            const size_t d = count[(key[i] >> shift) & (BUCKETS - 1)]++;
            key2[d] = key[i];
            val2[d] = val[i];
        }
        key.swap(key2);
        val.swap(val2);
    }
}

struct Row { uint32_t first, begin, len; };   // first local index, position in the sorted list, copies

int setup_impl(nk_ctx *c, const double *coords, const int64_t *glo_num, const double *mask, cudaStream_t st)
{
    const int64_t L = c->L;
    // ---- validate ids and mask ------------------------------------------------------------------
    uint64_t max_id = 0;
    for (int64_t l = 0; l < L; ++l) {
        if (glo_num[l] < 0) return NK_ERR_ID;
        if ((uint64_t)glo_num[l] > max_id) max_id = (uint64_t)glo_num[l];
        if (!(mask[l] == 0.0 || mask[l] == 1.0)) return NK_ERR_MASK;
    }
    // ---- group local indices by global id (stable: ascending local index inside a group) ---------
    std::vector<uint64_t> key((size_t)L);
    std::vector<uint32_t> loc((size_t)L);
    for (int64_t l = 0; l < L; ++l) { key[l] = (uint64_t)glo_num[l]; loc[l] = (uint32_t)l; }
    radix_sort_pairs(key, loc, max_id);

    std::vector<uint8_t> code((size_t)L);
    std::vector<Row> sum_rows, msk_rows;
    std::vector<int64_t> mult_values;                 // distinct multiplicities, ascending after the walk
    int64_t n_unique = 0, n_shared = 0, n_masked = 0;
    // first pass over groups: sizes, mask consistency, distinct multiplicities
    for (int64_t b = 0; b < L;) {
        int64_t e = b + 1;
        while (e < L && key[e] == key[b]) ++e;
        const int64_t len = e - b;
        const double m0 = mask[loc[b]];
        for (int64_t q = b + 1; q < e; ++q)
            if (mask[loc[q]] != m0) return NK_ERR_MASK;
        ++n_unique;
        if (len > 1) ++n_shared;
        if (m0 == 0.0) ++n_masked;
        if (std::find(mult_values.begin(), mult_values.end(), len) == mult_values.end()) {
            if (mult_values.size() >= NK_CTAB) return NK_ERR_MULT;
            mult_values.push_back(len);
        }
        Row r{loc[b], (uint32_t)b, (uint32_t)len};
        if (m0 == 0.0) msk_rows.push_back(r);
        else if (len > 1) sum_rows.push_back(r);
        b = e;
    }
    std::sort(mult_values.begin(), mult_values.end());
    double ctab[NK_CTAB], mtab[NK_CTAB];
    for (int t = 0; t < NK_CTAB; ++t) { ctab[t] = 0.0; mtab[t] = 0.0; }
    for (size_t t = 0; t < mult_values.size(); ++t) {
        mtab[t] = (double)mult_values[t];
        ctab[t] = 1.0 / (double)mult_values[t];
    }
    // second pass: per-point codes
    for (int64_t b = 0; b < L;) {
        int64_t e = b + 1;
        while (e < L && key[e] == key[b]) ++e;
        const int64_t len = e - b;
        const int t = (int)(std::lower_bound(mult_values.begin(), mult_values.end(), len) - mult_values.begin());
        const uint8_t cd = (uint8_t)(t | (mask[loc[b]] == 0.0 ? NK_CODE_MASKED : 0u));
        for (int64_t q = b; q < e; ++q) code[loc[q]] = cd;
        b = e;
    }
    std::vector<uint64_t>().swap(key);
    // ---- order rows by first local index so neighbouring threads touch neighbouring memory ------
    auto by_first = [](const Row &x, const Row &y) { return x.first < y.first; };
    std::sort(sum_rows.begin(), sum_rows.end(), by_first);
    std::sort(msk_rows.begin(), msk_rows.end(), by_first);
    const int64_t n_sum_rows = (int64_t)sum_rows.size(), n_rows = n_sum_rows + (int64_t)msk_rows.size();
    std::vector<int32_t> off((size_t)n_rows + 1);
    int64_t n_listed = 0, n_sum_listed = 0;
    for (const Row &r : sum_rows) n_sum_listed += r.len;
    n_listed = n_sum_listed;
    for (const Row &r : msk_rows) n_listed += r.len;
    std::vector<int32_t> idx((size_t)std::max<int64_t>(n_listed, 1));
    {
        int64_t pos = 0, row = 0;
        for (const std::vector<Row> *rows : {&sum_rows, &msk_rows})
            for (const Row &r : *rows) {
                off[row++] = (int32_t)pos;
                for (uint32_t q = 0; q < r.len; ++q) idx[pos++] = (int32_t)loc[r.begin + q];
            }
        off[row] = (int32_t)pos;
    }
    // packed copy of the summed rows: chunks of NK_GS_CHUNK consecutive rows (ascending first local index,
    // so a chunk works on one neighbourhood of memory), inside a chunk the rows of 2, 4 and 8 copies
    // packed by length, rows of any other length as row ids into the CSR.  Descriptor per chunk:
    // {offset into pk, n2, n4, n8, n_other, 0, 0, 0}.
    const int64_t n_chunks = (n_sum_rows + NK_GS_CHUNK - 1) / NK_GS_CHUNK;
    std::vector<int32_t> pk, desc((size_t)std::max<int64_t>(n_chunks, 1) * 8, 0);
    pk.reserve((size_t)n_sum_listed + 4 * (size_t)n_chunks + 64);
    for (int64_t ch = 0; ch < n_chunks; ++ch) {
        const int64_t r0 = ch * NK_GS_CHUNK, r1 = std::min<int64_t>(r0 + NK_GS_CHUNK, n_sum_rows);
        int32_t *d = &desc[(size_t)ch * 8];
        d[0] = (int32_t)pk.size();
        for (int len : {2, 4, 8}) {
            int32_t cnt = 0;
            for (int64_t r = r0; r < r1; ++r) {
                const Row &row = sum_rows[(size_t)r];
                if ((int)row.len != len) continue;
                for (uint32_t q = 0; q < row.len; ++q) pk.push_back((int32_t)loc[row.begin + q]);
                ++cnt;
            }
            while (pk.size() % 4) pk.push_back(0);                     // 16-byte aligned class starts
            d[len == 2 ? 1 : len == 4 ? 2 : 3] = cnt;
        }
        int32_t no = 0;
        for (int64_t r = r0; r < r1; ++r) {
            const uint32_t len = sum_rows[(size_t)r].len;
            if (len != 2 && len != 4 && len != 8) { pk.push_back((int32_t)r); ++no; }
        }
        while (pk.size() % 4) pk.push_back(0);
        d[4] = no;
    }
    if (pk.empty()) pk.push_back(0);
    // per-point gather codes of the fused gs (nk_internal.h nk_ctx::nbr)
    std::vector<int32_t> nbr((size_t)L), gx, gx_rows;
    for (int64_t l = 0; l < L; ++l) nbr[(size_t)l] = (int32_t)l;
    for (int64_t r = 0; r < n_sum_rows; ++r) {
        const Row &row = sum_rows[(size_t)r];
        if (row.len == 2) {
            const uint32_t a = loc[row.begin], b = loc[row.begin + 1];
            nbr[a] = (int32_t)b;
            nbr[b] = (int32_t)a;
        } else {
            while ((gx.size() + 1) % 4) gx.push_back(0);
            gx.push_back((int32_t)row.len);
            const int32_t p4 = (int32_t)(gx.size() / 4);
            gx_rows.push_back(p4);
            for (uint32_t q = 0; q < row.len; ++q) {
                gx.push_back((int32_t)loc[row.begin + q]);
                nbr[loc[row.begin + q]] = -p4 - 2;
            }
        }
    }
    gx.resize((gx.size() + 12 + 3) / 4 * 4, 0);              // vector loads of the last row stay in bounds; 16-byte multiple
    c->n_gx_rows = (int64_t)gx_rows.size();
    c->gx_rows = c->gx + gx.size();
    for (const Row &row : msk_rows)
        for (uint32_t q = 0; q < row.len; ++q) nbr[loc[row.begin + q]] = -1;
    c->n_gs_chunks = n_chunks;
    c->gs_desc = c->pk + nk_align_up(pk.size(), 64);
    c->n_unique = n_unique; c->n_shared_unique = n_shared; c->n_masked_unique = n_masked;
    c->n_rows = n_rows; c->n_listed = n_listed; c->n_sum_rows = n_sum_rows; c->n_sum_listed = n_sum_listed;

    // ---- upload plan, tables, coordinates; geometry kernel -------------------------------------
    double *D_dev = c->ctab + 2 * NK_CTAB;
    double *wq_dev = D_dev + 16 * 16;
    NK_CUDA(cudaMemcpyAsync(c->code, code.data(), (size_t)L, cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemcpyAsync(c->row_off, off.data(), off.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    if (n_listed > 0)
        NK_CUDA(cudaMemcpyAsync(c->row_idx, idx.data(), (size_t)n_listed * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemcpyAsync(c->pk, pk.data(), pk.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemcpyAsync(c->nbr, nbr.data(), (size_t)L * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemcpyAsync(c->gx, gx.data(), gx.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    if (!gx_rows.empty())
        NK_CUDA(cudaMemcpyAsync(c->gx_rows, gx_rows.data(), gx_rows.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    NK_CUDA(cudaMemcpyAsync(c->gs_desc, desc.data(), desc.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
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
    return NK_OK;
}

}  // namespace

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
    c->opt_fuse_pap = 1; c->opt_fuse_p = 2; c->opt_fuse_gs = 2; c->opt_coop = 2; c->opt_graph = 2; c->opt_pdl = 3; c->pdl_now = 0;
    nk_host_basis(N, c->xi, c->wq, c->D);
    char *q = static_cast<char *>(workspace);
    c->g = reinterpret_cast<double2 *>(q); q += cv.g;
    c->r = reinterpret_cast<double *>(q); q += cv.vec;
    c->p = reinterpret_cast<double *>(q); q += cv.vec;
    c->w = reinterpret_cast<double *>(q); q += cv.vec;
    c->hf = reinterpret_cast<double *>(q); q += cv.vec;
    c->hx = reinterpret_cast<double *>(q); q += cv.vec;
    c->dinv = reinterpret_cast<double *>(q); q += cv.vec;
    c->code = reinterpret_cast<uint8_t *>(q); q += cv.code;
    c->row_off = reinterpret_cast<int32_t *>(q); q += cv.off;
    c->row_idx = reinterpret_cast<int32_t *>(q); q += cv.idx;
    c->nbr = reinterpret_cast<int32_t *>(q); q += cv.nbr;
    c->gx = reinterpret_cast<int32_t *>(q); q += cv.gx;
    c->pk = reinterpret_cast<int32_t *>(q); q += cv.pk;
    c->ctab = reinterpret_cast<double *>(q); c->mtab = c->ctab + NK_CTAB; q += cv.tabs;
    c->red.partials = reinterpret_cast<double *>(q); q += cv.partials;
    c->hist = reinterpret_cast<double *>(q); q += cv.hist;
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
