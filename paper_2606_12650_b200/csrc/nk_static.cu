// nk_static.cu -- nk_dot_static: the weighted dot product (S 8(a) a4) for callers that must not allocate
// and have no nk_ctx workspace at hand (code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc).  A variant of dot_kernel (nk_vec.cu): same arithmetic per entry, same deterministic two-level sum
// (per-block partial, the block that draws the last ticket adds all partials in index order), but the scratch --
// the partials and the ticket counter -- lives in ONE file-scope __device__ array instead of the caller's workspace:
//   * 16 416 doubles (about 128 KB) that every GPU which loads libnk.so holds until the process exits;
//   * a block sums a fixed run of NK_STATIC_DOT_CHUNK = 8192 entries, so the grid, hence the rounding, depends on n
//     only (not on the GPU), and n <= NK_DOT_STATIC_MAX_N = 16384 x 8192 = 2^27 entries; more: NK_ERR_SIZE;
//   * every call shares the array and finds the previous call's partials in it: they are all rewritten before they
//     are read, and the ticket counter is cleared by a memset node ahead of the kernel.  Two calls that OVERLAP on
//     the GPU (different streams, no ordering between them) race on it: order them.
// The array's name is a host-side stand-in in host code, not a device address: the address is looked up once per
// device with cudaGetSymbolAddress (nk_static_setup, also run on the first nk_dot_static of a device) and that
// pointer is what the kernel gets.  No cudaMalloc, cudaFree or allocating library routine on this path.
#include <cstdint>

#include "nk_host.h"
#include "nk_reduce.cuh"

namespace {

constexpr int SD_THREADS = 512;
constexpr int SD_CHUNK = 8192;                         // entries per block: 8 pairs per thread
constexpr int SD_MAX_BLOCKS = 16384;
constexpr int SD_HEADER = 32;                          // doubles ahead of the partials: [0] holds the ticket counter
constexpr int SD_MAX_DEVICES = 64;

static __device__ __align__(256) double g_dot_scratch[SD_HEADER + SD_MAX_BLOCKS];

double *g_scratch_addr[SD_MAX_DEVICES];               // device address of g_dot_scratch, per device ordinal (host copy)

// out[0] = sum_i c_i a_i b_i (c == nullptr: c_i = 1) over this block's run of entries, then the ordered finish
__global__ void __launch_bounds__(SD_THREADS)
dot_static_kernel(const double *__restrict__ a, const double *__restrict__ b, const double *__restrict__ c, int64_t n,
                  nk_reduce_ws ws, double *out)
{
    __shared__ double s_red[33];
    const int64_t lo = (int64_t)blockIdx.x * SD_CHUNK;
    const int64_t hi = lo + SD_CHUNK < n ? lo + SD_CHUNK : n;
    double acc = 0.0;
    const bool vec = ((reinterpret_cast<uintptr_t>(a) | reinterpret_cast<uintptr_t>(b) | reinterpret_cast<uintptr_t>(c)) & 15u) == 0;
    if (vec) {
        const int64_t q0 = lo >> 1, q1 = hi >> 1;          // lo is even: whole pairs, then at most one odd entry
        for (int64_t q = q0 + threadIdx.x; q < q1; q += SD_THREADS) {
            const double2 av = reinterpret_cast<const double2 *>(a)[q];
            const double2 bv = reinterpret_cast<const double2 *>(b)[q];
            double2 cv = make_double2(1.0, 1.0);
            if (c) cv = reinterpret_cast<const double2 *>(c)[q];
            acc = fma(cv.x * av.x, bv.x, acc);
            acc = fma(cv.y * av.y, bv.y, acc);
        }
        if ((hi & 1) && threadIdx.x == 0) acc = fma((c ? c[hi - 1] : 1.0) * a[hi - 1], b[hi - 1], acc);
    } else {                                               // unaligned views: same entries per thread, scalar loads
        const int64_t q0 = lo >> 1, q1 = hi >> 1;
        for (int64_t q = q0 + threadIdx.x; q < q1; q += SD_THREADS) {
            acc = fma((c ? c[2 * q] : 1.0) * a[2 * q], b[2 * q], acc);
            acc = fma((c ? c[2 * q + 1] : 1.0) * a[2 * q + 1], b[2 * q + 1], acc);
        }
        if ((hi & 1) && threadIdx.x == 0) acc = fma((c ? c[hi - 1] : 1.0) * a[hi - 1], b[hi - 1], acc);
    }
    nk_grid_reduce(acc, s_red, ws, NK_EPI_STORE, out);
}

int static_setup(double **addr)
{
    int dev = 0;
    NK_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= SD_MAX_DEVICES) return NK_ERR_ARG;
    if (!g_scratch_addr[dev]) {
        double *p = nullptr;
        NK_CUDA(cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_dot_scratch));
        if (!p) return NK_ERR_CUDA;
        g_scratch_addr[dev] = p;                           // racing first calls store the same value
    }
    if (addr) *addr = g_scratch_addr[dev];
    return NK_OK;
}

}  // namespace

extern "C" int nk_static_setup(void) { return static_setup(nullptr); }

extern "C" int64_t nk_dot_static_max_n(void) { return (int64_t)SD_MAX_BLOCKS * SD_CHUNK; }

extern "C" int nk_dot_static(const double *a, const double *b, const double *c, int64_t n, double *out, void *stream)
{
    if (n < 0 || !out || (n > 0 && (!a || !b))) return NK_ERR_ARG;
    if (n > (int64_t)SD_MAX_BLOCKS * SD_CHUNK) return NK_ERR_SIZE;
    double *scratch = nullptr;
    const int rc = static_setup(&scratch);
    if (rc != NK_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    nk_reduce_ws ws;
    ws.partials = scratch + SD_HEADER;
    ws.counter = reinterpret_cast<unsigned *>(scratch);
    ws.scal = nullptr;
    ws.raw = nullptr;
    NK_CUDA(cudaMemsetAsync(scratch, 0, SD_HEADER * sizeof(double), st));      // the ticket counter starts at zero
    const int64_t nb = n == 0 ? 1 : (n + SD_CHUNK - 1) / SD_CHUNK;             // n = 0: one block stores 0
    dot_static_kernel<<<(unsigned)nb, SD_THREADS, 0, st>>>(a, b, c, n, ws, out);
    NK_CUDA(cudaGetLastError());
    return NK_OK;
}
