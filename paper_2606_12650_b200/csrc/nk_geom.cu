// nk_geom.cu -- set-up kernel: geometric factors (S 8(a) a0, S 8(c) O2; BJ "the 6 symmetric
// geometric factors G").  Per point: the 3x3 Jacobian d(x,y,z)/d(r,s,t) by applying D along
// r, s, t to the coordinates; J = det > 0; G_ab = w_i w_j w_k * J * (grad a . grad b).
//
// Conditioning (reading R22): differentiating ABSOLUTE coordinates cancels
// ~|D|max * |x| / (h/2) leading digits, so coordinates are first taken relative to the element's
// first node (D annihilates constants; the subtraction of nearby numbers is exact or 1 ulp of the
// small difference).  With inverse metrics = cofactors / J:
//   G_ab = w3 * (cof_a . cof_b) / J,   cof_r = (x_s x x_t), cof_s = (x_t x x_r), cof_t = (x_r x x_s).
// Output: double2 pairs (rr,rs) (rt,ss) (st,tt) in the layout of nk_g_index() -- always 16-byte
// aligned per point, also for odd (N+1)^3 (S 7 hard part 5).  One block per element; run once, not on the timed path.
#include "nk_internal.h"

namespace {

constexpr int GEOM_THREADS = 256;

// Double-double accumulation of one derivative sum: acc += (dh + dl) * v, products by FMA (exact
// two-product), sums by two-sum.  The nine coordinate derivatives cancel ~|D|max |x| / (h/2)
// leading digits even after the shift to the element's first node, and D rounded to double is
// itself only good to 2^-53: with D = hi + lo (from the host's long double) and a double-double
// accumulator the derivatives come out correctly rounded, and G to a few ulp (R22).
struct dd { double hi, lo; };
__device__ __forceinline__ void dd_fma(dd &acc, double dh, double dl, double v)
{
    const double p = dh * v;
    const double e = fma(dh, v, -p) + dl * v;        // exact product error + low part
    const double s = acc.hi + p;
    const double bb = s - acc.hi;
    const double err = (acc.hi - (s - bb)) + (p - bb);
    acc.hi = s;
    acc.lo += err + e;
}
__device__ __forceinline__ double dd_val(const dd &a) { return a.hi + a.lo; }

__global__ void __launch_bounds__(GEOM_THREADS)
geom_kernel(const double *__restrict__ coords, const double *__restrict__ Dg, const double *__restrict__ Dlg,
            const double *__restrict__ wq,
            int n, int64_t L, double2 *__restrict__ g, int *__restrict__ errflag)
{
    __shared__ double s_D[16 * 16], s_Dl[16 * 16];
    __shared__ double s_w[16];
    for (int t = threadIdx.x; t < n * n; t += GEOM_THREADS) { s_D[t] = Dg[t]; s_Dl[t] = Dlg[t]; }
    if (threadIdx.x < n) s_w[threadIdx.x] = wq[threadIdx.x];
    __syncthreads();
    const int P = n * n * n;
    const int64_t base = (int64_t)blockIdx.x * P;
    const double *xe = coords + base, *ye = coords + L + base, *ze = coords + 2 * L + base;
    const double x0 = xe[0], y0 = ye[0], z0 = ze[0];
    int bad = 0;
    for (int q = threadIdx.x; q < P; q += GEOM_THREADS) {
        const int i = q % n, j = (q / n) % n, k = q / (n * n);
        dd axr{0, 0}, axs{0, 0}, axt{0, 0}, ayr{0, 0}, ays{0, 0}, ayt{0, 0}, azr{0, 0}, azs{0, 0}, azt{0, 0};
        for (int m = 0; m < n; ++m) {
            const double di = s_D[i * n + m], dj = s_D[j * n + m], dk = s_D[k * n + m];
            const double li = s_Dl[i * n + m], lj = s_Dl[j * n + m], lk = s_Dl[k * n + m];
            const int qr = m + n * j + n * n * k, qs = i + n * m + n * n * k, qt = i + n * j + n * n * m;
            dd_fma(axr, di, li, xe[qr] - x0); dd_fma(ayr, di, li, ye[qr] - y0); dd_fma(azr, di, li, ze[qr] - z0);
            dd_fma(axs, dj, lj, xe[qs] - x0); dd_fma(ays, dj, lj, ye[qs] - y0); dd_fma(azs, dj, lj, ze[qs] - z0);
            dd_fma(axt, dk, lk, xe[qt] - x0); dd_fma(ayt, dk, lk, ye[qt] - y0); dd_fma(azt, dk, lk, ze[qt] - z0);
        }
        const double xr = dd_val(axr), xs = dd_val(axs), xt = dd_val(axt);
        const double yr = dd_val(ayr), ys = dd_val(ays), yt = dd_val(ayt);
        const double zr = dd_val(azr), zs = dd_val(azs), zt = dd_val(azt);
        // cofactor vectors (rows of J * inverse Jacobian)
        const double rx = ys * zt - yt * zs, ry = zs * xt - zt * xs, rz = xs * yt - xt * ys;   // x_s x x_t
        const double sx = yt * zr - yr * zt, sy = zt * xr - zr * xt, sz = xt * yr - xr * yt;   // x_t x x_r
        const double tx = yr * zs - ys * zr, ty = zr * xs - zs * xr, tz = xr * ys - xs * yr;   // x_r x x_s
        const double J = xr * rx + yr * ry + zr * rz;
        if (!(J > 0.0) || !isfinite(J)) bad = 1;
        const double sc = s_w[i] * s_w[j] * s_w[k] / J;
        const double grr = sc * (rx * rx + ry * ry + rz * rz);
        const double grs = sc * (rx * sx + ry * sy + rz * sz);
        const double grt = sc * (rx * tx + ry * ty + rz * tz);
        const double gss = sc * (sx * sx + sy * sy + sz * sz);
        const double gst = sc * (sx * tx + sy * ty + sz * tz);
        const double gtt = sc * (tx * tx + ty * ty + tz * tz);
        const int t2 = i + n * j;
        g[nk_g_index(blockIdx.x, k, 0, t2, n)] = make_double2(grr, grs);
        g[nk_g_index(blockIdx.x, k, 1, t2, n)] = make_double2(grt, gss);
        g[nk_g_index(blockIdx.x, k, 2, t2, n)] = make_double2(gst, gtt);
    }
    if (bad) atomicOr(errflag, 1);
}

// rr|rs|rt|ss|st|tt planes of L for nk_get_geom
__global__ void __launch_bounds__(GEOM_THREADS)
unpack_geom_kernel(const double2 *__restrict__ g, double *__restrict__ G6, int64_t L, int n)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int n2 = n * n, P = n2 * n;
    for (int64_t l = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; l < L; l += stride) {
        const int64_t e = l / P;
        const int q = (int)(l - e * P), k = q / n2, t2 = q - k * n2;
        const double2 a = g[nk_g_index(e, k, 0, t2, n)], b = g[nk_g_index(e, k, 1, t2, n)],
                      c = g[nk_g_index(e, k, 2, t2, n)];
        G6[l] = a.x; G6[L + l] = a.y; G6[2 * L + l] = b.x;
        G6[3 * L + l] = b.y; G6[4 * L + l] = c.x; G6[5 * L + l] = c.y;
    }
}

// diag(A_L) per local point (the Jacobi preconditioner of the original Nekbone):
//   sum_m ( D[m][i]^2 G_rr(m,j,k) + D[m][j]^2 G_ss(i,m,k) + D[m][k]^2 G_tt(i,j,m) )
//   + 2 ( D[i][i] D[j][j] G_rs + D[i][i] D[k][k] G_rt + D[j][j] D[k][k] G_st )(i,j,k)
// One block per element; run once per context, not on the timed path.
__global__ void __launch_bounds__(GEOM_THREADS)
diag_kernel(const double2 *__restrict__ g, const double *__restrict__ Dg, int n, double *__restrict__ diag)
{
    __shared__ double s_D[16 * 16];
    for (int t = threadIdx.x; t < n * n; t += GEOM_THREADS) s_D[t] = Dg[t];
    __syncthreads();
    const int n2 = n * n, P = n2 * n;
    const int64_t e = blockIdx.x;
    for (int q = threadIdx.x; q < P; q += GEOM_THREADS) {
        const int i = q % n, j = (q / n) % n, k = q / n2;
        double s = 0.0;
        for (int m = 0; m < n; ++m) {
            const double di = s_D[m * n + i], dj = s_D[m * n + j], dk = s_D[m * n + k];
            s = fma(di * di, g[nk_g_index(e, k, 0, m + n * j, n)].x, s);       // rr at (m,j,k)
            s = fma(dj * dj, g[nk_g_index(e, k, 1, i + n * m, n)].y, s);       // ss at (i,m,k)
            s = fma(dk * dk, g[nk_g_index(e, m, 2, i + n * j, n)].y, s);       // tt at (i,j,m)
        }
        const int t2 = i + n * j;
        const double grs = g[nk_g_index(e, k, 0, t2, n)].y, grt = g[nk_g_index(e, k, 1, t2, n)].x,
                     gst = g[nk_g_index(e, k, 2, t2, n)].x;
        const double dii = s_D[i * n + i], djj = s_D[j * n + j], dkk = s_D[k * n + k];
        s += 2.0 * (dii * djj * grs + dii * dkk * grt + djj * dkk * gst);
        diag[e * P + q] = s;
    }
}

// d = 1/d, and 0 on Dirichlet nodes (z = M^-1 r vanishes there)
__global__ void __launch_bounds__(GEOM_THREADS)
invert_diag_kernel(double *__restrict__ d, const uint8_t *__restrict__ code, int64_t L)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t l = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; l < L; l += stride)
        d[l] = (code[l] & NK_CODE_MASKED) ? 0.0 : 1.0 / d[l];
}

}  // namespace

cudaError_t nk_launch_geom(nk_ctx *c, const double *coords_dev, const double *D_dev, const double *Dlo_dev,
                           const double *wq_dev,
                           cudaStream_t st)
{
    geom_kernel<<<(unsigned)c->E, GEOM_THREADS, 0, st>>>(coords_dev, D_dev, Dlo_dev, wq_dev, c->n, c->L, c->g, c->errflag);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t nk_launch_get_geom(nk_ctx *c, double *G6, cudaStream_t st)
{
    int64_t nb = (c->L + GEOM_THREADS - 1) / GEOM_THREADS;
    if (nb > (int64_t)c->sm_count * 32) nb = (int64_t)c->sm_count * 32;
    unpack_geom_kernel<<<(unsigned)nb, GEOM_THREADS, 0, st>>>(c->g, G6, c->L, c->n);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t nk_launch_diag(nk_ctx *c, double *diag, cudaStream_t st)
{
    const double *D_dev = c->ctab + 2 * NK_CTAB;          // uploaded by nk_setup, kept
    diag_kernel<<<(unsigned)c->E, GEOM_THREADS, 0, st>>>(c->g, D_dev, c->n, diag);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t nk_launch_invert_diag(nk_ctx *c, double *d, cudaStream_t st)
{
    int64_t nb = (c->L + GEOM_THREADS - 1) / GEOM_THREADS;
    if (nb > (int64_t)c->sm_count * 32) nb = (int64_t)c->sm_count * 32;
    invert_diag_kernel<<<(unsigned)nb, GEOM_THREADS, 0, st>>>(d, c->code, c->L);
    c->launches++;
    return cudaGetLastError();
}
