// nk_basis.cpp -- Gauss-Lobatto-Legendre basis for order N on the host (S 8(c) O1; "derivative
// matrices ... depend only on the polynomial order").  Tiny, run once per nk_setup, long double.
//
// Nodes: -1, +1 and the N-1 zeros of q(x) = P_{N+1}(x) - P_{N-1}(x)  (q = -(2N+1)/(N(N+1)) (1-x^2) P_N'),
// found by Newton with q'(x) = (2N+1) P_N(x).  Weights w_i = 2 / (N (N+1) P_N(xi_i)^2).
// D_im = l_m'(xi_i) = P_N(xi_i) / (P_N(xi_m) (xi_i - xi_m)), i != m; D_00 = -N(N+1)/4 = -D_NN; else 0.
#include <cmath>

#include "nk_internal.h"

namespace {

// P_{k}(x) for k = deg-1, deg, deg+1 by the three-term recurrence (k+1)P_{k+1} = (2k+1)xP_k - kP_{k-1}.
void legendre3(int deg, long double x, long double *pm, long double *p0, long double *pp)
{
    long double a = 1.0L, b = x;   // P_0, P_1
    if (deg == 0) { *pm = 0.0L; *p0 = a; *pp = b; return; }
    for (int k = 1; k < deg; ++k) {
        const long double c = ((2 * k + 1) * x * b - k * a) / (k + 1);
        a = b; b = c;
    }
    // a = P_{deg-1}, b = P_deg
    *pm = a; *p0 = b;
    *pp = ((2 * deg + 1) * x * b - deg * a) / (deg + 1);
}

}  // namespace

void nk_host_basis_dd(int N, double *xi, double *w, double *D, double *Dlo)
{
    const int n = N + 1;
    long double x[16], pn[16];
    const long double pi = 3.14159265358979323846264338327950288L;
    x[0] = -1.0L; x[N] = 1.0L;
    for (int i = 1; i < N; ++i) {
        // start from the Chebyshev-Gauss-Lobatto point, which interlaces well enough for N <= 15
        long double t = -cosl(pi * i / N);
        for (int it = 0; it < 100; ++it) {
            long double pm, p0, pp;
            legendre3(N, t, &pm, &p0, &pp);
            const long double dt = (pp - pm) / ((2 * N + 1) * p0);
            t -= dt;
            if (fabsl(dt) < 1e-19L) break;
        }
        x[i] = t;
    }
    for (int i = 0; i <= N / 2; ++i) {       // enforce xi_i = -xi_{N-i}
        const long double s = 0.5L * (x[N - i] - x[i]);
        x[i] = -s; x[N - i] = s;
    }
    if (N % 2 == 0) x[N / 2] = 0.0L;
    for (int i = 0; i < n; ++i) {
        long double pm, pp;
        legendre3(N, x[i], &pm, &pn[i], &pp);
    }
    for (int i = 0; i < n; ++i) {
        xi[i] = (double)x[i];
        w[i] = (double)(2.0L / ((long double)N * (N + 1) * pn[i] * pn[i]));
    }
    for (int i = 0; i < n; ++i)
        for (int m = 0; m < n; ++m) {
            long double d;
            if (i != m) d = pn[i] / (pn[m] * (x[i] - x[m]));
            else if (i == 0) d = -(long double)N * (N + 1) / 4.0L;
            else if (i == N) d = (long double)N * (N + 1) / 4.0L;
            else d = 0.0L;
            D[i * n + m] = (double)d;
            if (Dlo) Dlo[i * n + m] = (double)(d - (long double)(double)d);   // D = hi + lo to ~2^-64
        }
}

void nk_host_basis(int N, double *xi, double *w, double *D) { nk_host_basis_dd(N, xi, w, D, nullptr); }
