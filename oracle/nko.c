/* nko.c -- ORACLE (test infrastructure, not the product).  See nko.h for scope and citations.
 *
 * Style: every function is the definition written out -- plain nested loops, summation index
 * ascending, no blocking, no fusion, no reordering.  OpenMP appears only as `parallel for` over
 * independent elements / node groups / fixed-size chunks, so results do not depend on the thread
 * count.  Compile with -ffp-contract=off (oracle/build.py); a second build with contraction on
 * is used by the tests to measure the oracle's own rounding band.
 */
#include "nko.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

struct nko_ctx {
    int64_t E, L;
    int N, n;
    double *xi, *wq, *D;      /* O1 basis                                   */
    double *G[6];             /* O2: rr rs rt ss st tt, each L              */
    double *J;                /* O2: Jacobian determinant, L                */
    double *mask;             /* O5: copy of the caller's mask, L           */
    double *c;                /* O7: 1/multiplicity, L                      */
    double *mult;             /* O7: multiplicity = gs(1), L                */
    /* O4: local indices grouped by global id; group g = order[start[g] .. start[g+1]) with the
     * local indices ascending inside a group. */
    int64_t n_groups;
    int64_t *start;
    int64_t *order;
    int64_t n_shared_unique, n_masked_unique;
    int dot_mode;
    long double Dl[65 * 65];      /* D before rounding to double (geometry only) */
};

/* ------------------------------------------------------------------------------------------
 * O1. GLL basis (textbook; the paper only says the derivative matrices depend on the
 * polynomial order).  Legendre three-term recurrence in long double.
 * ---------------------------------------------------------------------------------------- */
static void legendre(int N, long double x, long double *PN, long double *PNm1)
{
    long double p0 = 1.0L, p1 = x;
    if (N == 0) { *PN = 1.0L; *PNm1 = 0.0L; return; }
    for (int k = 1; k < N; ++k) {
        long double p2 = ((2 * k + 1) * x * p1 - k * p0) / (k + 1);
        p0 = p1;
        p1 = p2;
    }
    *PN = p1;
    *PNm1 = p0;
}

/* Dl (may be NULL): the derivative matrix before its rounding to double, for O2 (R22). */
static int basis_ld(int N, double *xi, double *w, double *D, long double *Dl)
{
    if (N < 1 || N > 64 || !xi || !w || !D) return NKO_ERR_ARG;
    const int n = N + 1;
    const long double pi = 3.14159265358979323846264338327950288L;
    long double *x = (long double *)malloc(sizeof(long double) * n);
    long double *P = (long double *)malloc(sizeof(long double) * n);
    if (!x || !P) { free(x); free(P); return NKO_ERR_ALLOC; }

    /* nodes: xi_0 = -1, xi_N = 1, interior = roots of P_N'.  Newton from the Chebyshev-Lobatto
     * guess -cos(pi i / N).  P_N' = N (x P_N - P_{N-1}) / (x^2 - 1);
     * P_N'' = (2 x P_N' - N(N+1) P_N) / (1 - x^2)  (Legendre's equation). */
    x[0] = -1.0L;
    x[N] = 1.0L;
    for (int i = 1; i < N; ++i) {
        long double xk = -cosl(pi * i / N);
        for (int it = 0; it < 200; ++it) {
            long double PN, PNm1;
            legendre(N, xk, &PN, &PNm1);
            long double d1 = N * (xk * PN - PNm1) / (xk * xk - 1.0L);
            long double d2 = (2.0L * xk * d1 - (long double)N * (N + 1) * PN) / (1.0L - xk * xk);
            long double dx = d1 / d2;
            xk -= dx;
            if (fabsl(dx) < 1e-21L) break;
        }
        x[i] = xk;
    }
    /* symmetrise: xi_i = -xi_{N-i} */
    for (int i = 0; i <= N / 2; ++i) {
        long double s = 0.5L * (x[N - i] - x[i]);
        x[i] = -s;
        x[N - i] = s;
    }
    for (int i = 0; i < n; ++i) {
        long double PN, PNm1;
        legendre(N, x[i], &PN, &PNm1);
        P[i] = PN;
    }
    for (int i = 0; i < n; ++i) {
        xi[i] = (double)x[i];
        w[i] = (double)(2.0L / ((long double)N * (N + 1) * P[i] * P[i]));
    }
    for (int i = 0; i < n; ++i)
        for (int m = 0; m < n; ++m) {
            long double d;
            if (i != m) d = P[i] / (P[m] * (x[i] - x[m]));
            else if (i == 0) d = -(long double)N * (N + 1) / 4.0L;
            else if (i == N) d = (long double)N * (N + 1) / 4.0L;
            else d = 0.0L;
            D[i * n + m] = (double)d;
            if (Dl) Dl[i * n + m] = d;
        }
    free(x);
    free(P);
    return NKO_OK;
}

int nko_basis(int N, double *xi, double *w, double *D) { return basis_ld(N, xi, w, D, NULL); }

/* ------------------------------------------------------------------------------------------
 * O2. Geometry: x_r = sum_m D[i][m] x(m,j,k), x_s = sum_m D[j][m] x(i,m,k),
 * x_t = sum_m D[k][m] x(i,j,m) (same for y, z); J = det d(x,y,z)/d(r,s,t) > 0; inverse metrics
 * by cofactors / J; G_ab = w_i w_j w_k J (grad a . grad b), order rr rs rt ss st tt.
 * ---------------------------------------------------------------------------------------- */
static int geometry(nko_ctx *c, const double *coords)
{
    const int n = c->n;
    const int64_t P = (int64_t)n * n * n, L = c->L;
    const long double *D = c->Dl;      /* unrounded: a rounded D has row sums ~1e-16 |D|, which
                                        * times |x| / (h/2) would cost G three digits (R22) */
    const double *wq = c->wq;
    const double *X = coords, *Y = coords + L, *Z = coords + 2 * L;
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(| : bad)
    for (int64_t e = 0; e < c->E; ++e) {
        const double *x = X + e * P, *y = Y + e * P, *z = Z + e * P;
        for (int k = 0; k < n; ++k)
            for (int j = 0; j < n; ++j)
                for (int i = 0; i < n; ++i) {
                    /* long double throughout: differentiating absolute coordinates cancels
                     * |D| |x| / (h/2) ~ 10^3 leading digits on fine meshes (R22), so
                     * the oracle evaluates O2 in extended precision and rounds G once. */
                    long double xr = 0, xs = 0, xt = 0, yr = 0, ys = 0, yt = 0, zr = 0, zs = 0, zt = 0;
                    for (int m = 0; m < n; ++m) {
                        const int64_t lr = m + n * j + n * n * k;
                        const int64_t ls = i + n * m + n * n * k;
                        const int64_t lt = i + n * j + n * n * m;
                        xr += D[i * n + m] * x[lr];
                        yr += D[i * n + m] * y[lr];
                        zr += D[i * n + m] * z[lr];
                        xs += D[j * n + m] * x[ls];
                        ys += D[j * n + m] * y[ls];
                        zs += D[j * n + m] * z[ls];
                        xt += D[k * n + m] * x[lt];
                        yt += D[k * n + m] * y[lt];
                        zt += D[k * n + m] * z[lt];
                    }
                    const long double J = xr * (ys * zt - yt * zs) - xs * (yr * zt - yt * zr)
                                        + xt * (yr * zs - ys * zr);
                    const int64_t l = e * P + i + n * j + n * n * k;
                    c->J[l] = (double)J;
                    if (!(J > 0.0L) || !isfinite((double)J)) { bad |= 1; continue; }
                    /* rows of the inverse Jacobian: grad r, grad s, grad t */
                    const long double rx = (ys * zt - yt * zs) / J;
                    const long double ry = -(xs * zt - xt * zs) / J;
                    const long double rz = (xs * yt - xt * ys) / J;
                    const long double sx = -(yr * zt - yt * zr) / J;
                    const long double sy = (xr * zt - xt * zr) / J;
                    const long double sz = -(xr * yt - xt * yr) / J;
                    const long double tx = (yr * zs - ys * zr) / J;
                    const long double ty = -(xr * zs - xs * zr) / J;
                    const long double tz = (xr * ys - xs * yr) / J;
                    const long double W = (long double)wq[i] * wq[j] * wq[k] * J;
                    c->G[0][l] = (double)(W * (rx * rx + ry * ry + rz * rz));
                    c->G[1][l] = (double)(W * (rx * sx + ry * sy + rz * sz));
                    c->G[2][l] = (double)(W * (rx * tx + ry * ty + rz * tz));
                    c->G[3][l] = (double)(W * (sx * sx + sy * sy + sz * sz));
                    c->G[4][l] = (double)(W * (sx * tx + sy * ty + sz * tz));
                    c->G[5][l] = (double)(W * (tx * tx + ty * ty + tz * tz));
                }
    }
    return bad ? NKO_ERR_GEOM : NKO_OK;
}

/* ------------------------------------------------------------------------------------------
 * O4 set-up: group local indices by global id (sort (id, l) pairs).
 * ---------------------------------------------------------------------------------------- */
typedef struct { int64_t g, l; } pair_t;

static int pair_cmp(const void *a, const void *b)
{
    const pair_t *p = (const pair_t *)a, *q = (const pair_t *)b;
    if (p->g != q->g) return p->g < q->g ? -1 : 1;
    if (p->l != q->l) return p->l < q->l ? -1 : 1;
    return 0;
}

static int build_groups(nko_ctx *c, const int64_t *glo, const double *mask)
{
    const int64_t L = c->L;
    pair_t *pr = (pair_t *)malloc(sizeof(pair_t) * (size_t)L);
    if (!pr) return NKO_ERR_ALLOC;
    for (int64_t l = 0; l < L; ++l) {
        if (glo[l] < 0) { free(pr); return NKO_ERR_ID; }
        if (!(mask[l] == 0.0 || mask[l] == 1.0)) { free(pr); return NKO_ERR_MASK; }
        pr[l].g = glo[l];
        pr[l].l = l;
    }
    qsort(pr, (size_t)L, sizeof(pair_t), pair_cmp);
    int64_t ng = 0;
    for (int64_t q = 0; q < L; ++q)
        if (q == 0 || pr[q].g != pr[q - 1].g) ++ng;
    c->n_groups = ng;
    c->start = (int64_t *)malloc(sizeof(int64_t) * (size_t)(ng + 1));
    c->order = (int64_t *)malloc(sizeof(int64_t) * (size_t)L);
    if (!c->start || !c->order) { free(pr); return NKO_ERR_ALLOC; }
    int64_t g = -1;
    for (int64_t q = 0; q < L; ++q) {
        if (q == 0 || pr[q].g != pr[q - 1].g) c->start[++g] = q;
        c->order[q] = pr[q].l;
    }
    c->start[ng] = L;
    free(pr);
    /* counts, and mask consistency over the copies of a node */
    c->n_shared_unique = 0;
    c->n_masked_unique = 0;
    for (int64_t gi = 0; gi < ng; ++gi) {
        const int64_t a = c->start[gi], b = c->start[gi + 1];
        const double m0 = mask[c->order[a]];
        for (int64_t q = a + 1; q < b; ++q)
            if (mask[c->order[q]] != m0) return NKO_ERR_MASK;
        if (b - a > 1) c->n_shared_unique++;
        if (m0 == 0.0) c->n_masked_unique++;
    }
    return NKO_OK;
}

int nko_setup(nko_ctx **out, int64_t E, int N, const double *coords,
              const int64_t *glo_num, const double *mask)
{
    if (!out) return NKO_ERR_ARG;
    *out = NULL;
    if (E <= 0 || N < 1 || N > 64 || !coords || !glo_num || !mask) return NKO_ERR_ARG;
    nko_ctx *c = (nko_ctx *)calloc(1, sizeof(nko_ctx));
    if (!c) return NKO_ERR_ALLOC;
    c->E = E;
    c->N = N;
    c->n = N + 1;
    c->L = E * (int64_t)c->n * c->n * c->n;
    const size_t Lb = sizeof(double) * (size_t)c->L;
    c->xi = (double *)malloc(sizeof(double) * c->n);
    c->wq = (double *)malloc(sizeof(double) * c->n);
    c->D = (double *)malloc(sizeof(double) * c->n * c->n);
    for (int a = 0; a < 6; ++a) c->G[a] = (double *)calloc(1, Lb);
    c->J = (double *)malloc(Lb);
    c->mask = (double *)malloc(Lb);
    c->c = (double *)malloc(Lb);
    c->mult = (double *)malloc(Lb);
    int ok = c->xi && c->wq && c->D && c->J && c->mask && c->c && c->mult;
    for (int a = 0; a < 6; ++a) ok = ok && c->G[a];
    if (!ok) { nko_free(c); return NKO_ERR_ALLOC; }
    int rc = basis_ld(N, c->xi, c->wq, c->D, c->Dl);
    if (rc == NKO_OK) rc = build_groups(c, glo_num, mask);
    if (rc == NKO_OK) rc = geometry(c, coords);
    if (rc != NKO_OK) { nko_free(c); return rc; }
    memcpy(c->mask, mask, Lb);
    /* O7: mult = gs(1); c = 1/mult */
    for (int64_t l = 0; l < c->L; ++l) c->mult[l] = 1.0;
    nko_gs(c, c->mult);
    for (int64_t l = 0; l < c->L; ++l) c->c[l] = 1.0 / c->mult[l];
    *out = c;
    return NKO_OK;
}

void nko_free(nko_ctx *c)
{
    if (!c) return;
    free(c->xi); free(c->wq); free(c->D);
    for (int a = 0; a < 6; ++a) free(c->G[a]);
    free(c->J); free(c->mask); free(c->c); free(c->mult);
    free(c->start); free(c->order);
    free(c);
}

/* ------------------------------------------------------------------------------------------
 * O3. ax_e: u_r, u_s, u_t = D along r, s, t; (w_r, w_s, w_t) = G (u_r, u_s, u_t);
 * w = D^T along r of w_r + D^T along s of w_s + D^T along t of w_t.
 * ---------------------------------------------------------------------------------------- */
int nko_ax_e(nko_ctx *c, const double *u, double *w)
{
    if (!c || !u || !w || u == w) return NKO_ERR_ARG;
    const int n = c->n;
    const int64_t P = (int64_t)n * n * n;
    const double *D = c->D;
    int fail = 0;
#pragma omp parallel
    {
        double *wr = (double *)malloc(sizeof(double) * (size_t)P * 3);
        if (!wr) {
#pragma omp atomic write
            fail = 1;
        }
        double *ws = wr ? wr + P : NULL, *wt = wr ? wr + 2 * P : NULL;
#pragma omp for schedule(static)
        for (int64_t e = 0; e < c->E; ++e) {
            if (!wr) continue;
            const double *ue = u + e * P;
            double *we = w + e * P;
            for (int k = 0; k < n; ++k)
                for (int j = 0; j < n; ++j)
                    for (int i = 0; i < n; ++i) {
                        double ur = 0.0, us = 0.0, ut = 0.0;
                        for (int m = 0; m < n; ++m) ur += D[i * n + m] * ue[m + n * j + n * n * k];
                        for (int m = 0; m < n; ++m) us += D[j * n + m] * ue[i + n * m + n * n * k];
                        for (int m = 0; m < n; ++m) ut += D[k * n + m] * ue[i + n * j + n * n * m];
                        const int64_t q = i + n * j + n * n * k, l = e * P + q;
                        const double grr = c->G[0][l], grs = c->G[1][l], grt = c->G[2][l];
                        const double gss = c->G[3][l], gst = c->G[4][l], gtt = c->G[5][l];
                        wr[q] = grr * ur + grs * us + grt * ut;
                        ws[q] = grs * ur + gss * us + gst * ut;
                        wt[q] = grt * ur + gst * us + gtt * ut;
                    }
            for (int k = 0; k < n; ++k)
                for (int j = 0; j < n; ++j)
                    for (int i = 0; i < n; ++i) {
                        double s = 0.0;
                        for (int m = 0; m < n; ++m) s += D[m * n + i] * wr[m + n * j + n * n * k];
                        for (int m = 0; m < n; ++m) s += D[m * n + j] * ws[i + n * m + n * n * k];
                        for (int m = 0; m < n; ++m) s += D[m * n + k] * wt[i + n * j + n * n * m];
                        we[i + n * j + n * n * k] = s;
                    }
        }
        free(wr);
    }
    return fail ? NKO_ERR_ALLOC : NKO_OK;
}

/* O4. gs: for each distinct global id, sum the copies in ascending local index, then every copy
 * receives the sum.  (per-node ordered gather loop, then ordered scatter loop.) */
int nko_gs(nko_ctx *c, double *v)
{
    if (!c || !v) return NKO_ERR_ARG;
#pragma omp parallel for schedule(static)
    for (int64_t g = 0; g < c->n_groups; ++g) {
        const int64_t a = c->start[g], b = c->start[g + 1];
        if (b - a == 1) continue;                 /* single copy: untouched, bitwise */
        double s = 0.0;
        for (int64_t q = a; q < b; ++q) s += v[c->order[q]];
        for (int64_t q = a; q < b; ++q) v[c->order[q]] = s;
    }
    return NKO_OK;
}

/* O5. mask */
int nko_mask(nko_ctx *c, double *v)
{
    if (!c || !v) return NKO_ERR_ARG;
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < c->L; ++l) v[l] = c->mask[l] * v[l];
    return NKO_OK;
}

/* O6. ax = mask o gs o ax_e */
int nko_ax(nko_ctx *c, const double *u, double *w)
{
    int rc = nko_ax_e(c, u, w);
    if (rc == NKO_OK) rc = nko_gs(c, w);
    if (rc == NKO_OK) rc = nko_mask(c, w);
    return rc;
}

/* O8 inner product <a,b>_c = sum_l c_l a_l b_l, each unique node counted once (reading R3).
 * Accumulated in long double over fixed chunks of 65536 points (chunk sums then added in
 * order), so the value does not depend on the OpenMP thread count. */
#define NKO_CHUNK 65536
int nko_dot(nko_ctx *c, const double *a, const double *b, double *out)
{
    if (!c || !a || !b || !out) return NKO_ERR_ARG;
    const int64_t L = c->L;
    if (c->dot_mode == 1) {
        double s = 0.0;
        for (int64_t l = 0; l < L; ++l) s += c->c[l] * a[l] * b[l];
        *out = s;
        return NKO_OK;
    }
    const int64_t nch = (L + NKO_CHUNK - 1) / NKO_CHUNK;
    long double *part = (long double *)malloc(sizeof(long double) * (size_t)nch);
    if (!part) return NKO_ERR_ALLOC;
#pragma omp parallel for schedule(static)
    for (int64_t ch = 0; ch < nch; ++ch) {
        const int64_t l0 = ch * NKO_CHUNK, l1 = (l0 + NKO_CHUNK < L) ? l0 + NKO_CHUNK : L;
        long double s = 0.0L;
        for (int64_t l = l0; l < l1; ++l) s += (long double)c->c[l] * (long double)a[l] * (long double)b[l];
        part[ch] = s;
    }
    long double s = 0.0L;
    for (int64_t ch = 0; ch < nch; ++ch) s += part[ch];
    free(part);
    *out = (double)s;
    return NKO_OK;
}

/* O8. CG: r = mask o f; x = 0; p = r; rho = <r,r>_c. */
int nko_cg_init(nko_ctx *c, const double *f, double *x, double *r, double *p, double *rho)
{
    if (!c || !f || !x || !r || !p || !rho) return NKO_ERR_ARG;
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < c->L; ++l) {
        r[l] = c->mask[l] * f[l];
        x[l] = 0.0;
        p[l] = r[l];
    }
    return nko_dot(c, r, r, rho);
}

/* O8, iteration k: w = ax(p); pap = <w,p>_c; alpha = rho/pap; x += alpha p; r -= alpha w;
 * rho' = <r,r>_c; beta = rho'/rho; p = r + beta p.  Guards: rho = 0 or pap = 0 -> alpha = beta = 0. */
int nko_cg_step(nko_ctx *c, double *x, double *r, double *p, double *w, double *scal)
{
    if (!c || !x || !r || !p || !w || !scal) return NKO_ERR_ARG;
    const int64_t L = c->L;
    const double rho = scal[0];
    int rc = nko_ax(c, p, w);
    if (rc != NKO_OK) return rc;
    double pap;
    rc = nko_dot(c, w, p, &pap);
    if (rc != NKO_OK) return rc;
    const double alpha = (rho == 0.0 || pap == 0.0) ? 0.0 : rho / pap;
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < L; ++l) x[l] = x[l] + alpha * p[l];
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < L; ++l) r[l] = r[l] - alpha * w[l];
    double rho1;
    rc = nko_dot(c, r, r, &rho1);
    if (rc != NKO_OK) return rc;
    const double beta = (rho == 0.0 || pap == 0.0) ? 0.0 : rho1 / rho;
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < L; ++l) p[l] = r[l] + beta * p[l];
    scal[1] = pap;
    scal[2] = alpha;
    scal[3] = rho1;
    scal[4] = beta;
    return NKO_OK;
}

int nko_cg(nko_ctx *c, const double *f, double *x, int niter, double *res_hist)
{
    if (!c || !f || !x || niter < 0 || !res_hist) return NKO_ERR_ARG;
    const size_t Lb = sizeof(double) * (size_t)c->L;
    double *r = (double *)malloc(Lb), *p = (double *)malloc(Lb), *w = (double *)malloc(Lb);
    if (!r || !p || !w) { free(r); free(p); free(w); return NKO_ERR_ALLOC; }
    double scal[5] = {0, 0, 0, 0, 0};
    int rc = nko_cg_init(c, f, x, r, p, &scal[0]);
    if (rc == NKO_OK) res_hist[0] = sqrt(scal[0]);
    for (int k = 1; k <= niter && rc == NKO_OK; ++k) {
        rc = nko_cg_step(c, x, r, p, w, scal);
        res_hist[k] = sqrt(scal[3]);
        scal[0] = scal[3];
    }
    free(r); free(p); free(w);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * NEXT row f-3: the Jacobi (diagonal) preconditioner of the original Nekbone, which
 * the paper's variant omits.
 * diag = Q Q^T diag(A_L): the diagonal of the assembled operator in local layout.  Entry l = (i,j,k)
 * of A_L = sum_ab D_a^T diag(G_ab) D_b, written out:
 *   sum_m ( D[m][i]^2 G_rr(m,j,k) + D[m][j]^2 G_ss(i,m,k) + D[m][k]^2 G_tt(i,j,m) )
 *   + 2 ( D[i][i] D[j][j] G_rs(l) + D[i][i] D[k][k] G_rt(l) + D[j][j] D[k][k] G_st(l) )
 * (a cross term D_a[q,l] D_b[q,l], a != b, is non-zero only for q = l).
 * ---------------------------------------------------------------------------------------- */
int nko_diag(nko_ctx *c, double *diag)
{
    if (!c || !diag) return NKO_ERR_ARG;
    const int n = c->n;
    const int64_t P = (int64_t)n * n * n;
    const double *D = c->D;
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < c->E; ++e) {
        const double *grr = c->G[0] + e * P, *grs = c->G[1] + e * P, *grt = c->G[2] + e * P;
        const double *gss = c->G[3] + e * P, *gst = c->G[4] + e * P, *gtt = c->G[5] + e * P;
        for (int k = 0; k < n; ++k)
            for (int j = 0; j < n; ++j)
                for (int i = 0; i < n; ++i) {
                    const int64_t l = i + n * j + (int64_t)n * n * k;
                    double s = 0.0;
                    for (int m = 0; m < n; ++m) {
                        s += D[m * n + i] * D[m * n + i] * grr[m + n * j + n * n * k];
                        s += D[m * n + j] * D[m * n + j] * gss[i + n * m + n * n * k];
                        s += D[m * n + k] * D[m * n + k] * gtt[i + n * j + n * n * m];
                    }
                    s += 2.0 * (D[i * n + i] * D[j * n + j] * grs[l] + D[i * n + i] * D[k * n + k] * grt[l]
                                + D[j * n + j] * D[k * n + k] * gst[l]);
                    diag[e * P + l] = s;
                }
    }
    return nko_gs(c, diag);
}

/* Jacobi-preconditioned CG (the original Nekbone's iteration; z = M^-1 r with M = diag, z = 0 on
 * Dirichlet nodes): r = mask o f; x = 0; z = r/diag; p = z; rho = <r,z>_c; hist[0] = sqrt<r,r>_c.
 * k = 1..niter: w = ax(p); pap = <w,p>_c; alpha = rho/pap; x += alpha p; r -= alpha w; z = r/diag;
 * rho' = <r,z>_c; hist[k] = sqrt<r,r>_c; beta = rho'/rho; p = z + beta p.  Guards as in O8. */
int nko_pcg(nko_ctx *c, const double *f, double *x, int niter, double *res_hist)
{
    if (!c || !f || !x || niter < 0 || !res_hist) return NKO_ERR_ARG;
    const int64_t L = c->L;
    const size_t Lb = sizeof(double) * (size_t)L;
    double *r = (double *)malloc(Lb), *p = (double *)malloc(Lb), *w = (double *)malloc(Lb);
    double *z = (double *)malloc(Lb), *dg = (double *)malloc(Lb);
    int rc = (r && p && w && z && dg) ? nko_diag(c, dg) : NKO_ERR_ALLOC;
    double rho = 0.0, rr = 0.0;
    if (rc == NKO_OK) {
#pragma omp parallel for schedule(static)
        for (int64_t l = 0; l < L; ++l) {
            r[l] = c->mask[l] * f[l];
            x[l] = 0.0;
            z[l] = (c->mask[l] == 0.0) ? 0.0 : r[l] / dg[l];
            p[l] = z[l];
        }
        rc = nko_dot(c, r, z, &rho);
        if (rc == NKO_OK) rc = nko_dot(c, r, r, &rr);
        res_hist[0] = sqrt(rr);
    }
    for (int k = 1; k <= niter && rc == NKO_OK; ++k) {
        double pap, rho1;
        rc = nko_ax(c, p, w);
        if (rc == NKO_OK) rc = nko_dot(c, w, p, &pap);
        if (rc != NKO_OK) break;
        const double alpha = (rho == 0.0 || pap == 0.0) ? 0.0 : rho / pap;
#pragma omp parallel for schedule(static)
        for (int64_t l = 0; l < L; ++l) x[l] = x[l] + alpha * p[l];
#pragma omp parallel for schedule(static)
        for (int64_t l = 0; l < L; ++l) r[l] = r[l] - alpha * w[l];
#pragma omp parallel for schedule(static)
        for (int64_t l = 0; l < L; ++l) z[l] = (c->mask[l] == 0.0) ? 0.0 : r[l] / dg[l];
        rc = nko_dot(c, r, z, &rho1);
        if (rc == NKO_OK) rc = nko_dot(c, r, r, &rr);
        res_hist[k] = sqrt(rr);
        const double beta = (rho == 0.0 || pap == 0.0) ? 0.0 : rho1 / rho;
#pragma omp parallel for schedule(static)
        for (int64_t l = 0; l < L; ++l) p[l] = z[l] + beta * p[l];
        rho = rho1;
    }
    free(r); free(p); free(w); free(z); free(dg);
    return rc;
}

int nko_set_dot_mode(nko_ctx *c, int mode)
{
    if (!c || (mode != 0 && mode != 1)) return NKO_ERR_ARG;
    c->dot_mode = mode;
    return NKO_OK;
}

int nko_get_sizes(nko_ctx *c, int64_t *n_local, int64_t *n_unique,
                  int64_t *n_shared_unique, int64_t *n_masked_unique)
{
    if (!c) return NKO_ERR_ARG;
    if (n_local) *n_local = c->L;
    if (n_unique) *n_unique = c->n_groups;
    if (n_shared_unique) *n_shared_unique = c->n_shared_unique;
    if (n_masked_unique) *n_masked_unique = c->n_masked_unique;
    return NKO_OK;
}

int nko_get_mult(nko_ctx *c, double *mult)
{
    if (!c || !mult) return NKO_ERR_ARG;
    memcpy(mult, c->mult, sizeof(double) * (size_t)c->L);
    return NKO_OK;
}

int nko_get_geom(nko_ctx *c, double *G6, double *J)
{
    if (!c || !G6) return NKO_ERR_ARG;
    for (int a = 0; a < 6; ++a) memcpy(G6 + a * c->L, c->G[a], sizeof(double) * (size_t)c->L);
    if (J) memcpy(J, c->J, sizeof(double) * (size_t)c->L);
    return NKO_OK;
}

int nko_get_D(nko_ctx *c, double *D, double *xi, double *w)
{
    if (!c) return NKO_ERR_ARG;
    if (D) memcpy(D, c->D, sizeof(double) * c->n * c->n);
    if (xi) memcpy(xi, c->xi, sizeof(double) * c->n);
    if (w) memcpy(w, c->wq, sizeof(double) * c->n);
    return NKO_OK;
}

/* Timing aid for bench.py's 1-thread CPU figure; no effect on any value:
 * every sum is taken over fixed chunks in a fixed order. */
void nko_set_num_threads(int nthreads)
{
#ifdef _OPENMP
    if (nthreads >= 1) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
}

int nko_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

const char *nko_strerror(int code)
{
    switch (code) {
    case NKO_OK: return "ok";
    case NKO_ERR_ARG: return "bad argument";
    case NKO_ERR_ALLOC: return "out of host memory";
    case NKO_ERR_ID: return "negative global id";
    case NKO_ERR_MASK: return "mask value not 0/1 or copies of a node disagree";
    case NKO_ERR_GEOM: return "Jacobian determinant <= 0 or non-finite";
    default: return "unknown error";
    }
}
