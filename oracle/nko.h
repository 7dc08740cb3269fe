/* nko.h -- ORACLE for the Nekbone CG hot path.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU implementation (C99 + OpenMP `parallel for` only; fp64,
 * long double for the basis and for dot-product accumulation) of what the CUDA library
 * `libnk.so` computes.  It shares no code with `paper_2606_12650_b200/` and neither imports the
 * other.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
 * `--impl reference` legs may load it.
 *
 * What it follows.  The paper (/root/reference/PAPER.md, "P:") fixes only the outline:
 *   P:225-226, P:290  3-D Poisson problem on a box of E hexahedral elements, (N+1)^3 DOFs per
 *                     element, conjugate gradients, fixed iteration count, NO preconditioner;
 *   P:314             `ax` = action of the Poisson operator (most expensive kernel);
 *   P:183-187         `gs` = gather-scatter over the copies of shared nodes;
 *   P:312             dot products of CG.
 * Everything more specific is the textbook spectral-element method as written out in
 * SURVEY.md §8(c) O1-O8 and the readings R1-R21 (listed in DESIGN.md).
 *
 * Layout: n = N+1, P = n^3, L = E*P; local index l = e*P + i + n*j + n^2*k (i<->r fastest).
 * Every pointer is a HOST pointer.  Every call returns 0 or a negative NKO_ERR_* code.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): closed-form GLL nodes/weights/D, exact
 * differentiation and quadrature degrees, closed-form G on a stretched box, analytic Jacobian of
 * a trilinear hex, rotation/scaling/axis-relabelling invariances, strong-form -Laplace identity
 * and the weak-form value 23/24 on the undeformed brick, symmetry, null space, dense Kronecker
 * assembly, brute-force multiplicities and analytic node counts, dense LU solve for CG.
 * Unpinned: nothing, except the free-running CG trajectory beyond the oracle's own rounding
 * band on config 3.
 */
#ifndef NKO_H
#define NKO_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NKO_OK          0
#define NKO_ERR_ARG    -1
#define NKO_ERR_ALLOC  -2
#define NKO_ERR_ID     -3
#define NKO_ERR_MASK   -4
#define NKO_ERR_GEOM   -5

typedef struct nko_ctx nko_ctx;

/* O1: GLL nodes xi[n], weights w[n], derivative matrix D[n*n] row-major D[i*n+m] = l_m'(xi_i). */
int nko_basis(int N, double *xi, double *w, double *D);

/* O2 + O4 + O7 set-up: geometry (G, J), node groups, multiplicity.  coords = x|y|z planes of L. */
int nko_setup(nko_ctx **ctx, int64_t E, int N, const double *coords,
              const int64_t *glo_num, const double *mask);
void nko_free(nko_ctx *ctx);

int nko_ax_e(nko_ctx *ctx, const double *u, double *w);   /* O3: w = A_L u  (u != w)        */
int nko_gs(nko_ctx *ctx, double *v);                      /* O4: v = Q Q^T v, in place       */
int nko_mask(nko_ctx *ctx, double *v);                    /* O5: v = mask o v                */
int nko_ax(nko_ctx *ctx, const double *u, double *w);     /* O6: w = mask o gs o ax_e (u)    */
int nko_dot(nko_ctx *ctx, const double *a, const double *b, double *out); /* <a,b>_c, O8     */

/* O8: unpreconditioned CG, x0 = 0, recursive residual; res_hist has niter+1 entries. */
int nko_cg(nko_ctx *ctx, const double *f, double *x, int niter, double *res_hist);
/* O8, one iteration from a given state (x, r, p updated in place; w = ax(p) returned).
 * scal[0] = rho (in); out: scal[1] = pap, scal[2] = alpha, scal[3] = rho', scal[4] = beta. */
int nko_cg_step(nko_ctx *ctx, double *x, double *r, double *p, double *w, double *scal);
/* O8 initialisation: r = mask o f, x = 0, p = r; *rho = <r,r>_c. */
int nko_cg_init(nko_ctx *ctx, const double *f, double *x, double *r, double *p, double *rho);

/* 0 (default): dot products accumulate in long double; 1: in plain double, ascending l. */
/* NEXT row f-3: Jacobi preconditioner of the original Nekbone (the paper's variant omits it).
 * diag (HOST out, L) = Q Q^T diag(A_L); nko_pcg = diagonally preconditioned CG, hist[k] = sqrt<r_k,r_k>_c. */
int nko_diag(nko_ctx *ctx, double *diag);
int nko_pcg(nko_ctx *ctx, const double *f, double *x, int niter, double *res_hist);
int nko_set_dot_mode(nko_ctx *ctx, int mode);

int nko_get_sizes(nko_ctx *ctx, int64_t *n_local, int64_t *n_unique,
                  int64_t *n_shared_unique, int64_t *n_masked_unique);
int nko_get_mult(nko_ctx *ctx, double *mult);             /* L, multiplicity = gs(1)         */
int nko_get_geom(nko_ctx *ctx, double *G6, double *J);    /* G6: rr|rs|rt|ss|st|tt planes of L; J: L (may be NULL) */
int nko_get_D(nko_ctx *ctx, double *D, double *xi, double *w);
int nko_num_threads(void);
void nko_set_num_threads(int nthreads);   /* timing aid only (bench.py's 1-thread figure) */
const char *nko_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif
