/*
 * tpt_oracle.c — plain, slow, obviously-correct CPU oracle.  TEST INFRASTRUCTURE ONLY
 * (see tpt_oracle.h for the contract, the citations and the list of pins).
 *
 * Notation follows PAPER.md (P:line): T (1-D Laplacian, Eq. 3–4), D = diag(cell widths w),
 * T~ = D^{1/2} T D^{-1/2} = Q~ Lambda Q~^T (Eq. 5), Q = D^{-1/2} Q~, Q^{-1} = Q~^T D^{1/2} (Eq. 6),
 * lambda_ij = lambda_x,i + lambda_y,j (Eq. 9).
 */
#include "tpt_oracle.h"

#include <float.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static int bc_ok(int bc) { return bc == ORC_BC_NEUMANN || bc == ORC_BC_DIRICHLET || bc == ORC_BC_PERIODIC; }

static int faces_ok(int n, const double *xf) {
    if (n < 2 || !xf) return 0;
    for (int i = 0; i <= n; ++i) if (!isfinite(xf[i])) return 0;
    for (int i = 0; i < n; ++i) if (!(xf[i + 1] > xf[i])) return 0;
    return 1;
}

/* Centre spacings delta[0..n] [A2,A3]: delta_i = x_c,i - x_c,i-1 for interior faces (the paper's
 * Delta x_{i-1/2}); boundary faces use the mirror ghost cell, delta_0 = w_0, delta_n = w_{n-1}.
 * Periodic [A17]: face 0 and face n are the same face, between cell n-1 (one period back) and cell 0:
 * delta_0 = delta_n = (w_0 + w_{n-1})/2. */
static void centre_spacings(int n, const double *xf, int bc, double *delta) {
    for (int i = 1; i < n; ++i) {
        double xc_i = 0.5 * (xf[i] + xf[i + 1]);
        double xc_im = 0.5 * (xf[i - 1] + xf[i]);
        delta[i] = xc_i - xc_im;
    }
    delta[0] = xf[1] - xf[0];
    delta[n] = xf[n] - xf[n - 1];
    if (bc == ORC_BC_PERIODIC) delta[0] = delta[n] = 0.5 * ((xf[1] - xf[0]) + (xf[n] - xf[n - 1]));
}

/* ------------------------------------------------------------------------------------------
 * 1-D operator, Eq. 3–4.  a_i = 1/(w_i delta_i) (printed); c_i = 1/(w_i delta_{i+1}),
 * b_i = -(a_i + c_i) follow from Eq. 3 [A1].  Boundary rows [A3]: homogeneous Neumann mirrors
 * phi_{-1} = phi_0 (b_0 += a_0); homogeneous Dirichlet at the boundary FACE mirrors
 * phi_{-1} = -phi_0 (b_0 -= a_0); likewise at the far end.  a_0 and c_{n-1} are then zeroed.
 * Periodic ("periodic couplings add the cyclic corner entries") [A17]: phi_{-1} = phi_{n-1},
 * phi_n = phi_0; rows 0 and n-1 are ordinary rows and a_0 (coupling to cell n-1), c_{n-1} (coupling
 * to cell 0) are KEPT as the corner entries.  Needs n >= 3 (with n = 2 the two couplings coincide).
 * ------------------------------------------------------------------------------------------ */
int orc_operator_1d(int n, const double *xf, int bc, double *w, double *a, double *b, double *c) {
    if (!faces_ok(n, xf) || !bc_ok(bc) || !w || !a || !b || !c) return ORC_EINVAL;
    if (bc == ORC_BC_PERIODIC && n < 3) return ORC_EINVAL;
    double *delta = (double *)malloc((size_t)(n + 1) * sizeof(double));
    if (!delta) return ORC_ENOMEM;
    centre_spacings(n, xf, bc, delta);
    for (int i = 0; i < n; ++i) {
        w[i] = xf[i + 1] - xf[i];
        a[i] = 1.0 / (w[i] * delta[i]);
        c[i] = 1.0 / (w[i] * delta[i + 1]);
        b[i] = -(a[i] + c[i]);
    }
    if (bc == ORC_BC_PERIODIC) {
        free(delta);
        return ORC_OK;
    }
    if (bc == ORC_BC_NEUMANN) {
        b[0] += a[0];
        b[n - 1] += c[n - 1];
    } else {
        b[0] -= a[0];
        b[n - 1] -= c[n - 1];
    }
    a[0] = 0.0;
    c[n - 1] = 0.0;
    free(delta);
    return ORC_OK;
}

/* Eq. 5: T~ = D^{1/2} T D^{-1/2}: T~_ii = b_i, T~_{i,i+1} = sqrt(w_i/w_{i+1}) c_i
 * (= sqrt(c_i a_{i+1}) by P:106's identity w_i c_i = w_{i+1} a_{i+1}). */
int orc_symmetrize_1d(int n, const double *w, const double *a, const double *b, const double *c,
                      double *diag, double *off) {
    (void)a;
    if (n < 2) return ORC_EINVAL;
    for (int i = 0; i < n; ++i) diag[i] = b[i];
    for (int i = 0; i + 1 < n; ++i) off[i] = sqrt(w[i] / w[i + 1]) * c[i];
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------------
 * Cyclic (row-ordered) two-sided Jacobi on a dense symmetric matrix A (n x n, row-major).
 * On return diag(A) holds the eigenvalues and row m of Vt the m-th eigenvector.
 * Textbook rotation: theta = (a_qq - a_pp)/(2 a_pq), t = sgn(theta)/(|theta| + sqrt(theta^2+1)).
 * ------------------------------------------------------------------------------------------ */
static int jacobi_eig(int n, double *A, double *Vt) {
    const double eps = DBL_EPSILON;
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) Vt[(size_t)i * n + j] = (i == j) ? 1.0 : 0.0;
    double fro = 0.0;
    for (size_t t = 0; t < (size_t)n * n; ++t) fro += A[t] * A[t];
    fro = sqrt(fro);
    const double tiny_abs = eps * eps * fro;
    for (int sweep = 0; sweep < 60; ++sweep) {
        long rotations = 0;
        for (int p = 0; p < n - 1; ++p) {
            double *Ap = A + (size_t)p * n;
            double *Vp = Vt + (size_t)p * n;
            for (int q = p + 1; q < n; ++q) {
                double *Aq = A + (size_t)q * n;
                double apq = Ap[q];
                if (apq == 0.0) continue;
                double app = Ap[p], aqq = Aq[q];
                if (fabs(apq) <= eps * sqrt(fabs(app * aqq)) || fabs(apq) <= tiny_abs) continue;
                double theta = (aqq - app) / (2.0 * apq);
                double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                double cs = 1.0 / sqrt(t * t + 1.0);
                double sn = t * cs;
                for (int k = 0; k < n; ++k) {
                    double x = Ap[k], y = Aq[k];
                    Ap[k] = cs * x - sn * y;
                    Aq[k] = sn * x + cs * y;
                }
                Ap[p] = app - t * apq;
                Aq[q] = aqq + t * apq;
                Ap[q] = 0.0;
                Aq[p] = 0.0;
                for (int k = 0; k < n; ++k) {          /* mirror the two rows into the two columns */
                    if (k == p || k == q) continue;
                    A[(size_t)k * n + p] = Ap[k];
                    A[(size_t)k * n + q] = Aq[k];
                }
                double *Vq = Vt + (size_t)q * n;
                for (int k = 0; k < n; ++k) {
                    double x = Vp[k], y = Vq[k];
                    Vp[k] = cs * x - sn * y;
                    Vq[k] = sn * x + cs * y;
                }
                ++rotations;
            }
        }
        if (rotations == 0) return ORC_OK;
    }
    return ORC_OK; /* not fully converged by the relative criterion; refinement follows */
}

/* ------------------------------------------------------------------------------------------
 * Factored form  -T~ = B^T B  [A9; DESIGN.md §Accuracy rule].  Rows of B, one per face carrying a
 * flux: interior face f (between cells f-1 and f): (B q)_f = (q_f/sqrt(w_f) - q_{f-1}/sqrt(w_{f-1}))/sqrt(delta_f);
 * Dirichlet boundary face: sqrt(2) q_0 / w_0 (resp. q_{n-1}/w_{n-1}); Neumann boundary face: no row;
 * periodic: one more interior row for the wrap-around face.
 * BX has nrows_B rows and n columns; X is n x n row-major, column m = vector m.
 * ------------------------------------------------------------------------------------------ */
static int apply_B(int n, const double *w, const double *delta, int bc, const double *X, double *BX) {
    int row = 0;
    if (bc == ORC_BC_PERIODIC) {   /* the wrap-around face between cell n-1 and cell 0 is an interior face */
        double sf = 1.0 / sqrt(w[0]), sm = 1.0 / sqrt(w[n - 1]), sd = 1.0 / sqrt(delta[0]);
        const double *Xm = X + (size_t)(n - 1) * n;
        for (int m = 0; m < n; ++m) BX[m] = (X[m] * sf - Xm[m] * sm) * sd;
        ++row;
    }
    if (bc == ORC_BC_DIRICHLET) {
        double s = sqrt(2.0) / w[0];
        for (int m = 0; m < n; ++m) BX[(size_t)row * n + m] = s * X[m];
        ++row;
    }
    for (int f = 1; f < n; ++f) {
        double sf = 1.0 / sqrt(w[f]), sm = 1.0 / sqrt(w[f - 1]), sd = 1.0 / sqrt(delta[f]);
        const double *Xf = X + (size_t)f * n, *Xm = X + (size_t)(f - 1) * n;
        double *o = BX + (size_t)row * n;
        for (int m = 0; m < n; ++m) o[m] = (Xf[m] * sf - Xm[m] * sm) * sd;
        ++row;
    }
    if (bc == ORC_BC_DIRICHLET) {
        double s = sqrt(2.0) / w[n - 1];
        const double *Xl = X + (size_t)(n - 1) * n;
        for (int m = 0; m < n; ++m) BX[(size_t)row * n + m] = s * Xl[m];
        ++row;
    }
    return row;
}

/* G = P^T P for a (rows x n) row-major P; G is n x n. */
static void gram(int rows, int n, const double *P, double *G) {
#pragma omp parallel for schedule(static)
    for (int i = 0; i < n; ++i) {
        double *g = G + (size_t)i * n;
        for (int j = 0; j < n; ++j) g[j] = 0.0;
        for (int r = 0; r < rows; ++r) {
            double t = P[(size_t)r * n + i];
            const double *pr = P + (size_t)r * n;
            for (int j = 0; j < n; ++j) g[j] += t * pr[j];
        }
    }
}

/* One evaluation of the Ogita–Aishima quantities for the current X:
 *   R = I - X^T X,  S~ = X^T T~ X = -(BX)^T(BX),  lambda_i = S~_ii / (1 - R_ii),
 *   E_ij = (S~_ij + lambda_j R_ij)/(lambda_j - lambda_i)  if the pair (i,j) is separated, else R_ij/2.
 * Separation test [A9]: Ogita–Aishima's normwise delta = 2(||S~-D|| + ||T~|| ||R||) presumes S~ is
 * known to eps*||T~||; in factored form S~_ij is known to ~n*eps*sqrt(|lambda_i lambda_j|), so the
 * test is made RELATIVE: separated  <=>  |lambda_i - lambda_j| > tau * max(|lambda_i|,|lambda_j|),
 * tau = 1e6 * n * eps (rounding noise in E_ij then stays below ~1e-6).  Pairs closer than that are
 * the wall-localised even/odd twins of a grid clustered at both ends; any orthonormal basis of
 * their span serves (the solution changes by < tau times their share of it).
 * Returns ||E||_F and ||R||_F.  G and Sm are n x n work arrays; E is written over G. */
static double oa_evaluate(int n, const double *w, const double *delta, int bc,
                          const double *X, double *BX, double *G, double *Sm, double *lam, double *normR) {
    int rows = apply_B(n, w, delta, bc, X, BX);
    gram(rows, n, BX, Sm);                    /* Sm = (BX)^T(BX) = -S~ */
    gram(n, n, X, G);                         /* G = X^T X */
    for (int i = 0; i < n; ++i)
        lam[i] = -Sm[(size_t)i * n + i] / G[(size_t)i * n + i];   /* S~_ii/(1-R_ii), 1-R_ii = G_ii */
    const double tau = 1e6 * n * DBL_EPSILON;
    double nE = 0.0, nR = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : nE, nR)
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) {
            double r = (i == j ? 1.0 : 0.0) - G[(size_t)i * n + j];
            double s = -Sm[(size_t)i * n + j];
            double big = fabs(lam[i]) > fabs(lam[j]) ? fabs(lam[i]) : fabs(lam[j]);
            double e;
            if (i != j && fabs(lam[i] - lam[j]) > tau * big) e = (s + lam[j] * r) / (lam[j] - lam[i]);
            else e = 0.5 * r;
            G[(size_t)i * n + j] = e;
            nE += e * e;
            nR += r * r;
        }
    *normR = sqrt(nR);
    return sqrt(nE);
}

/* X <- X + X E  (n x n, row-major). */
static void oa_update(int n, const double *X, const double *E, double *Xnew) {
#pragma omp parallel for schedule(static)
    for (int r = 0; r < n; ++r) {
        const double *x = X + (size_t)r * n;
        double *o = Xnew + (size_t)r * n;
        for (int j = 0; j < n; ++j) o[j] = x[j];
        for (int i = 0; i < n; ++i) {
            double t = x[i];
            const double *e = E + (size_t)i * n;
            for (int j = 0; j < n; ++j) o[j] += t * e[j];
        }
    }
}

typedef struct { double lam; int idx; } lam_idx;
static int cmp_desc(const void *a, const void *b) {
    double x = ((const lam_idx *)a)->lam, y = ((const lam_idx *)b)->lam;
    return (x < y) - (x > y);
}

int orc_eig_1d(int n, const double *xf, int bc, int refine_steps, double *lambda, double *qtilde) {
    if (!faces_ok(n, xf) || !bc_ok(bc) || !lambda || !qtilde || refine_steps < 0) return ORC_EINVAL;
    size_t nn = (size_t)n * n;
    double *w = malloc(sizeof(double) * n), *a = malloc(sizeof(double) * n);
    double *b = malloc(sizeof(double) * n), *c = malloc(sizeof(double) * n);
    double *dg = malloc(sizeof(double) * n), *of = malloc(sizeof(double) * n);
    double *delta = malloc(sizeof(double) * (n + 1));
    double *A = malloc(sizeof(double) * nn), *Vt = malloc(sizeof(double) * nn);
    double *X = malloc(sizeof(double) * nn), *Xn = malloc(sizeof(double) * nn);
    double *G = malloc(sizeof(double) * nn), *Sm = malloc(sizeof(double) * nn);
    double *BX = malloc(sizeof(double) * (size_t)(n + 1) * n);
    double *lam = malloc(sizeof(double) * n), *lamprev = malloc(sizeof(double) * n);
    lam_idx *order = malloc(sizeof(lam_idx) * n);
    int rc = ORC_OK;
    if (!w || !a || !b || !c || !dg || !of || !delta || !A || !Vt || !X || !Xn || !G || !Sm || !BX || !lam ||
        !lamprev || !order) { rc = ORC_ENOMEM; goto done; }

    orc_operator_1d(n, xf, bc, w, a, b, c);
    orc_symmetrize_1d(n, w, a, b, c, dg, of);
    centre_spacings(n, xf, bc, delta);

    /* 1.2: T~ = Q~ Lambda Q~^T — base solver: cyclic Jacobi on the dense form of T~. */
    memset(A, 0, sizeof(double) * nn);
    for (int i = 0; i < n; ++i) A[(size_t)i * n + i] = dg[i];
    for (int i = 0; i + 1 < n; ++i) {
        A[(size_t)i * n + i + 1] = of[i];
        A[(size_t)(i + 1) * n + i] = of[i];
    }
    if (bc == ORC_BC_PERIODIC) {   /* cyclic corners ("symmetric cyclic operator, stored as a dense matrix") */
        double corner = sqrt(w[n - 1] / w[0]) * c[n - 1];      /* = sqrt(c_{n-1} a_0) */
        A[(size_t)(n - 1) * n] = corner;
        A[n - 1] = corner;
    }
    jacobi_eig(n, A, Vt);
    for (int i = 0; i < n; ++i)
        for (int m = 0; m < n; ++m) X[(size_t)i * n + m] = Vt[(size_t)m * n + i];
    for (int m = 0; m < n; ++m) lam[m] = A[(size_t)m * n + m];

    /* Guarded Ogita–Aishima refinement in factored form [A9]: `refine_steps` updates X <- X + XE;
     * an update is undone (and refinement stops) if it made the orthogonality defect ||R||_F worse
     * while that defect is above rounding level.  The eigenvalues returned are the factored-form
     * Rayleigh quotients of the final X. */
    if (refine_steps > 0) {
        double prevR = HUGE_VAL;
        for (int step = 0;; ++step) {
            double nR;
            (void)oa_evaluate(n, w, delta, bc, X, BX, G, Sm, lam, &nR);
            if (step > 0 && !(nR <= prevR || nR <= 1e-12 * n)) {      /* worse (or NaN): revert */
                memcpy(X, Xn, sizeof(double) * nn);
                memcpy(lam, lamprev, sizeof(double) * n);
                break;
            }
            if (step == refine_steps) break;
            memcpy(lamprev, lam, sizeof(double) * n);
            oa_update(n, X, G, Vt);              /* Vt is scratch for the new X */
            memcpy(Xn, X, sizeof(double) * nn);  /* Xn keeps the previous X for a possible revert */
            memcpy(X, Vt, sizeof(double) * nn);
            prevR = nR;
        }
    }

    /* Order: descending lambda so that mode 0 is the smoothest [A6]. */
    for (int m = 0; m < n; ++m) { order[m].lam = lam[m]; order[m].idx = m; }
    qsort(order, n, sizeof(lam_idx), cmp_desc);
    for (int m = 0; m < n; ++m) {
        int src = order[m].idx;
        lambda[m] = order[m].lam;
        double nrm = 0.0;
        for (int i = 0; i < n; ++i) nrm += X[(size_t)i * n + src] * X[(size_t)i * n + src];
        nrm = sqrt(nrm);
        for (int i = 0; i < n; ++i) qtilde[(size_t)i * n + m] = X[(size_t)i * n + src] / nrm;
    }
    /* Neumann–Neumann: the null pair is known exactly: lambda = 0, q~_i = sqrt(w_i/L)
     * (T 1 = 0  =>  T~ D^{1/2} 1 = 0). */
    if (bc == ORC_BC_NEUMANN || bc == ORC_BC_PERIODIC) {
        double L = 0.0;
        for (int i = 0; i < n; ++i) L += w[i];
        lambda[0] = 0.0;
        for (int i = 0; i < n; ++i) qtilde[(size_t)i * n + 0] = sqrt(w[i] / L);
    }
    /* Sign convention [A6]: sum_i q~_i sqrt(w_i) >= 0; if that sum vanishes (odd modes of a
     * symmetric grid) the first entry of non-negligible size is made positive. */
    {
        double L = 0.0;
        for (int i = 0; i < n; ++i) L += w[i];
        for (int m = 0; m < n; ++m) {
            double s = 0.0;
            for (int i = 0; i < n; ++i) s += qtilde[(size_t)i * n + m] * sqrt(w[i]);
            int flip = 0;
            if (fabs(s) > 1e-8 * sqrt(L)) flip = s < 0.0;
            else
                for (int i = 0; i < n; ++i)
                    if (fabs(qtilde[(size_t)i * n + m]) > 1e-8) { flip = qtilde[(size_t)i * n + m] < 0.0; break; }
            if (flip) for (int i = 0; i < n; ++i) qtilde[(size_t)i * n + m] = -qtilde[(size_t)i * n + m];
        }
    }
done:
    free(w); free(a); free(b); free(c); free(dg); free(of); free(delta); free(A); free(Vt); free(X); free(Xn);
    free(G); free(Sm); free(BX); free(lam); free(lamprev); free(order);
    return rc;
}

/* ------------------------------------------------------------------------------------------ */
struct orc_plan {
    int nx, ny, nz;
    int bc[3];
    double alpha;
    int singular;
    int dirs;              /* implicitly treated directions of L_I: bit 0 = x, 1 = y, 2 = z; 7 = the full operator */
    double *wx, *wy, *wz;
    double *az, *bz, *cz;
    double *lamx, *lamy;
    double *qx, *qy;       /* Q~ row-major: q[i*n+m] */
    double *qxt, *qyt;     /* transposes: qt[m*n+i] */
};

void orc_plan_destroy(orc_plan *p) {
    if (!p) return;
    free(p->wx); free(p->wy); free(p->wz); free(p->az); free(p->bz); free(p->cz);
    free(p->lamx); free(p->lamy); free(p->qx); free(p->qy); free(p->qxt); free(p->qyt);
    free(p);
}

static double *dup_array(const double *src, size_t count) {
    double *d = (double *)malloc(sizeof(double) * count);
    if (d && src) memcpy(d, src, sizeof(double) * count);
    return d;
}

int orc_plan_create_with_eig(orc_plan **out, int nx, int ny, int nz,
                             const double *xf, const double *yf, const double *zf,
                             const int bc[3], double alpha,
                             const double *lamx, const double *qx, const double *lamy, const double *qy) {
    if (!out || !bc || !faces_ok(nx, xf) || !faces_ok(ny, yf) || !faces_ok(nz, zf)) return ORC_EINVAL;
    if (!bc_ok(bc[0]) || !bc_ok(bc[1]) || !bc_ok(bc[2]) || !(alpha >= 0.0) || !isfinite(alpha)) return ORC_EINVAL;
    /* periodic x, y are diagonalised; a periodic z makes the sweep a CYCLIC tridiagonal solve ("cyclic corner entries") [A19] */
    if ((bc[2] == ORC_BC_PERIODIC && nz < 3) || (bc[0] == ORC_BC_PERIODIC && nx < 3) || (bc[1] == ORC_BC_PERIODIC && ny < 3)) return ORC_EINVAL;
    if (!lamx || !qx || !lamy || !qy) return ORC_EINVAL;
    orc_plan *p = (orc_plan *)calloc(1, sizeof(orc_plan));
    if (!p) return ORC_ENOMEM;
    p->nx = nx; p->ny = ny; p->nz = nz; p->alpha = alpha;
    p->dirs = ORC_DIRS_XYZ;
    p->bc[0] = bc[0]; p->bc[1] = bc[1]; p->bc[2] = bc[2];
    /* [A7] structural detection of the null mode: no Dirichlet direction and Poisson. */
    p->singular = (alpha == 0.0 && bc[0] != ORC_BC_DIRICHLET && bc[1] != ORC_BC_DIRICHLET && bc[2] != ORC_BC_DIRICHLET);
    p->wx = dup_array(NULL, nx); p->wy = dup_array(NULL, ny); p->wz = dup_array(NULL, nz);
    p->az = dup_array(NULL, nz); p->bz = dup_array(NULL, nz); p->cz = dup_array(NULL, nz);
    p->lamx = dup_array(lamx, nx); p->lamy = dup_array(lamy, ny);
    p->qx = dup_array(qx, (size_t)nx * nx); p->qy = dup_array(qy, (size_t)ny * ny);
    p->qxt = dup_array(NULL, (size_t)nx * nx); p->qyt = dup_array(NULL, (size_t)ny * ny);
    double *tmp = dup_array(NULL, (size_t)(nx > ny ? nx : ny) * 3);
    if (!p->wx || !p->wy || !p->wz || !p->az || !p->bz || !p->cz || !p->lamx || !p->lamy || !p->qx || !p->qy ||
        !p->qxt || !p->qyt || !tmp) { free(tmp); orc_plan_destroy(p); return ORC_ENOMEM; }
    int m = nx > ny ? nx : ny;
    orc_operator_1d(nx, xf, bc[0], p->wx, tmp, tmp + m, tmp + 2 * m);
    orc_operator_1d(ny, yf, bc[1], p->wy, tmp, tmp + m, tmp + 2 * m);
    orc_operator_1d(nz, zf, bc[2], p->wz, p->az, p->bz, p->cz);
    free(tmp);
    for (int i = 0; i < nx; ++i) for (int k = 0; k < nx; ++k) p->qxt[(size_t)k * nx + i] = p->qx[(size_t)i * nx + k];
    for (int i = 0; i < ny; ++i) for (int k = 0; k < ny; ++k) p->qyt[(size_t)k * ny + i] = p->qy[(size_t)i * ny + k];
    *out = p;
    return ORC_OK;
}

int orc_plan_create(orc_plan **out, int nx, int ny, int nz,
                    const double *xf, const double *yf, const double *zf, const int bc[3], double alpha) {
    if (!out || !bc || !faces_ok(nx, xf) || !faces_ok(ny, yf) || !faces_ok(nz, zf)) return ORC_EINVAL;
    if (!bc_ok(bc[0]) || !bc_ok(bc[1]) || !bc_ok(bc[2])) return ORC_EINVAL;
    double *lamx = dup_array(NULL, nx), *lamy = dup_array(NULL, ny);
    double *qx = dup_array(NULL, (size_t)nx * nx), *qy = dup_array(NULL, (size_t)ny * ny);
    int rc = ORC_ENOMEM;
    if (lamx && lamy && qx && qy) {
        rc = orc_eig_1d(nx, xf, bc[0], 2, lamx, qx);
        if (rc == ORC_OK) rc = orc_eig_1d(ny, yf, bc[1], 2, lamy, qy);
        if (rc == ORC_OK) rc = orc_plan_create_with_eig(out, nx, ny, nz, xf, yf, zf, bc, alpha, lamx, qx, lamy, qy);
    }
    free(lamx); free(lamy); free(qx); free(qy);
    return rc;
}

int orc_plan_is_singular(const orc_plan *p) { return p ? p->singular : ORC_EINVAL; }

/* L_I = L_z ("z"), L_y + L_z ("yz") or L ("xyz").  The partial choices exist for the Helmholtz
 * problem of Eq. 2b only (the pressure Poisson equation always carries the full Laplacian, Eq. 2c). */
int orc_plan_set_implicit_dirs(orc_plan *p, int dirs) {
    if (!p || (dirs != ORC_DIRS_XYZ && dirs != ORC_DIRS_YZ && dirs != ORC_DIRS_Z)) return ORC_EINVAL;
    if (dirs != ORC_DIRS_XYZ && !(p->alpha > 0.0)) return ORC_EINVAL;
    p->dirs = dirs;
    return ORC_OK;
}

int orc_plan_get_eigen(const orc_plan *p, int dir, double *lambda, double *qtilde) {
    if (!p || (dir != 0 && dir != 1)) return ORC_EINVAL;
    int n = dir == 0 ? p->nx : p->ny;
    if (lambda) memcpy(lambda, dir == 0 ? p->lamx : p->lamy, sizeof(double) * n);
    if (qtilde) memcpy(qtilde, dir == 0 ? p->qx : p->qy, sizeof(double) * (size_t)n * n);
    return ORC_OK;
}

/* Step 2.1 (Eq. 10a): f^(x) = (Qx^{-1} (x) I (x) I) f with Qx^{-1} = Q~x^T Dx^{1/2} (Eq. 6):
 * out[k,j,m] = sum_i Q~x[i,m] sqrt(wx_i) in[k,j,i]. */
void orc_forward_x(const orc_plan *p, const double *in, double *out) {
    const int nx = p->nx;
    const long lines = (long)p->ny * p->nz;
#pragma omp parallel for schedule(static)
    for (long r = 0; r < lines; ++r) {
        const double *f = in + (size_t)r * nx;
        double *o = out + (size_t)r * nx;
        for (int m = 0; m < nx; ++m) o[m] = 0.0;
        for (int i = 0; i < nx; ++i) {
            double g = sqrt(p->wx[i]) * f[i];
            const double *q = p->qx + (size_t)i * nx;
            for (int m = 0; m < nx; ++m) o[m] += q[m] * g;
        }
    }
}

/* Step 2.2 (Eq. 10b): out[k,m,i] = sum_j Q~y[j,m] sqrt(wy_j) in[k,j,i]. */
void orc_forward_y(const orc_plan *p, const double *in, double *out) {
    const int nx = p->nx, ny = p->ny;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < p->nz; ++k) {
        const double *fk = in + (size_t)k * nx * ny;
        double *ok = out + (size_t)k * nx * ny;
        for (int m = 0; m < ny; ++m) {
            double *o = ok + (size_t)m * nx;
            for (int i = 0; i < nx; ++i) o[i] = 0.0;
            for (int j = 0; j < ny; ++j) {
                double t = p->qy[(size_t)j * ny + m] * sqrt(p->wy[j]);
                const double *f = fk + (size_t)j * nx;
                for (int i = 0; i < nx; ++i) o[i] += t * f[i];
            }
        }
    }
}

/* Step 2.4 (Eq. 12a): Qy = Dy^{-1/2} Q~y: out[k,j,i] = wy_j^{-1/2} sum_m Q~y[j,m] in[k,m,i]. */
void orc_inverse_y(const orc_plan *p, const double *in, double *out) {
    const int nx = p->nx, ny = p->ny;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < p->nz; ++k) {
        const double *fk = in + (size_t)k * nx * ny;
        double *ok = out + (size_t)k * nx * ny;
        for (int j = 0; j < ny; ++j) {
            double *o = ok + (size_t)j * nx;
            for (int i = 0; i < nx; ++i) o[i] = 0.0;
            for (int m = 0; m < ny; ++m) {
                double t = p->qy[(size_t)j * ny + m];
                const double *f = fk + (size_t)m * nx;
                for (int i = 0; i < nx; ++i) o[i] += t * f[i];
            }
            double s = 1.0 / sqrt(p->wy[j]);
            for (int i = 0; i < nx; ++i) o[i] *= s;
        }
    }
}

/* Step 2.5 (Eq. 12b): out[k,j,i] = wx_i^{-1/2} sum_m Q~x[i,m] in[k,j,m]. */
void orc_inverse_x(const orc_plan *p, const double *in, double *out) {
    const int nx = p->nx;
    const long lines = (long)p->ny * p->nz;
#pragma omp parallel for schedule(static)
    for (long r = 0; r < lines; ++r) {
        const double *f = in + (size_t)r * nx;
        double *o = out + (size_t)r * nx;
        for (int i = 0; i < nx; ++i) o[i] = 0.0;
        for (int m = 0; m < nx; ++m) {
            double g = f[m];
            const double *q = p->qxt + (size_t)m * nx;   /* q[i] = Q~x[i,m] */
            for (int i = 0; i < nx; ++i) o[i] += q[i] * g;
        }
        for (int i = 0; i < nx; ++i) o[i] *= 1.0 / sqrt(p->wx[i]);
    }
}

/* Step 2.3: for every (my,mx), sigma = lambda_x[mx] + lambda_y[my] (Eq. 9):
 *   Poisson   (T_z + sigma I) x = p          [A4]
 *   Helmholtz ((1 - alpha sigma) I - alpha T_z) x = p    [A5]
 * Textbook Thomas without pivoting, one column at a time (the i loop below only walks nx
 * independent columns side by side so that memory is read along x).
 * Singular plan, column (0,0): the final pivot vanishes -> last unknown := 0, then the
 * Delta z-weighted mean of that column is removed (zero volume-weighted mean gauge) [A7]. */
/* Textbook Thomas for one tridiagonal system of size n (sub[0], sup[n-1] unused), in place on d; cp = scratch. */
static void thomas_line(int n, const double *sub, const double *dia, const double *sup, double *d, double *cp) {
    double den = dia[0];
    cp[0] = sup[0] / den;
    d[0] = d[0] / den;
    for (int k = 1; k < n; ++k) {
        den = dia[k] - sub[k] * cp[k - 1];
        cp[k] = sup[k] / den;
        d[k] = (d[k] - sub[k] * d[k - 1]) / den;
    }
    for (int k = n - 2; k >= 0; --k) d[k] -= cp[k] * d[k + 1];
}

/* Periodic z [A19]: row 0 couples to x_{n-1} through sub[0], row n-1 to x_0 through sup[n-1] ("cyclic corner
 * entries").  The paper does not say how it sweeps such a system; the textbook way is taken: the cyclic matrix is a
 * tridiagonal matrix A' plus a rank-one term u v^T (u = (g, 0, .., 0, sup[n-1]), v = (1, 0, .., 0, sub[0]/g), g = -dia[0];
 * A' = A with dia[0] - g and dia[n-1] - sup[n-1] sub[0] / g), so by the Sherman-Morrison formula
 *     x = y - q (v.y) / (1 + v.q),   A' y = d,  A' q = u.
 * Null column of a singular plan: the cyclic T_z is singular (constant null vector); following P:219 the last unknown
 * is set to 0 — which removes both corner couplings — the remaining n-1 equations are a plain tridiagonal system, and
 * the Delta z-weighted mean of the column is removed afterwards [A7]. */
static int thomas_z_cyclic(const orc_plan *p, double *field) {
    const int nx = p->nx, ny = p->ny, nz = p->nz;
    const double alpha = p->alpha;
    const size_t plane = (size_t)nx * ny;
    int status = ORC_OK;
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * 7 * (size_t)nz);
        if (!buf) {
#pragma omp critical
            status = ORC_ENOMEM;
        }
        double *sub = buf, *dia = buf + nz, *sup = buf + 2 * nz, *y = buf + 3 * nz, *q = buf + 4 * nz, *cp = buf + 5 * nz, *bb = buf + 6 * nz;
        for (int k = 0; buf && k < nz; ++k) {
            if (alpha == 0.0) { sub[k] = p->az[k]; dia[k] = p->bz[k]; sup[k] = p->cz[k]; }
            else { sub[k] = -alpha * p->az[k]; dia[k] = 1.0 - alpha * p->bz[k]; sup[k] = -alpha * p->cz[k]; }
        }
#pragma omp for schedule(static) collapse(2)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                if (!buf) continue;
                double *col = field + (size_t)j * nx + i;
                double sigma = ((p->dirs & 1) ? p->lamx[i] : 0.0) + ((p->dirs & 2) ? p->lamy[j] : 0.0);
                double shift = (alpha == 0.0) ? sigma : -alpha * sigma;
                for (int k = 0; k < nz; ++k) { y[k] = col[k * plane]; bb[k] = dia[k] + shift; }
                if (p->singular && i == 0 && j == 0) {
                    thomas_line(nz - 1, sub, bb, sup, y, cp);
                    y[nz - 1] = 0.0;
                    double s = 0.0, L = 0.0;
                    for (int k = 0; k < nz; ++k) { s += p->wz[k] * y[k]; L += p->wz[k]; }
                    for (int k = 0; k < nz; ++k) col[k * plane] = y[k] - s / L;
                    continue;
                }
                const double g = -bb[0];
                bb[0] -= g;
                bb[nz - 1] -= sup[nz - 1] * sub[0] / g;
                for (int k = 0; k < nz; ++k) q[k] = 0.0;
                q[0] = g;
                q[nz - 1] = sup[nz - 1];
                thomas_line(nz, sub, bb, sup, y, cp);
                thomas_line(nz, sub, bb, sup, q, cp);
                const double fact = (y[0] + sub[0] * y[nz - 1] / g) / (1.0 + q[0] + sub[0] * q[nz - 1] / g);
                for (int k = 0; k < nz; ++k) col[k * plane] = y[k] - fact * q[k];
            }
        free(buf);
    }
    return status;
}

int orc_thomas_z(const orc_plan *p, double *field) {
    if (p->bc[2] == ORC_BC_PERIODIC) return thomas_z_cyclic(p, field);
    const int nx = p->nx, ny = p->ny, nz = p->nz;
    const double alpha = p->alpha;
    const size_t plane = (size_t)nx * ny;
    int status = ORC_OK;
    double bscale = 0.0;
    for (int k = 0; k < nz; ++k) if (fabs(p->bz[k]) > bscale) bscale = fabs(p->bz[k]);
#pragma omp parallel
    {
        double *cp = (double *)malloc(sizeof(double) * (size_t)nz * nx);
        double *low = (double *)malloc(sizeof(double) * 3 * (size_t)nz);   /* sub, diag0, sup per k */
        const int ok = cp && low;
        if (!ok) {
#pragma omp critical
            status = ORC_ENOMEM;
        }
        {
            double *sub = low, *dia = low + nz, *sup = low + 2 * nz;
            for (int k = 0; ok && k < nz; ++k) {
                if (alpha == 0.0) { sub[k] = p->az[k]; dia[k] = p->bz[k]; sup[k] = p->cz[k]; }
                else { sub[k] = -alpha * p->az[k]; dia[k] = 1.0 - alpha * p->bz[k]; sup[k] = -alpha * p->cz[k]; }
            }
#pragma omp for schedule(static)
            for (int j = 0; j < ny; ++j) {
                if (!ok) continue;
                double *d = field + (size_t)j * nx;           /* d[k*plane + i] */
                for (int i = 0; i < nx; ++i) {
                    /* Eq. 9 restricted to the diagonalised directions ("the yz option omits the x
                     * transforms, and the z option performs only the tridiagonal solve") */
                    double sigma = ((p->dirs & 1) ? p->lamx[i] : 0.0) + ((p->dirs & 2) ? p->lamy[j] : 0.0);
                    double shift = (alpha == 0.0) ? sigma : -alpha * sigma;
                    int null_col = p->singular && i == 0 && j == 0;
                    /* forward elimination */
                    double den = dia[0] + shift;
                    cp[i] = sup[0] / den;
                    d[i] = d[i] / den;
                    for (int k = 1; k < nz; ++k) {
                        den = (dia[k] + shift) - sub[k] * cp[(size_t)(k - 1) * nx + i];
                        if (k == nz - 1 && null_col) {
                            /* paper's rule kept as an assertion: |final pivot| <= 1e-10 * scale */
                            if (!(fabs(den) <= 1e-10 * bscale)) {
#pragma omp critical
                                status = ORC_ENUMERIC;
                            }
                            d[k * plane + i] = 0.0;
                            cp[(size_t)k * nx + i] = 0.0;
                        } else {
                            if (k == nz - 1 && !(fabs(den) > 1e-10 * bscale) && alpha == 0.0) {
#pragma omp critical
                                status = ORC_ENUMERIC;
                            }
                            cp[(size_t)k * nx + i] = sup[k] / den;
                            d[k * plane + i] = (d[k * plane + i] - sub[k] * d[(k - 1) * plane + i]) / den;
                        }
                    }
                    /* back substitution */
                    for (int k = nz - 2; k >= 0; --k)
                        d[k * plane + i] -= cp[(size_t)k * nx + i] * d[(k + 1) * plane + i];
                    if (null_col) {
                        double s = 0.0, L = 0.0;
                        for (int k = 0; k < nz; ++k) { s += p->wz[k] * d[k * plane + i]; L += p->wz[k]; }
                        double mean = s / L;
                        for (int k = 0; k < nz; ++k) d[k * plane + i] -= mean;
                    }
                }
            }
        }
        free(cp);
        free(low);
    }
    return status;
}

int orc_solve(const orc_plan *p, const double *f, double *phi, double *work) {
    if (!p || !f || !phi || !work || f == phi) return ORC_EINVAL;
    const size_t bytes = sizeof(double) * (size_t)p->nx * p->ny * p->nz;
    if (p->dirs & 1) orc_forward_x(p, f, work); else memcpy(work, f, bytes);       /* 2.1 */
    if (p->dirs & 2) orc_forward_y(p, work, phi); else memcpy(phi, work, bytes);   /* 2.2 */
    int rc = orc_thomas_z(p, phi);                                                 /* 2.3 */
    if (p->dirs & 2) orc_inverse_y(p, phi, work); else memcpy(work, phi, bytes);   /* 2.4 */
    if (p->dirs & 1) orc_inverse_x(p, work, phi); else memcpy(phi, work, bytes);   /* 2.5 */
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * Independent definitions: Eq. 3 evaluated as a difference of face fluxes.
 * Ghost values [A3]: Neumann phi_ghost = phi_boundary-cell (zero flux); Dirichlet phi_ghost = -phi.
 * ------------------------------------------------------------------------------------------ */
static double lap1d_flux(const double *xf, int n, int bc, int i, double um, double u0, double up) {
    /* um/up are neighbours (periodic: the wrapped ones) or ignored at a Neumann/Dirichlet boundary */
    double w = xf[i + 1] - xf[i];
    double fl, fr;
    if (bc == ORC_BC_PERIODIC && (i == 0 || i == n - 1)) {
        double dwrap = 0.5 * ((xf[1] - xf[0]) + (xf[n] - xf[n - 1]));
        double dl = i == 0 ? dwrap : 0.5 * (xf[i] + xf[i + 1]) - 0.5 * (xf[i - 1] + xf[i]);
        double dr = i == n - 1 ? dwrap : 0.5 * (xf[i + 1] + xf[i + 2]) - 0.5 * (xf[i] + xf[i + 1]);
        return ((up - u0) / dr - (u0 - um) / dl) / w;
    }
    if (i > 0) {
        double dl = 0.5 * (xf[i] + xf[i + 1]) - 0.5 * (xf[i - 1] + xf[i]);
        fl = (u0 - um) / dl;
    } else fl = (bc == ORC_BC_NEUMANN) ? 0.0 : (u0 - (-u0)) / w;
    if (i < n - 1) {
        double dr = 0.5 * (xf[i + 1] + xf[i + 2]) - 0.5 * (xf[i] + xf[i + 1]);
        fr = (up - u0) / dr;
    } else fr = (bc == ORC_BC_NEUMANN) ? 0.0 : ((-u0) - u0) / w;
    return (fr - fl) / w;
}

int orc_apply_operator_flux(int nx, int ny, int nz, const double *xf, const double *yf, const double *zf,
                            const int bc[3], double alpha, const double *phi, double *out) {
    return orc_apply_operator_flux_dirs(nx, ny, nz, xf, yf, zf, bc, alpha, ORC_DIRS_XYZ, phi, out);
}

static int dirs_ok(int dirs, double alpha) {
    if (dirs == ORC_DIRS_XYZ) return 1;
    return (dirs == ORC_DIRS_YZ || dirs == ORC_DIRS_Z) && alpha > 0.0;
}

/* (I - alpha L_I) phi with L_I the sum of the 1-D Laplacians of the directions in `dirs`. */
int orc_apply_operator_flux_dirs(int nx, int ny, int nz, const double *xf, const double *yf, const double *zf,
                                 const int bc[3], double alpha, int dirs, const double *phi, double *out) {
    if (!dirs_ok(dirs, alpha)) return ORC_EINVAL;
    if (!faces_ok(nx, xf) || !faces_ok(ny, yf) || !faces_ok(nz, zf) || !bc || !phi || !out) return ORC_EINVAL;
    const size_t plane = (size_t)nx * ny;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t id = i + (size_t)nx * j + plane * k;
                double u0 = phi[id];
                const int px = bc[0] == ORC_BC_PERIODIC, py = bc[1] == ORC_BC_PERIODIC, pz = bc[2] == ORC_BC_PERIODIC;
                double lx = lap1d_flux(xf, nx, bc[0], i, i > 0 ? phi[id - 1] : (px ? phi[id + (nx - 1)] : 0.0), u0,
                                       i < nx - 1 ? phi[id + 1] : (px ? phi[id - (nx - 1)] : 0.0));
                double ly = lap1d_flux(yf, ny, bc[1], j, j > 0 ? phi[id - nx] : (py ? phi[id + (size_t)nx * (ny - 1)] : 0.0), u0,
                                       j < ny - 1 ? phi[id + nx] : (py ? phi[id - (size_t)nx * (ny - 1)] : 0.0));
                double lz = lap1d_flux(zf, nz, bc[2], k, k > 0 ? phi[id - plane] : (pz ? phi[id + plane * (nz - 1)] : 0.0), u0,
                                       k < nz - 1 ? phi[id + plane] : (pz ? phi[id - plane * (nz - 1)] : 0.0));
                double lap = ((dirs & 1) ? lx : 0.0) + ((dirs & 2) ? ly : 0.0) + lz;
                out[id] = (alpha == 0.0) ? lap : u0 - alpha * lap;
            }
    return ORC_OK;
}

int orc_residual_norms(int nx, int ny, int nz, const double *xf, const double *yf, const double *zf,
                       const int bc[3], double alpha, const double *f, const double *phi, double norms[4]) {
    return orc_residual_norms_dirs(nx, ny, nz, xf, yf, zf, bc, alpha, ORC_DIRS_XYZ, f, phi, norms);
}

int orc_residual_norms_dirs(int nx, int ny, int nz, const double *xf, const double *yf, const double *zf,
                            const int bc[3], double alpha, int dirs, const double *f, const double *phi,
                            double norms[4]) {
    if (!f || !norms) return ORC_EINVAL;
    size_t n = (size_t)nx * ny * nz;
    double *op = (double *)malloc(sizeof(double) * n);
    if (!op) return ORC_ENOMEM;
    int rc = orc_apply_operator_flux_dirs(nx, ny, nz, xf, yf, zf, bc, alpha, dirs, phi, op);
    if (rc != ORC_OK) { free(op); return rc; }
    double r2 = 0, f2 = 0, rv = 0, fv = 0, rmax = 0, fmax = 0, pmax = 0;
    const size_t plane = (size_t)nx * ny;
#pragma omp parallel for schedule(static) reduction(+ : r2, f2, rv, fv) reduction(max : rmax, fmax, pmax)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t id = i + (size_t)nx * j + plane * k;
                double V = (xf[i + 1] - xf[i]) * (yf[j + 1] - yf[j]) * (zf[k + 1] - zf[k]);
                double r = f[id] - op[id];
                r2 += r * r; f2 += f[id] * f[id];
                rv += V * r * r; fv += V * f[id] * f[id];
                if (fabs(r) > rmax) rmax = fabs(r);
                if (fabs(f[id]) > fmax) fmax = fabs(f[id]);
                if (fabs(phi[id]) > pmax) pmax = fabs(phi[id]);
            }
    free(op);
    /* ||Op||_inf <= sum over directions of max row sum = 4/(w delta)_max-ish; use the exact
     * bound from the coefficients: max_i (|a|+|b|+|c|) per direction. */
    double opn = 0.0;
    const double *ff[3] = {xf, yf, zf};
    int nn[3] = {nx, ny, nz};
    for (int d = 0; d < 3; ++d) {
        if (!(dirs & (1 << d))) continue;
        int m = nn[d];
        double *w = malloc(sizeof(double) * m), *a = malloc(sizeof(double) * m), *b = malloc(sizeof(double) * m),
               *c = malloc(sizeof(double) * m);
        if (!w || !a || !b || !c) { free(w); free(a); free(b); free(c); return ORC_ENOMEM; }
        orc_operator_1d(m, ff[d], bc[d], w, a, b, c);
        double mx = 0.0;
        for (int i = 0; i < m; ++i) { double s = fabs(a[i]) + fabs(b[i]) + fabs(c[i]); if (s > mx) mx = s; }
        opn += mx;
        free(w); free(a); free(b); free(c);
    }
    if (alpha != 0.0) opn = 1.0 + alpha * opn;
    norms[0] = sqrt(r2) / sqrt(f2);
    norms[1] = sqrt(rv) / sqrt(fv);
    norms[2] = rmax / fmax;
    norms[3] = rmax / (opn * pmax + fmax);
    return ORC_OK;
}

/* Brute force (pin): dense assembly of Eq. 7 from the 1-D coefficients, Gaussian elimination with
 * partial pivoting. */
int orc_dense_solve_3d(int nx, int ny, int nz, const double *xf, const double *yf, const double *zf,
                       const int bc[3], double alpha, const double *f, double *phi) {
    return orc_dense_solve_3d_dirs(nx, ny, nz, xf, yf, zf, bc, alpha, ORC_DIRS_XYZ, f, phi);
}

int orc_dense_solve_3d_dirs(int nx, int ny, int nz, const double *xf, const double *yf, const double *zf,
                            const int bc[3], double alpha, int dirs, const double *f, double *phi) {
    if (!dirs_ok(dirs, alpha)) return ORC_EINVAL;
    if (!faces_ok(nx, xf) || !faces_ok(ny, yf) || !faces_ok(nz, zf) || !bc || !f || !phi) return ORC_EINVAL;
    long n = (long)nx * ny * nz;
    if (n > 4096) return ORC_EINVAL;
    int singular = (alpha == 0.0 && bc[0] != ORC_BC_DIRICHLET && bc[1] != ORC_BC_DIRICHLET && bc[2] != ORC_BC_DIRICHLET);
    long N = n + (singular ? 1 : 0);
    double *M = (double *)calloc((size_t)N * (N + 1), sizeof(double));   /* augmented [M | rhs] */
    double *co[3][4];
    int nn[3] = {nx, ny, nz};
    const double *ff[3] = {xf, yf, zf};
    for (int d = 0; d < 3; ++d) for (int t = 0; t < 4; ++t) co[d][t] = (double *)malloc(sizeof(double) * nn[d]);
    for (int d = 0; d < 3; ++d) orc_operator_1d(nn[d], ff[d], bc[d], co[d][0], co[d][1], co[d][2], co[d][3]);
    const long W = N + 1;
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                long r = i + (long)nx * (j + (long)ny * k);
                double *row = M + r * W;
                int id[3] = {i, j, k};
                long st[3] = {1, nx, (long)nx * ny};
                for (int d = 0; d < 3; ++d) {
                    if (!(dirs & (1 << d))) continue;
                    int q = id[d];
                    row[r] += co[d][2][q];
                    if (q > 0) row[r - st[d]] += co[d][1][q];
                    else if (bc[d] == ORC_BC_PERIODIC) row[r + st[d] * (nn[d] - 1)] += co[d][1][q];   /* cyclic corner */
                    if (q < nn[d] - 1) row[r + st[d]] += co[d][3][q];
                    else if (bc[d] == ORC_BC_PERIODIC) row[r - st[d] * (nn[d] - 1)] += co[d][3][q];
                }
                if (alpha != 0.0) {
                    for (long cidx = 0; cidx < n; ++cidx) row[cidx] *= -alpha;
                    row[r] += 1.0;
                }
                row[N] = f[r];
                if (singular) {
                    double V = co[0][0][i] * co[1][0][j] * co[2][0][k];
                    row[n] = V;
                    M[n * W + r] = V;
                }
            }
    int rc = ORC_OK;
    for (long col = 0; col < N; ++col) {
        long piv = col;
        double best = fabs(M[col * W + col]);
        for (long r = col + 1; r < N; ++r) if (fabs(M[r * W + col]) > best) { best = fabs(M[r * W + col]); piv = r; }
        if (best == 0.0) { rc = ORC_ENUMERIC; break; }
        if (piv != col)
            for (long c2 = col; c2 <= N; ++c2) { double t = M[col * W + c2]; M[col * W + c2] = M[piv * W + c2]; M[piv * W + c2] = t; }
        for (long r = col + 1; r < N; ++r) {
            double m = M[r * W + col] / M[col * W + col];
            if (m == 0.0) continue;
            for (long c2 = col; c2 <= N; ++c2) M[r * W + c2] -= m * M[col * W + c2];
        }
    }
    if (rc == ORC_OK) {
        for (long r = N - 1; r >= 0; --r) {
            double s = M[r * W + N];
            for (long c2 = r + 1; c2 < N; ++c2) s -= M[r * W + c2] * M[c2 * W + N];
            M[r * W + N] = s / M[r * W + r];
        }
        for (long r = 0; r < n; ++r) phi[r] = M[r * W + N];
    }
    for (int d = 0; d < 3; ++d) for (int t = 0; t < 4; ++t) free(co[d][t]);
    free(M);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * Pressure projection on the staggered grid, Eq. 2c-2e (staggered arrangement P:57).
 *
 * [A18] Layout and boundary closure (the paper gives neither; both follow from L = D G having to be the
 * operator of Eq. 3 with the boundary rows of [A3] and the cyclic corners of P:102):
 *   velocities live on faces: u[k][j][f] on x-faces f = 0..nx (row length nx+1), v[k][g][i] on y-faces
 *   g = 0..ny, w[h][j][i] on z-faces h = 0..nz; face f lies between cells f-1 and f.
 *   divergence (cells):  (D u)_i = (u_{i+1} - u_i)/w_i  + the same in y and z.
 *   gradient (faces):    interior (G phi)_f = (phi_f - phi_{f-1}) / delta_f,  delta_f = x_c,f - x_c,f-1;
 *                        Neumann boundary face: 0 (mirror ghost phi_-1 = phi_0: a wall, the normal velocity there
 *                        is prescribed and not corrected); Dirichlet boundary face: ghost phi_-1 = -phi_0 at
 *                        distance w_0: (G phi)_0 = 2 phi_0 / w_0, (G phi)_n = -2 phi_{n-1} / w_{n-1};
 *                        periodic: faces 0 and n are the same face, (phi_0 - phi_{n-1}) / ((w_0 + w_{n-1})/2) [A17];
 *                        on input the entry of face n is ignored (D takes face 0 as the high face of cell n-1), on
 *                        output it is written as a copy of face 0.
 * ------------------------------------------------------------------------------------------ */
static double grad_face(const double *xf, int n, int bc, int f, const double *phi, size_t stride) {
    /* phi points at cell 0 of the line, cells `stride` apart */
    if (f > 0 && f < n) {
        double delta = 0.5 * (xf[f] + xf[f + 1]) - 0.5 * (xf[f - 1] + xf[f]);
        return (phi[(size_t)f * stride] - phi[(size_t)(f - 1) * stride]) / delta;
    }
    if (bc == ORC_BC_NEUMANN) return 0.0;
    if (bc == ORC_BC_PERIODIC) {
        double delta = 0.5 * ((xf[1] - xf[0]) + (xf[n] - xf[n - 1]));
        return (phi[0] - phi[(size_t)(n - 1) * stride]) / delta;
    }
    if (f == 0) return (phi[0] - (-phi[0])) / (xf[1] - xf[0]);
    return ((-phi[(size_t)(n - 1) * stride]) - phi[(size_t)(n - 1) * stride]) / (xf[n] - xf[n - 1]);
}

/* out = scale * D(u, v, w)   (Eq. 2c's right-hand side with scale = 1/(gamma_k dt)) */
int orc_divergence(int nx, int ny, int nz, const double *xf, const double *yf, const double *zf, const int bc[3],
                   const double *u, const double *v, const double *w, double scale, double *out) {
    if (!faces_ok(nx, xf) || !faces_ok(ny, yf) || !faces_ok(nz, zf) || !bc || !u || !v || !w || !out) return ORC_EINVAL;
    const size_t plane = (size_t)nx * ny;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                /* high faces: in a periodic direction face n is face 0 */
                int ih = (bc[0] == ORC_BC_PERIODIC && i == nx - 1) ? 0 : i + 1;
                int jh = (bc[1] == ORC_BC_PERIODIC && j == ny - 1) ? 0 : j + 1;
                int kh = (bc[2] == ORC_BC_PERIODIC && k == nz - 1) ? 0 : k + 1;
                double du = (u[ih + (size_t)(nx + 1) * (j + (size_t)ny * k)] - u[i + (size_t)(nx + 1) * (j + (size_t)ny * k)]) / (xf[i + 1] - xf[i]);
                double dv = (v[i + (size_t)nx * (jh + (size_t)(ny + 1) * k)] - v[i + (size_t)nx * (j + (size_t)(ny + 1) * k)]) / (yf[j + 1] - yf[j]);
                double dw = (w[i + (size_t)nx * j + plane * kh] - w[i + (size_t)nx * j + plane * k]) / (zf[k + 1] - zf[k]);
                out[i + (size_t)nx * j + plane * k] = scale * (du + dv + dw);
            }
    return ORC_OK;
}

/* (gu, gv, gw) = G phi on every face (boundary faces by the closure above). */
int orc_gradient(int nx, int ny, int nz, const double *xf, const double *yf, const double *zf, const int bc[3],
                 const double *phi, double *gu, double *gv, double *gw) {
    if (!faces_ok(nx, xf) || !faces_ok(ny, yf) || !faces_ok(nz, zf) || !bc || !phi || !gu || !gv || !gw) return ORC_EINVAL;
    const size_t plane = (size_t)nx * ny;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int f = 0; f <= nx; ++f)
                gu[f + (size_t)(nx + 1) * (j + (size_t)ny * k)] = grad_face(xf, nx, bc[0], f, phi + (size_t)nx * j + plane * k, 1);
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int g = 0; g <= ny; ++g)
            for (int i = 0; i < nx; ++i)
                gv[i + (size_t)nx * (g + (size_t)(ny + 1) * k)] = grad_face(yf, ny, bc[1], g, phi + i + plane * k, (size_t)nx);
#pragma omp parallel for schedule(static)
    for (int h = 0; h <= nz; ++h)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i)
                gw[i + (size_t)nx * j + plane * h] = grad_face(zf, nz, bc[2], h, phi + i + (size_t)nx * j, plane);
    return ORC_OK;
}

/* One projection, in the paper's order:
 *   Eq. 2c   L Phi = D u* / c          (c = gamma_k dt; `poisson` is a plan of the full operator, alpha = 0)
 *   Eq. 2d   u <- u* - c G Phi
 *   Eq. 2e   P <- P + Phi - alpha_p L_I Phi   (skipped if p == NULL; alpha_p = gamma_k nu dt / 2; L_I by `dirs`,
 *            evaluated in flux form; alpha_p == 0 is the fully explicit choice L_I = 0)
 * u, v, w are updated in place; phi receives Phi. */
int orc_project(const orc_plan *poisson, const double *xf, const double *yf, const double *zf, double c,
                double *u, double *v, double *w, double *phi, double *p, double alpha_p, int dirs) {
    if (!poisson || poisson->alpha != 0.0 || poisson->dirs != ORC_DIRS_XYZ || !(c > 0.0) || !u || !v || !w || !phi) return ORC_EINVAL;
    if (p && alpha_p != 0.0 && dirs != ORC_DIRS_XYZ && dirs != ORC_DIRS_YZ && dirs != ORC_DIRS_Z) return ORC_EINVAL;
    const int nx = poisson->nx, ny = poisson->ny, nz = poisson->nz;
    const int *bc = poisson->bc;
    const size_t n = (size_t)nx * ny * nz;
    const size_t nu = (size_t)(nx + 1) * ny * nz, nv = (size_t)nx * (ny + 1) * nz, nw = (size_t)nx * ny * (nz + 1);
    double *rhs = (double *)malloc(sizeof(double) * n), *work = (double *)malloc(sizeof(double) * n);
    double *gu = (double *)malloc(sizeof(double) * nu), *gv = (double *)malloc(sizeof(double) * nv), *gw = (double *)malloc(sizeof(double) * nw);
    int rc = (rhs && work && gu && gv && gw) ? ORC_OK : ORC_ENOMEM;
    if (rc == ORC_OK) rc = orc_divergence(nx, ny, nz, xf, yf, zf, bc, u, v, w, 1.0 / c, rhs);     /* 2c, rhs */
    if (rc == ORC_OK) rc = orc_solve(poisson, rhs, phi, work);                                    /* 2c */
    if (rc == ORC_OK) rc = orc_gradient(nx, ny, nz, xf, yf, zf, bc, phi, gu, gv, gw);
    if (rc == ORC_OK) {                                                                           /* 2d */
        for (size_t q = 0; q < nu; ++q) u[q] -= c * gu[q];
        for (size_t q = 0; q < nv; ++q) v[q] -= c * gv[q];
        for (size_t q = 0; q < nw; ++q) w[q] -= c * gw[q];
        /* periodic: face n is written as a copy of face 0 */
        if (bc[0] == ORC_BC_PERIODIC)
            for (size_t r = 0; r < (size_t)ny * nz; ++r) u[r * (nx + 1) + nx] = u[r * (nx + 1)];
        if (bc[1] == ORC_BC_PERIODIC)
            for (int k = 0; k < nz; ++k)
                for (int i = 0; i < nx; ++i) v[i + (size_t)nx * (ny + (size_t)(ny + 1) * k)] = v[i + (size_t)nx * (0 + (size_t)(ny + 1) * k)];
        if (bc[2] == ORC_BC_PERIODIC)
            for (size_t c = 0; c < (size_t)nx * ny; ++c) w[c + (size_t)nx * ny * nz] = w[c];
    }
    if (rc == ORC_OK && p) {                                                                      /* 2e */
        if (alpha_p == 0.0) {
            for (size_t q = 0; q < n; ++q) p[q] += phi[q];
        } else {
            rc = orc_apply_operator_flux_dirs(nx, ny, nz, xf, yf, zf, bc, alpha_p, dirs, phi, work);   /* (I - alpha L_I) Phi */
            if (rc == ORC_OK)
                for (size_t q = 0; q < n; ++q) p[q] += work[q];
        }
    }
    free(rhs); free(work); free(gu); free(gv); free(gw);
    return rc;
}
