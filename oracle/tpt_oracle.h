/*
 * tpt_oracle.h — CPU ORACLE for the tensor-product–Thomas Poisson/Helmholtz solver.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code, header, table
 * or helper with the CUDA path under paper_2603_09528_b200/ and neither includes the other.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md, cited as P:line):
 *   the solution of  T phi = f            (Poisson,   helmholtz_alpha == 0)     P:139 Eq. 7
 *               or  (I - alpha T) u = f   (Helmholtz, helmholtz_alpha  > 0)     P:68  Eq. 2b
 *   with T = Tx (x) Iy (x) Iz + Ix (x) Ty (x) Iz + Ix (x) Iy (x) Tz, each T_d the second-order
 *   finite-difference Laplacian of Eq. 3–4 on a non-uniform staggered grid,
 *   by the paper's five steps: forward x, forward y eigenbasis transforms,
 *   one Thomas solve along z per mode, inverse y, inverse x.
 *   Everything is FP64, plain loops, no blocking/fusion; OpenMP only over independent
 *   lines/planes/columns.
 *
 * Field layout everywhere: idx = i + nx*(j + ny*k)  (x contiguous, z slowest; "leading
 * dimension N_x").
 *
 * Readings of silent/garbled passages (A1–A16) are marked "[A#]" in the .c.
 *
 * Parity pins (tests/, -m "not gpu"): brute-force dense LU of the assembled operator on <= 8^3
 * grids; closed-form eigenvalues / DCT-II eigenvectors on uniform grids; Q^T Q = I; flux-form
 * residual at round-off; discrete eigenfunction rhs; manufactured smooth solutions; lambda_1
 * -> -pi^2; gauge invariance; footnote-4 grading ratios (inputs); for the projection (Eq. 2c-2e): D G = the
 * flux-form Laplacian, closed forms of D and G on polynomial fields, summation by parts (D = -G^T in the cell /
 * face volume inner products), discretely divergence-free result.  No function here is "parity unpinned".
 */
#ifndef TPT_ORACLE_H
#define TPT_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

/* PERIODIC (P:102 cyclic corners, P:211 dense cyclic operator): x and y are diagonalised; a periodic z makes the sweep a cyclic
 * tridiagonal solve (Sherman-Morrison, A19). */
enum { ORC_BC_NEUMANN = 0, ORC_BC_DIRICHLET = 1, ORC_BC_PERIODIC = 2 };
/* Implicitly treated directions L_I of the Helmholtz problem, Eq. 2b: bit 0 = x, 1 = y, 2 = z. */
enum { ORC_DIRS_Z = 4, ORC_DIRS_YZ = 6, ORC_DIRS_XYZ = 7 };
enum { ORC_OK = 0, ORC_EINVAL = -1, ORC_ENOMEM = -2, ORC_ENUMERIC = -4 };

typedef struct orc_plan orc_plan;

/* ---- 1-D building blocks (each individually pinned) ------------------------------------ */

/* Eq. 3–4 with boundary rows [A1,A2,A3]. faces xf[0..n]; outputs w,a,b,c of length n. */
int orc_operator_1d(int n, const double *xf, int bc, double *w, double *a, double *b, double *c);

/* Eq. 5: S = D^{1/2} T D^{-1/2}; diag[0..n-1], off[0..n-2]. */
int orc_symmetrize_1d(int n, const double *w, const double *a, const double *b, const double *c,
                      double *diag, double *off);

/* Eigendecomposition of S by cyclic Jacobi + `refine_steps` guarded Ogita–Aishima
 * refinement steps in factored form [A9]; sorted descending (mode 0 smoothest), sign-fixed [A6],
 * Neumann null pair overwritten analytically.  lambda[n]; qtilde[n*n] row-major,
 * qtilde[i*n+m] = component i of mode m. */
int orc_eig_1d(int n, const double *xf, int bc, int refine_steps, double *lambda, double *qtilde);

/* ---- 3-D plan and the five steps --------------------------------------------------------- */

int  orc_plan_create(orc_plan **out, int nx, int ny, int nz,
                     const double *xf, const double *yf, const double *zf,
                     const int bc[3], double helmholtz_alpha);
/* Same, but takes eigen-decompositions computed earlier by orc_eig_1d (lets tests cache the
 * O(N^3) Jacobi across plans that share a direction's grid). */
int  orc_plan_create_with_eig(orc_plan **out, int nx, int ny, int nz,
                              const double *xf, const double *yf, const double *zf,
                              const int bc[3], double helmholtz_alpha,
                              const double *lamx, const double *qx,
                              const double *lamy, const double *qy);
void orc_plan_destroy(orc_plan *p);
int  orc_plan_is_singular(const orc_plan *p);
int  orc_plan_get_eigen(const orc_plan *p, int dir, double *lambda, double *qtilde);
/* Partial implicit diffusion: (I - alpha L_I) u = f with L_I = L_z (ORC_DIRS_Z: only the tridiagonal
 * solve), L_y + L_z (ORC_DIRS_YZ: the x transforms are omitted) or L (default).  Helmholtz plans only. */
int  orc_plan_set_implicit_dirs(orc_plan *p, int dirs);

void orc_forward_x(const orc_plan *p, const double *in, double *out);   /* Eq. 10a */
void orc_forward_y(const orc_plan *p, const double *in, double *out);   /* Eq. 10b */
int  orc_thomas_z (const orc_plan *p, double *field);                   /* P:161–163, gauge P:219 */
void orc_inverse_y(const orc_plan *p, const double *in, double *out);   /* Eq. 12a */
void orc_inverse_x(const orc_plan *p, const double *in, double *out);   /* Eq. 12b */

/* Steps 2.1–2.5. work: nx*ny*nz doubles of scratch. phi may not alias f. */
int  orc_solve(const orc_plan *p, const double *f, double *phi, double *work);

/* ---- independent definitions used as pins / checks ---------------------------------------- */

/* out = T phi (alpha == 0) or (I - alpha T) phi, evaluated in FLUX form directly from Eq. 3
 * (differences first), not through a,b,c. */
int  orc_apply_operator_flux(int nx, int ny, int nz,
                             const double *xf, const double *yf, const double *zf,
                             const int bc[3], double alpha, const double *phi, double *out);

/* The same for a partial operator I - alpha L_I, L_I = sum of the 1-D Laplacians of the directions in `dirs`. */
int  orc_apply_operator_flux_dirs(int nx, int ny, int nz,
                                  const double *xf, const double *yf, const double *zf,
                                  const int bc[3], double alpha, int dirs, const double *phi, double *out);

/* Residual r = f - Op(phi) in flux form; norms[0] = ||r||2/||f||2, norms[1] = volume-weighted
 * L2 ratio, norms[2] = max|r|/max|f|, norms[3] = normwise backward error
 * max|r| / (||Op||_inf max|phi| + max|f|). */
int  orc_residual_norms(int nx, int ny, int nz,
                        const double *xf, const double *yf, const double *zf,
                        const int bc[3], double alpha, const double *f, const double *phi,
                        double norms[4]);

int  orc_residual_norms_dirs(int nx, int ny, int nz,
                             const double *xf, const double *yf, const double *zf,
                             const int bc[3], double alpha, int dirs, const double *f, const double *phi,
                             double norms[4]);

/* Brute force: assemble the dense operator of Eq. 7 (n = nx*ny*nz <= 4096) and solve by
 * Gaussian elimination with partial pivoting.  Singular (all-Neumann Poisson): bordered system
 * [T v; v^T 0] with v = cell volumes (zero volume-weighted mean). */
int  orc_dense_solve_3d(int nx, int ny, int nz,
                        const double *xf, const double *yf, const double *zf,
                        const int bc[3], double alpha, const double *f, double *phi);

int  orc_dense_solve_3d_dirs(int nx, int ny, int nz,
                             const double *xf, const double *yf, const double *zf,
                             const int bc[3], double alpha, int dirs, const double *f, double *phi);

/* ---- pressure projection on the staggered grid, Eq. 2c-2e ------------------------------ */
/* Face arrays: u (nz, ny, nx+1), v (nz, ny+1, nx), w (nz+1, ny, nx); closure of the boundary faces: reading [A18]. */
int  orc_divergence(int nx, int ny, int nz, const double *xf, const double *yf, const double *zf, const int bc[3],
                    const double *u, const double *v, const double *w, double scale, double *out);
int  orc_gradient(int nx, int ny, int nz, const double *xf, const double *yf, const double *zf, const int bc[3],
                  const double *phi, double *gu, double *gv, double *gw);
/* L Phi = D u / c;  u -= c G Phi;  p += Phi - alpha_p L_I Phi  (p may be NULL).  `poisson`: alpha = 0 plan. */
int  orc_project(const orc_plan *poisson, const double *xf, const double *yf, const double *zf, double c,
                 double *u, double *v, double *w, double *phi, double *p, double alpha_p, int dirs);

int  orc_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
