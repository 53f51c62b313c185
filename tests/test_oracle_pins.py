"""Pins for the CPU oracle: everything here checks oracle/ against what the paper and the
mathematics fix (closed forms, invariants, brute force) — never against the CUDA path."""
import math

import numpy as np
import pytest

from paper_2603_09528_b200 import inputs as I

N_, D_ = I.NEUMANN, I.DIRICHLET


def _rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


# ------------------------------------------------------------------ 1-D operator (Eq. 3-4)
@pytest.mark.parametrize("bc", [N_, D_])
def test_operator_weighted_symmetry_and_uniform_stencil(orc, bc):
    xf = I.tanh_faces(33, 2.0, 1.7)
    w, a, b, c = orc.operator_1d(xf, bc)
    # D T symmetric because w_i c_i = w_{i+1} a_{i+1}
    assert np.allclose(w[:-1] * c[:-1], w[1:] * a[1:], rtol=1e-14)
    assert a[0] == 0.0 and c[-1] == 0.0
    # interior rows sum to zero; Neumann boundary rows too (T 1 = 0); Dirichlet rows do not
    rs = a + b + c
    assert np.abs(rs[1:-1]).max() < 1e-10 * np.abs(b).max()
    if bc == N_:
        assert abs(rs[0]) < 1e-10 * abs(b[0]) and abs(rs[-1]) < 1e-10 * abs(b[-1])
    # uniform grid -> [1,-2,1]/dx^2, boundary diagonal -1/dx^2 (Neumann) or -3/dx^2 (Dirichlet at the face)
    xf = I.tanh_faces(10, 5.0, 0.0)
    w, a, b, c = orc.operator_1d(xf, bc)
    dx2 = 0.25
    assert np.allclose(a[1:] * dx2, 1) and np.allclose(c[:-1] * dx2, 1) and np.allclose(b[1:-1] * dx2, -2)
    assert np.allclose([b[0] * dx2, b[-1] * dx2], -1.0 if bc == N_ else -3.0)


def test_operator_solution_converges_second_order(orc):
    # The scheme of Eq. 3 is second-order accurate in the SOLUTION (its pointwise truncation error
    # is only first order on a non-uniform grid).  u'' = f on [0,1]: Dirichlet u = sin(pi x)
    # (zero at the boundary faces, [A3]); Neumann u = cos(pi x) with the null constant fixed by hand.
    for bc in (D_, N_):
        errs = []
        for n in (32, 64, 128):
            xf = I.tanh_faces(n, 1.0, 1.0)
            xc = 0.5 * (xf[1:] + xf[:-1])
            w, a, b, c = orc.operator_1d(xf, bc)
            T = np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
            exact = np.sin(math.pi * xc) if bc == D_ else np.cos(math.pi * xc)
            f = -math.pi ** 2 * exact
            if bc == N_:
                f = f - (w * f).sum() / w.sum()
                u = np.linalg.lstsq(T, f, rcond=None)[0]
                u += (exact - u).mean()
            else:
                u = np.linalg.solve(T, f)
            errs.append(np.abs(u - exact).max())
        assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5


def test_coefficient_form_equals_flux_form(orc):
    # a,b,c (Eq. 4) and the difference-of-fluxes evaluation (Eq. 3) are two writings of the same operator.
    P = I.Problem("t", (7, 5, 6), (1.0, 2.0, 0.5), (1.5, 0.0, 2.0), (N_, D_, D_), 0.0, 1)
    xf, yf, zf = P.faces()
    phi = P.rhs()
    out = orc.apply_operator_flux(xf, yf, zf, P.bc, 0.0, phi)
    ref = np.zeros_like(phi)
    for axis, (ff, bc) in zip((2, 1, 0), ((xf, P.bc[0]), (yf, P.bc[1]), (zf, P.bc[2]))):
        w, a, b, c = orc.operator_1d(ff, bc)
        n = w.size
        T = np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
        ref += np.moveaxis(np.tensordot(T, np.moveaxis(phi, axis, 0), axes=(1, 0)), 0, axis)
        assert n == phi.shape[axis]
    assert _rel(out, ref) < 1e-13
    outh = orc.apply_operator_flux(xf, yf, zf, P.bc, 0.01, phi)
    assert _rel(outh, phi - 0.01 * ref) < 1e-13


# ------------------------------------------------------------------ eigendecomposition (Eq. 5-6)
@pytest.mark.parametrize("bc,n,L", [(N_, 32, 1.0), (D_, 32, 1.0), (N_, 96, 8.0), (D_, 45, 2.0)])
def test_uniform_grid_closed_form_eigenpairs(orc, bc, n, L):
    xf = I.tanh_faces(n, L, 0.0)
    dx = L / n
    lam, q = orc.eig_1d(xf, bc)
    k = np.arange(n)
    i = np.arange(n)[:, None]
    if bc == N_:   # BASELINE.json north_star / P:133: modified wavenumbers, DCT-II vectors
        cf = -(4 / dx ** 2) * np.sin(math.pi * k / (2 * n)) ** 2
        vec = np.cos(math.pi * k[None, :] * (i + 0.5) / n) * np.sqrt((2.0 - (k == 0)) / n)[None, :]
    else:          # DST-II
        cf = -(4 / dx ** 2) * np.sin(math.pi * (k + 1) / (2 * n)) ** 2
        vec = np.sin(math.pi * (k[None, :] + 1) * (i + 0.5) / n) * math.sqrt(2.0 / n)
        vec[:, -1] /= math.sqrt(2.0)
    assert np.abs(lam - cf).max() < 4e-15 * np.abs(cf).max() * n
    sign = np.sign((vec * q).sum(axis=0))
    assert np.abs(q - vec * sign).max() < 1e-9          # "up to sign" [A6]
    assert np.all((q * np.sqrt(np.diff(xf))[:, None]).sum(axis=0) > -1e-12)


@pytest.mark.parametrize("bc,n,beta", [(N_, 64, 2.0), (D_, 64, 2.0), (N_, 160, 3.0), (D_, 100, 2.5)])
def test_eigenbasis_orthogonal_and_diagonalising(orc, bc, n, beta):
    xf = I.tanh_faces(n, 1.0, beta)
    w, a, b, c = orc.operator_1d(xf, bc)
    d, o = orc.symmetrize_1d(w, a, b, c)
    S = np.diag(d) + np.diag(o, 1) + np.diag(o, -1)
    assert np.allclose(S, np.diag(np.sqrt(w)) @ (np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)) @ np.diag(1 / np.sqrt(w)),
                       rtol=1e-13, atol=1e-13 * np.abs(S).max())        # Eq. 5
    lam, q = orc.eig_1d(xf, bc)
    assert np.abs(q.T @ q - np.eye(n)).max() < 1e-13                    # P:110 Q~ orthogonal
    assert np.abs(S @ q - q * lam).max() < 1e-14 * n * np.abs(S).max()
    assert np.all(np.diff(lam) <= 0) and lam[0] <= 1e-300 and np.all(lam[1:] < 0)
    if bc == N_:
        assert lam[0] == 0.0 and np.allclose(q[:, 0], np.sqrt(w / w.sum()), rtol=1e-15)
    # Eq. 6: Q^{-1} Q = I with Q = D^{-1/2} Q~, Q^{-1} = Q~^T D^{1/2}
    Q = q / np.sqrt(w)[:, None]
    Qinv = q.T * np.sqrt(w)[None, :]
    assert np.abs(Qinv @ Q - np.eye(n)).max() < 1e-13
    T = np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
    assert np.abs(Qinv @ T @ Q - np.diag(lam)).max() < 1e-13 * n * np.abs(T).max()


def test_small_eigenvalues_are_relatively_accurate(orc):
    # [A9] accuracy rule: lambda_1.. must be right to ~1e-13 RELATIVE although ||S|| ~ 1e8.
    # Truth: extended-precision Rayleigh quotient in factored form of the returned vector
    # (quadratically accurate in the vector error).
    n, beta = 192, 3.0
    xf = I.tanh_faces(n, 1.0, beta)
    for bc in (N_, D_):
        lam, q = orc.eig_1d(xf, bc)
        L = np.longdouble
        xl = xf.astype(L)
        wl = np.diff(xl)
        dl = np.diff((xl[1:] + xl[:-1]) / 2)
        for m in range(1, 8):
            v = q[:, m].astype(L)
            g = v / np.sqrt(wl)
            fl = np.diff(g) / np.sqrt(dl)
            num = fl @ fl
            if bc == D_:
                num += 2 * (v[0] / wl[0]) ** 2 + 2 * (v[-1] / wl[-1]) ** 2
            truth = -num / (v @ v)
            assert abs(float((lam[m] - truth) / truth)) < 5e-14
        # the unrefined base solver (Jacobi alone) is visibly worse on the semi-definite operator
        lam0, _ = orc.eig_1d(xf, bc, refine_steps=0)
        if bc == N_:
            assert abs(lam0[1] / lam[1] - 1) > 1e-13
        assert abs(lam0[1] / lam[1] - 1) < 1e-8


def test_lambda1_converges_to_minus_pi_squared_second_order(orc):
    # continuous operator on [0,1]: first non-trivial Neumann eigenvalue -pi^2, Dirichlet -pi^2
    for bc, m in ((N_, 1), (D_, 0)):
        err = []
        for n in (32, 64, 128):
            lam, _ = orc.eig_1d(I.tanh_faces(n, 1.0, 1.5), bc)
            err.append(abs(lam[m] + math.pi ** 2))
        assert 3.5 < err[0] / err[1] < 4.5 and 3.5 < err[1] / err[2] < 4.5


# ------------------------------------------------------------------ 3-D solve vs brute-force dense LU (Eq. 7)
CASES = [
    # n,            L,               beta,            bc,            alpha
    ((4, 4, 4), (1.0, 1.0, 1.0), (1.2, 1.2, 1.5), (N_, N_, D_), 0.0),
    ((5, 7, 6), (1.0, 2.0, 1.5), (1.2, 2.0, 0.0), (N_, D_, D_), 0.0),
    ((7, 5, 6), (2.0, 1.0, 0.5), (0.0, 2.5, 1.0), (D_, N_, N_), 0.0),
    ((6, 7, 5), (1.0, 1.0, 3.0), (2.0, 1.0, 2.0), (D_, D_, D_), 0.0),
    ((8, 8, 8), (1.0, 1.0, 1.0), (2.0, 2.0, 2.0), (N_, N_, N_), 0.0),      # singular
    ((5, 6, 7), (1.0, 2.0, 1.5), (1.5, 0.0, 2.5), (N_, N_, N_), 0.0),      # singular, non-cubic
    ((8, 8, 8), (6.28, 3.14, 2.0), (2.0, 2.0, 2.5), (N_, N_, D_), 1e-3),   # Helmholtz
    ((6, 5, 7), (1.0, 1.0, 1.0), (3.0, 3.0, 3.0), (N_, N_, D_), 5e-1),     # Helmholtz, large alpha
    ((5, 7, 4), (1.0, 1.0, 1.0), (1.0, 2.0, 3.0), (N_, N_, N_), 2e-2),     # Helmholtz all-Neumann: non-singular
]


@pytest.mark.parametrize("n,L,beta,bc,alpha", CASES)
def test_solve_matches_bruteforce_dense_lu(orc, n, L, beta, bc, alpha):
    P = I.Problem("t", n, L, beta, bc, alpha, seed=sum(n))
    xf, yf, zf = P.faces()
    f = P.rhs()
    plan = orc.OraclePlan(xf, yf, zf, bc, alpha)
    phi = plan.solve(f)
    ref = orc.dense_solve_3d(xf, yf, zf, bc, alpha, f)
    assert plan.singular == P.singular
    assert _rel(phi, ref) < 1e-12
    if P.singular:   # gauge [A7]: zero volume-weighted mean
        V = np.diff(zf)[:, None, None] * np.diff(yf)[None, :, None] * np.diff(xf)[None, None, :]
        assert abs((V * phi).sum()) < 1e-13 * V.sum() * np.abs(phi).max()


def test_bruteforce_itself_satisfies_the_flux_form_equation(orc):
    # guards the pin: the dense assembly (coefficients) against the independent flux-form operator
    P = I.Problem("t", (5, 4, 6), (1.0, 2.0, 1.5), (1.2, 2.0, 1.0), (N_, D_, N_), 0.0, 5)
    xf, yf, zf = P.faces()
    f = P.rhs()
    ref = orc.dense_solve_3d(xf, yf, zf, P.bc, 0.0, f)
    assert _rel(orc.apply_operator_flux(xf, yf, zf, P.bc, 0.0, ref), f) < 1e-12


# ------------------------------------------------------------------ stage-level identities
def test_forward_then_inverse_transform_is_identity(orc):
    P = I.Problem("t", (24, 18, 5), (1.0, 2.0, 1.0), (2.0, 1.5, 1.0), (N_, D_, D_), 0.0, 3)
    xf, yf, zf = P.faces()
    f = P.rhs()
    plan = orc.OraclePlan(xf, yf, zf, P.bc, 0.0)
    assert _rel(plan.inverse_x(plan.forward_x(f)), f) < 1e-13
    assert _rel(plan.inverse_y(plan.forward_y(f)), f) < 1e-13
    # x and y transforms act on different axes: commute
    assert _rel(plan.forward_y(plan.forward_x(f)), plan.forward_x(plan.forward_y(f))) < 1e-13
    # forward_x on a single x-eigenvector line gives a unit vector in mode space (Eq. 6: Q^{-1} Q = I)
    lam, q = plan.eigen(0)
    g = np.zeros_like(f)
    g[2, 3, :] = q[:, 5] / np.sqrt(np.diff(xf))       # column 5 of Q = D^{-1/2} Q~
    h = plan.forward_x(g)
    e = np.zeros(24)
    e[5] = 1.0
    assert np.abs(h[2, 3] - e).max() < 1e-13 and np.abs(h).sum() - np.abs(h[2, 3]).sum() == 0.0


def test_thomas_stage_solves_shifted_tridiagonal_systems(orc):
    # (lambda_ij I + T_z) x = p for each mode, checked by multiplying back column by column
    P = I.Problem("t", (6, 5, 40), (1.0, 1.0, 2.0), (1.0, 1.5, 3.0), (N_, D_, D_), 0.0, 8)
    xf, yf, zf = P.faces()
    plan = orc.OraclePlan(xf, yf, zf, P.bc, 0.0)
    p = P.rhs()
    x = plan.thomas_z(p)
    lamx, _ = plan.eigen(0)
    lamy, _ = plan.eigen(1)
    w, a, b, c = orc.operator_1d(zf, P.bc[2])
    Tz = np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
    for j in range(5):
        for i in range(6):
            back = (Tz + (lamx[i] + lamy[j]) * np.eye(40)) @ x[:, j, i]
            assert np.abs(back - p[:, j, i]).max() < 1e-12 * max(1.0, np.abs(p[:, j, i]).max())
    # Helmholtz [A5]: ((1 - alpha sigma) I - alpha T_z) x = p
    alpha = 3e-3
    planh = orc.OraclePlan(xf, yf, zf, P.bc, alpha)
    xh = planh.thomas_z(p)
    for j, i in ((0, 0), (4, 5), (2, 3)):
        back = ((1 - alpha * (lamx[i] + lamy[j])) * np.eye(40) - alpha * Tz) @ xh[:, j, i]
        assert np.abs(back - p[:, j, i]).max() < 1e-13


# ------------------------------------------------------------------ residuals, eigenfunctions, manufactured solutions
@pytest.mark.parametrize("cfg", ["c1", "c2"])
def test_residual_at_roundoff_on_baseline_configs(orc, cfg):
    P = I.CONFIGS[cfg][0]
    xf, yf, zf = P.faces()
    f = P.rhs()
    phi = orc.OraclePlan(xf, yf, zf, P.bc, P.alpha).solve(f)
    r = orc.residual_norms(xf, yf, zf, P.bc, P.alpha, f, phi)
    assert r["rel2"] < 1e-11 and r["relL2vol"] < 1e-11 and r["relmax"] < 1e-10       # P:254, BASELINE north_star
    assert r["rel2"] < 2e-13                                                        # expected level (SURVEY c.6)


def test_residual_norms_special_cases(orc):
    # orc_residual_norms pinned by cases with a closed form: phi = 0 (residual = f: every relative norm is exactly 1);
    # f = 0 with phi a unit vector (residual = minus one column of the operator — the diagonal b_x + b_y + b_z of that cell and
    # six neighbour coefficients — whose largest entry the backward error divides by the sum of the 1-D absolute row sums);
    # invariance under a common scaling of f and phi.
    P = I.Problem("norms", (7, 5, 6), (1.0, 2.0, 1.5), (2.0, 1.0, 2.5), (N_, D_, N_), 0.0, 3)
    xf, yf, zf = P.faces()
    f = I.uniform_pm1(11, P.points).reshape(6, 5, 7)
    zero = np.zeros_like(f)
    r = orc.residual_norms(xf, yf, zf, P.bc, 0.0, f, zero)
    assert r["rel2"] == 1.0 and r["relL2vol"] == 1.0 and r["relmax"] == 1.0 and r["backward"] == 1.0
    ops = [orc.operator_1d(g, b) for g, b in zip((xf, yf, zf), P.bc)]          # (w, a, b, c) per direction
    rowsum = sum(float(np.max(np.abs(a) + np.abs(b) + np.abs(c))) for (_, a, b, c) in ops)
    i, j, k = 3, 2, 4
    e = zero.copy(); e[k, j, i] = 1.0
    # column (i, j, k) of the operator: the diagonal and, per direction, c of the row before and a of the row after
    col = [abs(ops[0][2][i] + ops[1][2][j] + ops[2][2][k])]
    for (_, a, b, c), m in zip(ops, (i, j, k)):
        col += [abs(c[m - 1]), abs(a[m + 1])]
    tiny = np.full_like(f, 1e-300)                                             # f = 0 would divide by zero in the relative norms
    r = orc.residual_norms(xf, yf, zf, P.bc, 0.0, tiny, e)
    assert abs(r["backward"] - max(col) / rowsum) <= 1e-12 * max(col) / rowsum
    assert 0.0 < r["backward"] < 1.0
    # a genuine solution: backward error at round-off, never above the max-norm residual; both scale-invariant
    phi = orc.OraclePlan(xf, yf, zf, P.bc, 0.0).solve(f)
    r1 = orc.residual_norms(xf, yf, zf, P.bc, 0.0, f, phi)
    r2 = orc.residual_norms(xf, yf, zf, P.bc, 0.0, 8.0 * f, 8.0 * phi)
    assert r1["backward"] <= r1["relmax"] < 1e-12 and r1["backward"] < 1e-15
    for key in r1:                                                             # (the OpenMP reductions may reorder the sums)
        assert abs(r1[key] - r2[key]) <= 1e-12 * r1[key], key


def test_residual_singular_stretched(orc):
    P = I.Problem("t", (64, 48, 56), (1.0, 1.0, 1.0), (2.0, 2.0, 2.0), (N_, N_, N_), 0.0, 2)
    xf, yf, zf = P.faces()
    f = P.rhs()
    phi = orc.OraclePlan(xf, yf, zf, P.bc, P.alpha).solve(f)
    r = orc.residual_norms(xf, yf, zf, P.bc, P.alpha, f, phi)
    assert r["rel2"] < 1e-12
    # [A8]: with only the PLAIN mean removed the rhs is incompatible and the residual is far from round-off
    g = I.uniform_pm1(2, f.size).reshape(f.shape)
    g -= g.mean()
    phig = orc.OraclePlan(xf, yf, zf, P.bc, P.alpha).solve(g)
    assert orc.residual_norms(xf, yf, zf, P.bc, P.alpha, g, phig)["rel2"] > 1e-7


def test_discrete_eigenfunction_rhs_uniform_grid(orc):
    # all-uniform grid: f = product of closed-form modes  =>  phi = f / (lx + ly + lz) exactly
    nx, ny, nz = 12, 10, 14
    Lx, Ly, Lz = 2.0, 1.0, 3.0
    xf, yf, zf = I.tanh_faces(nx, Lx, 0), I.tanh_faces(ny, Ly, 0), I.tanh_faces(nz, Lz, 0)
    kx, ky, kz = 3, 2, 4
    cx = np.cos(math.pi * kx * (np.arange(nx) + 0.5) / nx)                  # Neumann
    cy = np.cos(math.pi * ky * (np.arange(ny) + 0.5) / ny)                  # Neumann
    sz = np.sin(math.pi * (kz + 1) * (np.arange(nz) + 0.5) / nz)            # Dirichlet
    f = sz[:, None, None] * cy[None, :, None] * cx[None, None, :]
    lx = -(4 / (Lx / nx) ** 2) * math.sin(math.pi * kx / (2 * nx)) ** 2
    ly = -(4 / (Ly / ny) ** 2) * math.sin(math.pi * ky / (2 * ny)) ** 2
    lz = -(4 / (Lz / nz) ** 2) * math.sin(math.pi * (kz + 1) / (2 * nz)) ** 2
    phi = orc.OraclePlan(xf, yf, zf, (N_, N_, D_), 0.0).solve(f)
    assert _rel(phi, f / (lx + ly + lz)) < 1e-12
    alpha = 0.05
    u = orc.OraclePlan(xf, yf, zf, (N_, N_, D_), alpha).solve(f)
    assert _rel(u, f / (1 - alpha * (lx + ly + lz))) < 1e-12


@pytest.mark.parametrize("bc,alpha", [((N_, N_, D_), 0.0), ((N_, N_, N_), 0.0), ((D_, N_, D_), 2e-3)])
def test_manufactured_smooth_solution_on_stretched_grid(orc, bc, alpha):
    P = I.Problem("t", (40, 36, 44), (1.0, 2.0, 1.0), (2.0, 2.5, 3.0), bc, alpha, 0)
    xf, yf, zf = P.faces()
    xc, yc, zc = (0.5 * (g[1:] + g[:-1]) for g in (xf, yf, zf))
    star = (np.cos(2 * math.pi * zc)[:, None, None] * np.cos(math.pi * yc / 2.0)[None, :, None]
            * (1.0 + np.cos(3 * math.pi * xc))[None, None, :])
    V = np.diff(zf)[:, None, None] * np.diff(yf)[None, :, None] * np.diff(xf)[None, None, :]
    if P.singular:
        star -= (V * star).sum() / V.sum()
    f = orc.apply_operator_flux(xf, yf, zf, bc, alpha, star)
    phi = orc.OraclePlan(xf, yf, zf, bc, alpha).solve(f)
    assert _rel(phi, star) < 1e-9 if alpha == 0.0 else _rel(phi, star) < 1e-12


def test_gauge_of_singular_solve(orc):
    # [A7] P:219: the vanishing final pivot of mode (0,0) is replaced by "unknown := 0", then the
    # column's dz-weighted mean is removed -> zero volume-weighted mean of phi.
    P = I.Problem("t", (20, 16, 24), (1.0, 1.0, 1.0), (2.0, 1.0, 2.5), (N_, N_, N_), 0.0, 4)
    xf, yf, zf = P.faces()
    f = P.rhs()
    plan = orc.OraclePlan(xf, yf, zf, P.bc, 0.0)
    V = np.diff(zf)[:, None, None] * np.diff(yf)[None, :, None] * np.diff(xf)[None, None, :]
    a = plan.solve(f)
    assert abs((V * a).sum()) < 1e-13 * np.abs(a).max() * V.sum()
    # phi is recovered whatever null-space component the exact solution carried
    star = a + 0.77
    g = orc.apply_operator_flux(xf, yf, zf, P.bc, 0.0, star)
    assert np.abs(plan.solve(g) - a).max() < 1e-9 * np.abs(a).max()
    # An INCOMPATIBLE rhs (f + c) is not projected: the paper's rule drops the last z-equation of
    # mode (0,0), so the residual lives only in the last plane and is constant there [A8].
    b = plan.solve(f + 0.37)
    r = (f + 0.37) - orc.apply_operator_flux(xf, yf, zf, P.bc, 0.0, b)
    assert np.abs(r[:-1]).max() < 1e-10
    assert np.abs(r[-1] - r[-1].mean()).max() < 1e-10 and abs(r[-1].mean()) > 1.0
    assert abs((V * b).sum()) < 1e-13 * np.abs(b).max() * V.sum()


def test_helmholtz_tends_to_identity_and_to_poisson(orc):
    # (I - alpha L) u = f: alpha -> 0+ gives u -> f; large alpha gives u -> -phi/alpha (non-singular L)
    P = I.Problem("t", (10, 12, 14), (1.0, 1.0, 1.0), (1.5, 1.5, 2.0), (N_, N_, D_), 0.0, 6)
    xf, yf, zf = P.faces()
    f = P.rhs()
    u = orc.OraclePlan(xf, yf, zf, P.bc, 1e-12).solve(f)
    assert _rel(u, f) < 1e-6
    phi = orc.OraclePlan(xf, yf, zf, P.bc, 0.0).solve(f)
    big = 1e9
    ub = orc.OraclePlan(xf, yf, zf, P.bc, big).solve(f)
    assert _rel(ub * (-big), phi) < 1e-6
