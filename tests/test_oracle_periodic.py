"""Pins for the oracle's periodic directions (P:102 cyclic corners, P:211 dense cyclic operator, P:294 the paper's
benchmark BCs: periodic x, Neumann y, z) — closed forms, library FFT, brute force, invariances; never the CUDA path."""
import math

import numpy as np
import pytest

from paper_2603_09528_b200 import inputs as I

N_, D_, P_ = I.NEUMANN, I.DIRICHLET, I.PERIODIC


def _rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


def _dense_T(orc, xf, bc):
    w, a, b, c = orc.operator_1d(xf, bc)
    n = w.size
    T = np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
    if bc == P_:
        T[0, n - 1] += a[0]
        T[n - 1, 0] += c[n - 1]
    return w, T


def test_periodic_operator_rows_symmetry_and_uniform_stencil(orc):
    xf = I.tanh_faces(17, 2.0, 1.6)
    w, T = _dense_T(orc, xf, P_)
    assert np.abs(T.sum(axis=1)).max() < 1e-10 * np.abs(T).max()          # T 1 = 0: constants are in the null space
    assert np.allclose(w[:, None] * T, (w[:, None] * T).T, rtol=1e-13)     # D T symmetric, corners included
    # the wrap-around face sits between cell n-1 (one period back) and cell 0: spacing (w_0 + w_{n-1})/2
    assert math.isclose(T[0, 16], 1.0 / (w[0] * 0.5 * (w[0] + w[16])), rel_tol=1e-14)
    xf = I.tanh_faces(8, 4.0, 0.0)
    w, T = _dense_T(orc, xf, P_)
    C = np.roll(np.eye(8), 1, axis=1) + np.roll(np.eye(8), -1, axis=1) - 2 * np.eye(8)   # circulant [1,-2,1]
    assert np.allclose(T * 0.25, C, atol=1e-14)
    with pytest.raises(RuntimeError):
        orc.operator_1d(I.tanh_faces(2, 1.0, 0.0), P_)                     # n = 2: the two couplings coincide


def test_periodic_uniform_eigenpairs_are_fourier(orc):
    n, L = 24, 3.0
    xf = I.tanh_faces(n, L, 0.0)
    lam, q = orc.eig_1d(xf, P_)
    dx = L / n
    k = np.arange(n)
    cf = np.sort(-(4 / dx ** 2) * np.sin(math.pi * k / n) ** 2)[::-1]      # modified wavenumbers, pairs k / n-k
    assert np.abs(lam - cf).max() < 1e-13 * np.abs(cf).max()
    assert lam[0] == 0.0 and np.allclose(q[:, 0], 1 / math.sqrt(n), rtol=1e-14)
    assert np.abs(q.T @ q - np.eye(n)).max() < 1e-13
    # every eigenvector lies in the span of cos/sin of its own wavenumber: its DFT has support on {k, n-k} only
    F = np.fft.fft(q, axis=0)
    for m in range(n):
        kk = int(round(math.asin(math.sqrt(min(1.0, -lam[m] * dx * dx / 4))) * n / math.pi))
        mask = np.ones(n, bool)
        mask[[kk % n, (n - kk) % n]] = False
        assert np.abs(F[mask, m]).max() < 1e-12


def test_periodic_stretched_eigenpairs_satisfy_definition(orc):
    xf = I.tanh_faces(40, 1.0, 1.8)
    w, T = _dense_T(orc, xf, P_)
    S = np.sqrt(w)[:, None] * T / np.sqrt(w)[None, :]                      # Eq. 5
    assert np.allclose(S, S.T, rtol=1e-12, atol=1e-12 * np.abs(S).max())
    lam, q = orc.eig_1d(xf, P_)
    assert np.abs(q.T @ q - np.eye(40)).max() < 1e-13
    assert np.abs(S @ q - q * lam[None, :]).max() < 1e-12 * np.abs(S).max()
    ref = np.linalg.eigvalsh(S)[::-1]
    assert np.abs(lam - ref).max() < 1e-12 * np.abs(ref).max()
    assert np.all(np.diff(lam) <= 0) and lam[0] == 0.0


def test_periodic_uniform_1d_solve_equals_fft_division(orc):
    # uniform periodic x: the method "reduces to a Fourier expansion with analytical eigenvalues"; with one
    # cell in... rather: Helmholtz in z-decoupled form.  Use DIRS-free check: 3-D Helmholtz with periodic x, y and
    # tiny alpha*T_z contribution handled exactly by the same FFT diagonalisation in x, y and a dense solve in z.
    nx, ny, nz = 16, 12, 5
    xf, yf, zf = I.tanh_faces(nx, 2.0, 0.0), I.tanh_faces(ny, 1.5, 0.0), I.tanh_faces(nz, 1.0, 1.2)
    alpha = 0.05
    f = I.uniform_pm1(3, nx * ny * nz).reshape(nz, ny, nx)
    u = orc.OraclePlan(xf, yf, zf, (P_, P_, D_), alpha).solve(f)
    lx = -(4 / (2.0 / nx) ** 2) * np.sin(math.pi * np.arange(nx) / nx) ** 2
    ly = -(4 / (1.5 / ny) ** 2) * np.sin(math.pi * np.arange(ny) / ny) ** 2
    _, Tz = _dense_T(orc, zf, D_)
    fh = np.fft.fft2(f, axes=(1, 2))
    uh = np.empty_like(fh)
    for j in range(ny):
        for i in range(nx):
            A = (1 - alpha * (lx[i] + ly[j])) * np.eye(nz) - alpha * Tz
            uh[:, j, i] = np.linalg.solve(A, fh[:, j, i])
    ref = np.fft.ifft2(uh, axes=(1, 2)).real
    assert _rel(u, ref) < 1e-13


@pytest.mark.parametrize("bc,alpha", [((P_, N_, D_), 0.0), ((P_, P_, N_), 0.0), ((N_, P_, D_), 0.3), ((P_, D_, N_), 0.0),
                                      ((P_, N_, N_), 0.0),
                                      # periodic z: the sweep is a cyclic tridiagonal solve (A19)
                                      ((N_, D_, P_), 0.0), ((N_, N_, P_), 0.0), ((P_, P_, P_), 0.0), ((D_, N_, P_), 0.4),
                                      ((P_, N_, P_), 2e-3)])
def test_periodic_matches_brute_force_lu(orc, bc, alpha):
    xf, yf, zf = I.tanh_faces(5, 1.0, 1.3), I.tanh_faces(7, 2.0, 1.8), I.tanh_faces(6, 0.5, 2.2)
    f = I.uniform_pm1(21, 5 * 7 * 6).reshape(6, 7, 5)
    singular = alpha == 0.0 and D_ not in bc
    if singular:
        I.remove_weighted_mean(f, xf, yf, zf)
    plan = orc.OraclePlan(xf, yf, zf, bc, alpha)
    assert plan.singular == singular
    u = plan.solve(f)
    ref = orc.dense_solve_3d(xf, yf, zf, bc, alpha, f)
    assert _rel(u, ref) < 1e-12
    assert orc.residual_norms(xf, yf, zf, bc, alpha, f, u)["rel2"] < 1e-13
    if singular:
        V = np.diff(zf)[:, None, None] * np.diff(yf)[None, :, None] * np.diff(xf)[None, None, :]
        assert abs((V * u).sum()) < 1e-14 * np.abs(u).max() * V.sum()


def test_periodic_flux_operator_matches_dense_rows_and_translation_invariance(orc):
    nx, ny, nz = 9, 6, 4
    xf, yf, zf = I.tanh_faces(nx, 1.0, 1.1), I.tanh_faces(ny, 1.0, 0.0), I.tanh_faces(nz, 1.0, 0.9)
    bc = (P_, P_, N_)
    phi = I.uniform_pm1(5, nx * ny * nz).reshape(nz, ny, nx)
    _, Tx = _dense_T(orc, xf, P_)
    _, Ty = _dense_T(orc, yf, P_)
    _, Tz = _dense_T(orc, zf, N_)
    ref = np.einsum("im,kjm->kji", Tx, phi) + np.einsum("jm,kmi->kji", Ty, phi) + np.einsum("km,mji->kji", Tz, phi)
    assert np.allclose(orc.apply_operator_flux(xf, yf, zf, bc, 0.0, phi), ref, rtol=1e-12, atol=1e-11)
    # y is uniform and periodic: shifting the rhs cyclically in y shifts the solution (Helmholtz, non-singular)
    f = I.uniform_pm1(6, nx * ny * nz).reshape(nz, ny, nx)
    plan = orc.OraclePlan(xf, yf, zf, bc, 0.1)
    assert _rel(plan.solve(np.roll(f, 2, axis=1)), np.roll(plan.solve(f), 2, axis=1)) < 1e-13


def test_periodic_z_cyclic_sweep_closed_forms(orc):
    # (1) uniform periodic z, rhs = a discrete Fourier mode in z times eigenmodes in x, y: phi = f / (lx + ly + lz) exactly
    nx, ny, nz = 6, 5, 16
    xf, yf, zf = I.tanh_faces(nx, 1.0, 0.0), I.tanh_faces(ny, 2.0, 0.0), I.tanh_faces(nz, 3.0, 0.0)
    plan = orc.OraclePlan(xf, yf, zf, (N_, N_, P_), 0.0)
    lamx, qx = plan.eigen(0)
    lamy, qy = plan.eigen(1)
    dz = 3.0 / nz
    for m, (ix, iy) in ((3, (2, 1)), (8, (0, 4)), (1, (0, 0))):
        zmode = np.cos(2 * math.pi * m * (np.arange(nz) + 0.5) / nz + 0.3)
        f = zmode[:, None, None] * qy[:, iy][None, :, None] * qx[:, ix][None, None, :]
        lz = -(4 / dz ** 2) * math.sin(math.pi * m / nz) ** 2
        assert _rel(plan.solve(f), f / (lamx[ix] + lamy[iy] + lz)) < 1e-12
    # (2) a stretched periodic z against numpy's dense solve of the assembled cyclic column systems (Helmholtz, z only)
    zf = I.tanh_faces(11, 1.0, 1.7)
    xf2 = I.tanh_faces(3, 1.0, 0.0)
    w, T = _dense_T(orc, zf, P_)
    alpha = 0.07
    f = I.uniform_pm1(3, 11 * 3 * 3).reshape(11, 3, 3)
    u = orc.OraclePlan(xf2, xf2, zf, (N_, N_, P_), alpha, dirs=4).solve(f)
    ref = np.linalg.solve(np.eye(11) - alpha * T, f.reshape(11, 9)).reshape(11, 3, 3)
    assert _rel(u, ref) < 1e-13
    # (3) z uniform and periodic: a cyclic shift of the rhs in z shifts the solution (non-singular Helmholtz)
    zf = I.tanh_faces(9, 1.0, 0.0)
    xs, ys = I.tanh_faces(4, 1.0, 1.2), I.tanh_faces(5, 1.0, 0.8)
    plan = orc.OraclePlan(xs, ys, zf, (N_, D_, P_), 0.2)
    f = I.uniform_pm1(9, 9 * 5 * 4).reshape(9, 5, 4)
    assert _rel(plan.solve(np.roll(f, 4, axis=0)), np.roll(plan.solve(f), 4, axis=0)) < 1e-13
    # (4) n = 2 cells cannot be periodic (the two couplings coincide)
    with pytest.raises(RuntimeError):
        orc.OraclePlan(xs, ys, I.tanh_faces(2, 1.0, 0.0), (N_, N_, P_), 0.0)


def test_paper_benchmark_bcs_residual_on_stretched_grid(orc):
    # periodic x, Neumann y and z (singular Poisson).  48 x 40 x 32, uniform x, stretched y, z.
    P = I.Problem("duct", (48, 40, 32), (6.0, 1.0, 1.0), (0.0, 2.0, 2.0), (P_, N_, N_), 0.0, 4)
    assert P.singular
    xf, yf, zf = P.faces()
    f = P.rhs()
    u = orc.OraclePlan(xf, yf, zf, P.bc, 0.0).solve(f)
    r = orc.residual_norms(xf, yf, zf, P.bc, 0.0, f, u)
    assert r["rel2"] < 1e-12 and r["relL2vol"] < 1e-12
