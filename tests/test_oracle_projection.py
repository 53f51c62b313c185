"""Pins of the oracle's pressure projection (Eq. 2c-2e) on the staggered grid:
closed forms of D and G on polynomial fields, D G = the flux-form Laplacian of Eq. 3 (already pinned), summation by
parts (D = -G^T in the cell-volume / face-volume inner products), and the properties the paper states for the
projection ("discretely divergence-free to machine precision" on white noise)."""
import itertools

import numpy as np
import pytest

from paper_2603_09528_b200 import inputs as I

N_, D_, P_ = I.NEUMANN, I.DIRICHLET, I.PERIODIC


def _grid(n=(7, 6, 5), L=(1.0, 2.0, 1.5), beta=(1.5, 2.0, 1.2)):
    return [I.tanh_faces(n[d], L[d], beta[d]) for d in range(3)]


def _centres(f):
    return 0.5 * (f[1:] + f[:-1])


def _wall_zero(u, v, w, bc):
    """Neumann (wall) boundary faces carry the prescribed normal velocity: homogeneous here."""
    if bc[0] == N_:
        u[:, :, 0] = u[:, :, -1] = 0.0
    if bc[1] == N_:
        v[:, 0, :] = v[:, -1, :] = 0.0
    if bc[2] == N_:
        w[0] = w[-1] = 0.0
    if bc[0] == P_:
        u[:, :, -1] = u[:, :, 0]
    if bc[1] == P_:
        v[:, -1, :] = v[:, 0, :]
    return u, v, w


def _random_velocity(orc, n, bc, seed):
    rng = np.random.default_rng(seed)
    su, sv, sw = orc.face_shapes(*n)
    return _wall_zero(rng.uniform(-1, 1, su), rng.uniform(-1, 1, sv), rng.uniform(-1, 1, sw), bc)


def test_divergence_of_linear_fields_is_exact(orc):
    xf, yf, zf = _grid()
    nx, ny, nz = xf.size - 1, yf.size - 1, zf.size - 1
    su, sv, sw = orc.face_shapes(nx, ny, nz)
    u = np.broadcast_to(2.0 * xf[None, None, :], su).copy()           # u = 2x on x-faces
    v = np.broadcast_to(-3.0 * yf[None, :, None], sv).copy()          # v = -3y
    w = np.broadcast_to(0.5 * zf[:, None, None], sw).copy()           # w = z/2
    d = orc.divergence(xf, yf, zf, (D_, D_, D_), u, v, w)
    assert np.abs(d - (2.0 - 3.0 + 0.5)).max() < 1e-12
    assert np.abs(orc.divergence(xf, yf, zf, (D_, D_, D_), u, v, w, scale=4.0) - 4.0 * d).max() < 1e-12
    # each direction alone, and only that direction's array matters
    assert np.abs(orc.divergence(xf, yf, zf, (D_, D_, D_), u, 0 * v, 0 * w) - 2.0).max() < 1e-12
    assert np.abs(orc.divergence(xf, yf, zf, (D_, D_, D_), 0 * u, v, 0 * w) + 3.0).max() < 1e-12
    assert np.abs(orc.divergence(xf, yf, zf, (D_, D_, D_), 0 * u, 0 * v, w) - 0.5).max() < 1e-12


def test_gradient_of_polynomials_on_interior_faces_and_boundary_closures(orc):
    xf, yf, zf = _grid()
    xc, yc, zc = _centres(xf), _centres(yf), _centres(zf)
    phi = (xc[None, None, :] ** 2) + 3.0 * yc[None, :, None] - 2.0 * zc[:, None, None] ** 2
    gu, gv, gw = orc.gradient(xf, yf, zf, (N_, D_, P_), phi)
    # interior faces: the divided difference of x^2 is the sum of the two centres; of a linear function its slope
    assert np.abs(gu[:, :, 1:-1] - (xc[1:] + xc[:-1])[None, None, :]).max() < 1e-12
    assert np.abs(gv[:, 1:-1, :] - 3.0).max() < 1e-12
    assert np.abs(gw[1:-1] + 2.0 * (zc[1:] + zc[:-1])[:, None, None]).max() < 1e-11
    # Neumann faces: zero.  Dirichlet faces: ghost value -phi at distance w.  Periodic: the wrap-around difference.
    assert np.all(gu[:, :, 0] == 0.0) and np.all(gu[:, :, -1] == 0.0)
    wy = np.diff(yf)
    assert np.abs(gv[:, 0, :] - 2.0 * phi[:, 0, :] / wy[0]).max() < 1e-12
    assert np.abs(gv[:, -1, :] + 2.0 * phi[:, -1, :] / wy[-1]).max() < 1e-12
    wz = np.diff(zf)
    wrap = (phi[0] - phi[-1]) / (0.5 * (wz[0] + wz[-1]))
    assert np.abs(gw[0] - wrap).max() < 1e-12 and np.array_equal(gw[0], gw[-1])


@pytest.mark.parametrize("bc", list(itertools.product((N_, D_, P_), repeat=3))[::2])
def test_divergence_of_gradient_is_the_flux_form_laplacian(orc, bc):
    # L = D G must be the operator of Eq. 3 with the boundary rows of A3 / cyclic corners of P:102: compared with the
    # oracle's flux-form operator, which is itself pinned against brute force and closed forms
    xf, yf, zf = _grid()
    rng = np.random.default_rng(5)
    phi = rng.uniform(-1, 1, (zf.size - 1, yf.size - 1, xf.size - 1))
    gu, gv, gw = orc.gradient(xf, yf, zf, bc, phi)
    lap = orc.divergence(xf, yf, zf, bc, gu, gv, gw)
    ref = orc.apply_operator_flux(xf, yf, zf, bc, 0.0, phi)
    assert np.abs(lap - ref).max() <= 1e-12 * np.abs(ref).max()


@pytest.mark.parametrize("bc", [(N_, N_, N_), (N_, N_, D_), (P_, N_, D_), (D_, P_, N_), (P_, P_, P_)])
def test_summation_by_parts(orc, bc):
    # sum_cells V phi (D u) = - sum_faces (face volume) u (G phi): face volume = area x (centre spacing; half a cell
    # at a Dirichlet boundary face; the wrap spacing at a periodic one, counted once); Neumann boundary faces carry u = 0
    n = (7, 6, 5)
    xf, yf, zf = _grid(n)
    rng = np.random.default_rng(9)
    phi = rng.uniform(-1, 1, n[::-1])
    u, v, w = _random_velocity(orc, n, bc, 11)
    ws = [np.diff(f) for f in (xf, yf, zf)]

    def face_len(f, b):
        wd = np.diff(f)
        d = np.empty(f.size)
        d[1:-1] = np.diff(_centres(f))
        if b == D_:
            d[0], d[-1] = 0.5 * wd[0], 0.5 * wd[-1]
        elif b == P_:
            d[0], d[-1] = 0.5 * (wd[0] + wd[-1]), 0.0          # one face, stored twice
        else:
            d[0] = d[-1] = 0.0
        return d

    dx, dy, dz = (face_len(f, b) for f, b in zip((xf, yf, zf), bc))
    V = ws[2][:, None, None] * ws[1][None, :, None] * ws[0][None, None, :]
    lhs = (V * phi * orc.divergence(xf, yf, zf, bc, u, v, w)).sum()
    gu, gv, gw = orc.gradient(xf, yf, zf, bc, phi)
    rhs = -((ws[2][:, None, None] * ws[1][None, :, None] * dx[None, None, :]) * u * gu).sum()
    rhs -= ((ws[2][:, None, None] * dy[None, :, None] * ws[0][None, None, :]) * v * gv).sum()
    rhs -= ((dz[:, None, None] * ws[1][None, :, None] * ws[0][None, None, :]) * w * gw).sum()
    assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), 1.0)


@pytest.mark.parametrize("bc", [(N_, N_, N_), (N_, N_, D_), (P_, N_, N_), (P_, P_, D_), (N_, D_, P_), (P_, P_, P_)])
def test_projection_of_white_noise_is_divergence_free(orc, bc):
    # "Applying the pressure-projection step to a white-noise velocity field likewise produces a discretely
    # divergence-free field to machine precision"
    n = (24, 20, 18)
    xf, yf, zf = _grid(n, beta=(2.0, 2.0, 2.5))
    plan = orc.OraclePlan(xf, yf, zf, bc, 0.0)
    u, v, w = _random_velocity(orc, n, bc, 21)
    c = 0.37
    un, vn, wn, phi, _ = orc.project(plan, c, u, v, w)
    d0 = orc.divergence(xf, yf, zf, bc, u, v, w)
    d1 = orc.divergence(xf, yf, zf, bc, un, vn, wn)
    assert np.abs(d1).max() <= 1e-11 * np.abs(d0).max()
    # the correction is exactly -c G phi, and phi solves Eq. 2c
    gu, gv, gw = orc.gradient(xf, yf, zf, bc, phi)
    assert np.abs((un - u) + c * gu)[:, :, :-1].max() < 1e-14 * np.abs(c * gu).max()
    assert np.abs((wn - w) + c * gw)[:-1].max() < 1e-14 * np.abs(c * gw).max()     # (a periodic duplicate face is rewritten)
    r = orc.residual_norms(xf, yf, zf, bc, 0.0, d0 / c, phi)
    assert r["relL2vol"] <= 1e-11
    # wall faces keep their prescribed value; periodic duplicates stay equal
    if bc[0] == N_:
        assert np.all(un[:, :, 0] == 0.0) and np.all(un[:, :, -1] == 0.0)
    if bc[0] == P_:
        assert np.array_equal(un[:, :, 0], un[:, :, -1])
    if bc[2] == P_:
        assert np.array_equal(wn[0], wn[-1])
    # projecting twice changes nothing (idempotent up to round-off)
    u2, v2, w2, phi2, _ = orc.project(plan, c, un, vn, wn)
    assert max(np.abs(u2 - un).max(), np.abs(v2 - vn).max(), np.abs(w2 - wn).max()) <= 1e-10 * np.abs(u).max()


def test_projection_removes_a_pure_gradient_and_returns_its_potential(orc):
    n = (20, 16, 12)
    bc = (N_, N_, N_)
    xf, yf, zf = _grid(n, beta=(2.0, 1.5, 2.0))
    plan = orc.OraclePlan(xf, yf, zf, bc, 0.0)
    xc, yc, zc = _centres(xf), _centres(yf), _centres(zf)
    psi = np.cos(np.pi * xc)[None, None, :] * np.cos(np.pi * yc / 2.0)[None, :, None] + zc[:, None, None] ** 2
    u, v, w = orc.gradient(xf, yf, zf, bc, psi)
    c = 2.5
    un, vn, wn, phi, _ = orc.project(plan, c, u, v, w)
    scale = max(np.abs(u).max(), np.abs(v).max(), np.abs(w).max())
    assert max(np.abs(un).max(), np.abs(vn).max(), np.abs(wn).max()) <= 1e-10 * scale
    V = np.diff(zf)[:, None, None] * np.diff(yf)[None, :, None] * np.diff(xf)[None, None, :]
    psi0 = psi - (V * psi).sum() / V.sum()                      # the solver's gauge: zero volume-weighted mean
    assert np.abs(c * phi - psi0).max() <= 1e-10 * np.abs(psi0).max()


@pytest.mark.parametrize("dirs_name", ["xyz", "yz", "z"])
def test_pressure_update_eq_2e(orc, dirs_name):
    n = (12, 10, 14)
    bc = (N_, N_, D_)
    dirs = {"xyz": orc.DIRS_XYZ, "yz": orc.DIRS_YZ, "z": orc.DIRS_Z}[dirs_name]
    xf, yf, zf = _grid(n)
    plan = orc.OraclePlan(xf, yf, zf, bc, 0.0)
    u, v, w = _random_velocity(orc, n, bc, 3)
    rng = np.random.default_rng(4)
    p0 = rng.uniform(-1, 1, n[::-1])
    c, alpha_p = 0.8, 3e-3
    _, _, _, phi, p1 = orc.project(plan, c, u, v, w, p=p0, alpha_p=alpha_p, dirs=dirs)
    # P^{k+1/2} = P^{k-1/2} + Phi - alpha L_I Phi, with the pinned flux-form operator (I - alpha L_I)
    ref = p0 + orc.apply_operator_flux(xf, yf, zf, bc, alpha_p, phi, dirs=dirs)
    assert np.abs(p1 - ref).max() <= 1e-13 * np.abs(ref).max()
    if dirs == orc.DIRS_XYZ:      # L Phi is the right-hand side of Eq. 2c
        rhs = orc.divergence(xf, yf, zf, bc, u, v, w, scale=1.0 / c)
        assert np.abs(p1 - (p0 + phi - alpha_p * rhs)).max() <= 1e-9 * np.abs(p1).max()
    # alpha_p = 0 (fully explicit diffusion, L_I = 0): P += Phi
    _, _, _, phi0, p2 = orc.project(plan, c, u, v, w, p=p0, alpha_p=0.0)
    assert np.array_equal(p2, p0 + phi0)
