"""Pins for the oracle's partial implicit-diffusion variants: L_I = L_z ("z") and L_y + L_z ("yz").
Checked against brute force, a library tridiagonal/dense solve per line, and the limiting cases — never the CUDA path."""
import numpy as np
import pytest

from paper_2603_09528_b200 import inputs as I

N_, D_ = I.NEUMANN, I.DIRICHLET


def _rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


def _T(orc, xf, bc):
    w, a, b, c = orc.operator_1d(xf, bc)
    return np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)


@pytest.mark.parametrize("dirs_name", ["z", "yz", "xyz"])
@pytest.mark.parametrize("bc", [(N_, N_, D_), (D_, N_, N_), (N_, N_, N_)])
def test_partial_dirs_match_brute_force_lu(orc, dirs_name, bc):
    dirs = {"z": orc.DIRS_Z, "yz": orc.DIRS_YZ, "xyz": orc.DIRS_XYZ}[dirs_name]
    xf, yf, zf = I.tanh_faces(5, 1.0, 1.3), I.tanh_faces(7, 2.0, 1.8), I.tanh_faces(6, 0.5, 2.2)
    f = I.uniform_pm1(11, 5 * 7 * 6).reshape(6, 7, 5)
    alpha = 0.37
    u = orc.OraclePlan(xf, yf, zf, bc, alpha, dirs=dirs).solve(f)
    ref = orc.dense_solve_3d(xf, yf, zf, bc, alpha, f, dirs=dirs)
    assert _rel(u, ref) < 1e-12
    assert orc.residual_norms(xf, yf, zf, bc, alpha, f, u, dirs=dirs)["rel2"] < 1e-13


def test_z_only_is_one_tridiagonal_solve_per_line(orc):
    # "the z option performs only the tridiagonal solve": every (i,j) line is the 1-D system
    # (I - alpha T_z) u = f, solved here with the library's dense solver on the assembled T_z.
    xf, yf, zf = I.tanh_faces(4, 1.0, 0.0), I.tanh_faces(3, 1.0, 1.0), I.tanh_faces(24, 2.0, 2.5)
    f = I.uniform_pm1(5, 4 * 3 * 24).reshape(24, 3, 4)
    alpha = 2.5e-3
    u = orc.OraclePlan(xf, yf, zf, (N_, N_, D_), alpha, dirs=orc.DIRS_Z).solve(f)
    A = np.eye(24) - alpha * _T(orc, zf, D_)
    ref = np.linalg.solve(A, f.reshape(24, -1)).reshape(24, 3, 4)
    assert _rel(u, ref) < 1e-13


def test_yz_is_a_2d_helmholtz_solve_per_x_plane(orc):
    # "the yz option omits the x transforms": the x index is a pure batch index, so each x-plane solves
    # (I - alpha (T_y (+) T_z)) u = f, written here as a Kronecker sum and solved by the library.
    xf, yf, zf = I.tanh_faces(3, 1.0, 0.7), I.tanh_faces(6, 1.0, 1.5), I.tanh_faces(8, 1.0, 2.0)
    f = I.uniform_pm1(9, 3 * 6 * 8).reshape(8, 6, 3)
    alpha = 0.05
    u = orc.OraclePlan(xf, yf, zf, (D_, N_, D_), alpha, dirs=orc.DIRS_YZ).solve(f)
    Ty, Tz = _T(orc, yf, N_), _T(orc, zf, D_)
    A = np.eye(48) - alpha * (np.kron(Tz, np.eye(6)) + np.kron(np.eye(8), Ty))   # index = j + 6 k
    for i in range(3):
        ref = np.linalg.solve(A, f[:, :, i].reshape(-1)).reshape(8, 6)
        assert _rel(u[:, :, i], ref) < 1e-13


def test_partial_dirs_are_helmholtz_only_and_flux_operator_splits(orc):
    xf, yf, zf = I.tanh_faces(6, 1.0, 1.0), I.tanh_faces(5, 1.0, 1.0), I.tanh_faces(7, 1.0, 1.0)
    with pytest.raises(RuntimeError):
        orc.OraclePlan(xf, yf, zf, (N_, N_, D_), 0.0, dirs=orc.DIRS_YZ)     # Eq. 2c always carries the full Laplacian
    with pytest.raises(RuntimeError):
        orc.OraclePlan(xf, yf, zf, (N_, N_, D_), 0.1, dirs=5)
    # (I - aL) = (I - a L_yz) - a L_x:  the partial operators add up to the full one
    phi = I.uniform_pm1(3, 6 * 5 * 7).reshape(7, 5, 6)
    bc, a = (N_, D_, N_), 0.3
    full = orc.apply_operator_flux(xf, yf, zf, bc, a, phi)
    yz = orc.apply_operator_flux(xf, yf, zf, bc, a, phi, dirs=orc.DIRS_YZ)
    z = orc.apply_operator_flux(xf, yf, zf, bc, a, phi, dirs=orc.DIRS_Z)
    Tx, Ty = _T(orc, xf, bc[0]), _T(orc, yf, bc[1])
    assert np.allclose(yz - full, a * np.einsum("im,kjm->kji", Tx, phi), rtol=1e-12, atol=1e-12)
    assert np.allclose(z - yz, a * np.einsum("jm,kmi->kji", Ty, phi), rtol=1e-12, atol=1e-12)


def test_partial_dirs_on_a_stretched_config_residual(orc):
    # BASELINE configs[1]-like (Helmholtz, N,N,D), reduced to 32^3: round-off residual for each choice of L_I
    P = I.Problem("c2-32", (32, 32, 32), (2 * np.pi, np.pi, 2.0), (2.0, 2.0, 2.5), (N_, N_, D_), 1e-3, 1)
    xf, yf, zf = P.faces()
    f = P.rhs()
    sols = {}
    for dirs in (orc.DIRS_Z, orc.DIRS_YZ, orc.DIRS_XYZ):
        u = orc.OraclePlan(xf, yf, zf, P.bc, P.alpha, dirs=dirs).solve(f)
        assert orc.residual_norms(xf, yf, zf, P.bc, P.alpha, f, u, dirs=dirs)["rel2"] < 1e-13
        sols[dirs] = u
    # the three are different problems: their solutions differ at O(alpha |L_x u|)
    assert _rel(sols[orc.DIRS_Z], sols[orc.DIRS_XYZ]) > 1e-4
