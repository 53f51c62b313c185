"""Host-side model of the product's periodic-z sweep (A19; "periodic boundaries also introduce cyclic
corner entries"): csrc/api.cu modifies the corners of T_z at plan time so that the ordinary tridiagonal sweep solves
A' = A - u v^T, sweeps q = A'^{-1} u once per plan, and csrc/kernels.cu (cyclic_rden / cyclic_correct) puts the rank-one
term back after every solve (Sherman-Morrison):

    g = -b_0,  r = a_0 / g,  b'_0 = b_0 - g,  b'_{n-1} = b_{n-1} - c_{n-1} a_0 / g,  a'_0 = c'_{n-1} = 0,
    u = (g, 0, .., 0, c_{n-1}),   x = y - q (y_0 + r y_{n-1}) / (1 + q_0 + r q_{n-1}),   A' y = p,  A' q = u.

The formulas are restated here in numpy (test code only) and checked against dense solves of the cyclic matrix, so the
plan-time algebra is pinned without a GPU: the splitting reproduces A exactly, g = -b_0 keeps A' diagonally dominant for every
spectral shift s <= 0 (no pivoting in the sweep), the denominator stays away from zero for every non-null column, and the
null column of a singular plan — unmodified diagonal, last unknown = 0 — satisfies every other equation."""
import numpy as np
import pytest


def _periodic_operator(n, rng, stretch):
    """Periodic finite-volume 1-D Laplacian (Eq. 3-4 with the wrap face): a_0 couples to x_{n-1}, c_{n-1} to x_0."""
    dz = 1.0 + stretch * rng.uniform(-0.5, 0.5, n)
    dz /= dz.sum()
    dc = 0.5 * (dz + np.roll(dz, 1))                    # dc[k]: spacing between the centres of cells k-1 and k (wraps at 0)
    a = 1.0 / (dz * dc)
    c = 1.0 / (dz * np.roll(dc, -1))
    return a, -(a + c), c, dz


def _cyclic_dense(a, b, c, s):
    n = len(b)
    A = np.diag(b + s) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
    A[0, n - 1] += a[0]
    A[n - 1, 0] += c[n - 1]
    return A


def _plan_split(a, b, c):
    """What tpt_plan_create does to (a, b, c) for a periodic z: the tridiagonal A' and the rank-one data."""
    n = len(b)
    g = -b[0]
    cn = c[n - 1]
    r = a[0] / g
    a2, b2, c2 = a.copy(), b.copy(), c.copy()
    b2[0] -= g
    b2[n - 1] -= cn * a[0] / g
    a2[0] = 0.0
    c2[n - 1] = 0.0
    return a2, b2, c2, g, cn, r


def _tridiag(a, b, c, s):
    return np.diag(b + s) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)


@pytest.mark.parametrize("n,stretch", [(3, 0.0), (4, 0.5), (16, 0.0), (33, 0.8), (128, 0.5)])
def test_sherman_morrison_split_reproduces_the_cyclic_solve(n, stretch):
    rng = np.random.default_rng(n)
    a, b, c, _ = _periodic_operator(n, rng, stretch)
    a2, b2, c2, g, cn, r = _plan_split(a, b, c)
    u = np.zeros(n); u[0] = g; u[n - 1] = cn
    v = np.zeros(n); v[0] = 1.0; v[n - 1] = r
    scale = np.abs(b).max()
    for s in (-1e-6 * scale, -1e-2 * scale, -0.7 * scale, -30.0 * scale):          # lam_x + lam_y of a non-null column: < 0
        A = _cyclic_dense(a, b, c, s)
        Ap = _tridiag(a2, b2, c2, s)
        assert np.abs(Ap + np.outer(u, v) - A).max() <= 1e-13 * scale                # A = A' + u v^T, entry by entry
        # A' stays strictly diagonally dominant by rows: the sweep needs no pivoting (A13)
        off = np.abs(Ap).sum(axis=1) - np.abs(np.diag(Ap))
        assert np.all(np.abs(np.diag(Ap)) > off)
        q = np.linalg.solve(Ap, u)                                                   # plan time: cyclic_rhs + sweep
        den = 1.0 + q[0] + r * q[n - 1]                                              # cyclic_rden
        assert abs(den) > 1e-8
        p = rng.uniform(-1, 1, n)
        y = np.linalg.solve(Ap, p)                                                   # per solve: the ordinary sweep
        x = y - q * (y[0] + r * y[n - 1]) / den                                      # cyclic_correct
        ref = np.linalg.solve(A, p)
        assert np.abs(x - ref).max() <= 1e-10 * np.abs(ref).max(), (n, s)


@pytest.mark.parametrize("n,stretch", [(4, 0.3), (32, 0.0), (65, 0.8)])
def test_null_column_of_a_periodic_plan(n, stretch):
    # s = 0: the cyclic matrix is singular (constants).  The product sweeps the null column with the UNMODIFIED diagonal and
    # the last equation replaced by x_{n-1} = 0 (both corner couplings then vanish), applies no correction (rden = 0) and
    # removes the dz-weighted mean afterwards.
    rng = np.random.default_rng(100 + n)
    a, b, c, dz = _periodic_operator(n, rng, stretch)
    A = _cyclic_dense(a, b, c, 0.0)
    x_true = rng.uniform(-1, 1, n)
    p = A @ x_true                                                                   # compatible right-hand side
    assert abs((dz * p).sum()) <= 1e-9 * np.abs(p).max()                             # (flux form: the weighted sum vanishes)
    T = _tridiag(a, b, c, 0.0)                                                       # corners dropped, diagonal as it is
    T[n - 1, :] = 0.0
    T[n - 1, n - 1] = -1.0                                                           # "-x = p" with p zeroed (thomas_onchip_tables)
    rhs = p.copy(); rhs[n - 1] = 0.0
    x = np.linalg.solve(T, rhs)
    assert x[n - 1] == 0.0
    assert np.abs((A @ x - p)[: n - 1]).max() <= 1e-9 * np.abs(p).max()              # every other equation of the CYCLIC system
    shift = x - x_true
    assert np.abs(shift - shift.mean()).max() <= 1e-8 * np.abs(x_true).max()         # a solution up to the constant
    x -= (dz * x).sum() / dz.sum()                                                   # the gauge (A7)
    assert abs((dz * x).sum()) <= 1e-14
