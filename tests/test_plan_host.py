"""Host-only tests of the plan-time eigen-solver (csrc/plan_host.cpp) through tpt_host_eigen: no device, no oracle.
The accuracy rule of SURVEY 8(c.5) / DESIGN.md A9 says: ANY base solver followed by two guarded factored-form refinement
steps reaches forward errors ~1e-13 — so a deliberately crude base solver (normwise deflation, 64x looser: what a merely
backward-stable solver such as the paper's xSTEDC, delivers) must land on the same eigenpairs."""
import math

import numpy as np
import pytest

from paper_2603_09528_b200 import api
from paper_2603_09528_b200 import inputs as I


def _isolated(lam, tol=1e-6):
    gap = np.abs(np.diff(lam))
    left = np.concatenate([[np.inf], gap])
    right = np.concatenate([gap, [np.inf]])
    return np.minimum(left, right) > tol * np.maximum(np.abs(lam), 1e-300)


def _sym_tridiag(xf, bc):
    """T~ = D^{1/2} T D^{-1/2} (Eq. 5) assembled densely from the faces with the rows of reading A3."""
    w = np.diff(xf)
    n = w.size
    xc = 0.5 * (xf[1:] + xf[:-1])
    delta = np.concatenate([[w[0]], np.diff(xc), [w[-1]]])
    a, c = 1.0 / (w * delta[:-1]), 1.0 / (w * delta[1:])
    b = -(a + c)
    if bc == I.NEUMANN:
        b[0] += a[0]; b[-1] += c[-1]
    else:
        b[0] -= a[0]; b[-1] -= c[-1]
    S = np.diag(b)
    off = 1.0 / (delta[1:-1] * np.sqrt(w[:-1] * w[1:]))
    S += np.diag(off, 1) + np.diag(off, -1)
    return S


@pytest.mark.parametrize("n,beta,bc", [(192, 3.0, I.NEUMANN), (256, 2.0, I.DIRICHLET), (384, 3.0, I.NEUMANN)])
def test_crude_base_solver_lands_on_the_same_eigenpairs(n, beta, bc):
    xf = I.tanh_faces(n, 1.0, beta)
    lam0, q0 = api.host_eigen(xf, bc, base_kind=0)
    lam1, q1 = api.host_eigen(xf, bc, base_kind=1)
    S = _sym_tridiag(xf, bc)
    normS = np.abs(S).sum(axis=1).max()
    for lam, q in ((lam0, q0), (lam1, q1)):
        assert np.all(np.diff(lam) <= 0)                                        # descending, mode 0 smoothest
        assert np.abs(q.T @ q - np.eye(n)).max() < 1e-11 * n                    # accuracy rule: orthogonality defect after refinement
        assert np.abs(S @ q - q * lam[None, :]).max() <= 2e-15 * n * normS      # eigen-residual at rounding level (n eps ||T~||)
    iso = _isolated(lam0)
    iso[0] = bc != I.NEUMANN                                                    # the analytic null pair: lambda = 0 exactly
    assert iso.sum() > n // 5                                                   # the wall-mode pairs of the upper spectrum are near-degenerate (A14)
    # isolated eigenvalues (in particular the SMALL ones, which a normwise-stable solver alone gets only to
    # eps ||T~|| ~ 1e-8 relative on these grids) agree to 1e-12 relative between the two base solvers
    assert np.abs(lam1[iso] / lam0[iso] - 1.0).max() < 1e-12
    low = slice(1 if bc == I.NEUMANN else 0, 12)
    assert np.abs(lam1[low] / lam0[low] - 1.0).max() < 1e-13
    # ... and so do their eigenvectors (signs are fixed by the shared convention A6)
    assert np.abs(q1[:, :12] - q0[:, :12]).max() < 1e-10
    # lambda_1 -> -pi^2 (second order), the pin of SURVEY c.4 item 7
    k1 = 1 if bc == I.NEUMANN else 0
    assert abs(lam0[k1] + math.pi ** 2) < 50.0 / n ** 2 * math.pi ** 2


def test_host_eigen_rejects_bad_arguments():
    xf = I.tanh_faces(16, 1.0, 1.0)
    with pytest.raises(api.TptError):
        api.host_eigen(xf[::-1].copy(), 0)
    with pytest.raises(api.TptError):
        api.host_eigen(xf, 7)
    with pytest.raises(api.TptError):
        api.host_eigen(xf, 0, base_kind=3)
