"""GPU parity tests of the small-grid execution path (BASELINE.json configs[0]): the whole solve —
steps 2.1-2.5 of PAPER.md:181-185 and the gauge of PAPER.md:219 — as ONE cluster launch (csrc/fused_small.cu), against the
CPU oracle and against the five separate kernels."""
import numpy as np
import pytest

from paper_2603_09528_b200 import inputs as I

pytestmark = pytest.mark.gpu

PARITY_TOL = 1e-10
RESID_TOL = 1e-11
N_, D_, P_ = I.NEUMANN, I.DIRICHLET, I.PERIODIC


@pytest.fixture(scope="module")
def torch():
    import torch

    assert torch.cuda.is_available(), "these tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def tpt(torch):
    from paper_2603_09528_b200 import api

    api.lib()
    return api


def _rel(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


CASES = [
    # name, n, L, beta, bc, alpha                                              what it exercises
    ("c1-like", (16, 16, 16), (1.0, 1.0, 1.0), (1.2, 1.2, 1.5), (N_, N_, D_), 0.0),      # cluster of 8, two planes each
    ("limit-singular", (32, 32, 16), (1.0, 1.0, 1.0), (2.0, 2.0, 2.0), (N_, N_, N_), 0.0),    # the size limit (16384 points); gauge
    ("odd", (5, 7, 6), (1.0, 2.0, 1.5), (1.2, 2.0, 1.0), (N_, D_, D_), 0.0),             # ragged register tiles, cluster of 4
    ("ragged-z", (24, 20, 13), (1.0, 1.0, 2.0), (2.0, 1.5, 2.5), (D_, N_, N_), 0.0),     # 13 planes over 8 CTAs: one idle
    ("flat", (64, 48, 3), (2.0, 1.0, 1.0), (1.0, 2.0, 1.0), (N_, N_, D_), 0.0),          # cluster of 2
    ("two-planes", (10, 12, 2), (1.0, 1.0, 1.0), (1.0, 1.0, 0.0), (N_, N_, N_), 0.0),    # singular, cluster of 2
    ("helmholtz", (20, 28, 28), (1.0, 1.0, 1.0), (3.0, 3.0, 3.0), (N_, N_, D_), 5e-4),   # -1/alpha folded into the matrices
    ("periodic", (32, 16, 24), (2.0, 1.0, 1.0), (0.0, 2.0, 2.0), (P_, N_, N_), 0.0),     # dense cyclic basis, singular
    ("tall", (8, 8, 256), (1.0, 1.0, 4.0), (1.0, 1.0, 3.0), (N_, D_, N_), 0.0),          # long columns, 8 per CTA
]


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_fused_small_parity(tpt, torch, orc, case):
    name, n, L, beta, bc, alpha = case
    P = I.Problem(name, n, L, beta, bc, alpha, seed=17 + n[2])
    xf, yf, zf = P.faces()
    f = P.rhs()
    plan = tpt.plan_create(*n, xf, yf, zf, bc, alpha)
    paths = plan.paths()
    assert paths == [tpt.PATH_FUSED_SMALL] * 5
    d_f = torch.from_numpy(f).cuda()
    d_o = torch.empty_like(d_f)
    plan.solve(d_f, d_o)
    torch.cuda.synchronize()
    assert plan.launches_last() == 1
    phi = d_o.cpu().numpy()
    ref = orc.OraclePlan(xf, yf, zf, bc, alpha).solve(f)
    assert plan.singular == P.singular
    assert _rel(phi, ref) <= PARITY_TOL
    r = orc.residual_norms(xf, yf, zf, bc, alpha, f, phi)
    assert r["rel2"] <= RESID_TOL and r["relL2vol"] <= RESID_TOL
    if P.singular:      # gauge: zero volume-weighted mean (A7)
        V = np.diff(zf)[:, None, None] * np.diff(yf)[None, :, None] * np.diff(xf)[None, None, :]
        assert abs((V * phi).sum()) <= 1e-13 * np.abs(phi).max() * V.sum()
    # in place, and repeated (the workspace and the shared-memory buffers are reused)
    for _ in range(2):
        d_g = torch.from_numpy(f).cuda()
        plan.solve(d_g, d_g)
        torch.cuda.synchronize()
        assert np.array_equal(d_g.cpu().numpy(), phi)
    # the five separate kernels: same result to rounding (different summation order)
    plan.set_fused_small(False)
    assert tpt.PATH_FUSED_SMALL not in plan.paths()
    plan.solve(d_f, d_o)
    torch.cuda.synchronize()
    assert plan.launches_last() >= 5
    assert _rel(d_o.cpu().numpy(), phi) <= 1e-11
    plan.destroy()


@pytest.mark.parametrize("dirs_name", ["yz", "xyz"])
def test_fused_small_partial_dirs_and_batch(tpt, torch, orc, dirs_name):
    dirs = {"yz": tpt.DIRS_YZ, "xyz": tpt.DIRS_XYZ}[dirs_name]
    P = I.Problem("pd", (24, 16, 20), (1.0, 1.0, 1.0), (2.0, 1.5, 2.0), (N_, N_, D_), 2e-3, 9)
    xf, yf, zf = P.faces()
    plan = tpt.plan_create(*P.n, xf, yf, zf, P.bc, P.alpha, dirs=dirs)
    assert tpt.PATH_FUSED_SMALL in plan.paths()
    oplan = orc.OraclePlan(xf, yf, zf, P.bc, P.alpha, dirs=dirs)
    nrhs = 3
    F = np.stack([I.uniform_pm1(100 + q, P.points).reshape(P.n[::-1]) for q in range(nrhs)])
    plan.reserve_batch(nrhs)
    d_F = torch.from_numpy(F).cuda()
    d_O = torch.empty_like(d_F)
    plan.solve_batch(d_F, d_O)
    torch.cuda.synchronize()
    assert plan.launches_last() == nrhs
    out = d_O.cpu().numpy()
    for q in range(nrhs):
        assert _rel(out[q], oplan.solve(F[q])) <= PARITY_TOL
    plan.destroy()


def test_fused_small_limits(tpt, torch):
    # above 16384 points, with a fast transform, or with a non-default kernel variant: the separate kernels
    P = I.Problem("big", (32, 32, 20), (1.0, 1.0, 1.0), (1.0, 1.0, 1.0), (N_, N_, D_), 0.0, 1)
    xf, yf, zf = P.faces()
    plan = tpt.plan_create(*P.n, xf, yf, zf, P.bc, 0.0)
    assert tpt.PATH_FUSED_SMALL not in plan.paths()
    plan.destroy()
    P = I.Problem("u", (32, 16, 16), (1.0, 1.0, 1.0), (0.0, 1.0, 1.0), (N_, N_, D_), 0.0, 1)
    xf, yf, zf = P.faces()
    plan = tpt.plan_create(*P.n, xf, yf, zf, P.bc, 0.0, transform=(tpt.TRANSFORM_FFT, tpt.TRANSFORM_GEMM))
    assert plan.paths()[tpt.K_FWD_X] == tpt.PATH_FFT
    plan.destroy()
    plan = tpt.plan_create(*P.n, xf, yf, zf, P.bc, 0.0)
    assert plan.paths() == [tpt.PATH_FUSED_SMALL] * 5
    plan.set_gemm_variant(0)
    assert tpt.PATH_FUSED_SMALL not in plan.paths()
    plan.set_gemm_variant(2)
    plan.set_thomas_variant(0)
    assert tpt.PATH_FUSED_SMALL not in plan.paths()
    plan.destroy()
