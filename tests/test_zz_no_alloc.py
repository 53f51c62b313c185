"""GPU test of tpt_solve_static_scratch (include/tpt.h): the one-launch solve (steps 2.1-2.5 of PAPER.md:181-185 + the
gauge of PAPER.md:219) with its scratch in a static device array, for callers that may not call cudaMalloc.

Checked against the existing path (tpt_solve on the same plan, which uses the plan's workspace) on two calls in a row —
the second call finds the first call's contents in the shared array — and against the five separate kernels within the
parity tolerance of the other GPU tests.  Collected last on purpose (pytest -x: a failure here hides nothing)."""
import numpy as np
import pytest

from paper_2603_09528_b200 import inputs as I

pytestmark = pytest.mark.gpu

PARITY_TOL = 1e-10      # the tolerance of tests/test_gpu_fused_small.py and tests/test_gpu_parity.py
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
    # name, n, L, beta, bc, alpha
    ("c1", (16, 16, 16), (1.0, 1.0, 1.0), (1.2, 1.2, 1.5), (N_, N_, D_), 0.0),               # BASELINE.json configs[0]
    ("limit-singular", (32, 32, 16), (1.0, 1.0, 1.0), (2.0, 2.0, 2.0), (N_, N_, N_), 0.0),   # exactly the maximum; gauge
    ("odd-helmholtz", (5, 7, 6), (1.0, 2.0, 1.5), (0.0, 2.0, 1.0), (P_, D_, D_), 5e-4),      # ragged tiles, cluster of 4
]


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_static_scratch_matches_existing_path_twice(tpt, torch, case):
    name, n, L, beta, bc, alpha = case
    xf, yf, zf = I.Problem(name, n, L, beta, bc, alpha, seed=5).faces()
    plan = tpt.plan_create(*n, xf, yf, zf, bc, alpha)
    assert plan.points <= tpt.STATIC_SCRATCH_POINTS
    for call, seed in enumerate((31, 32)):      # two calls in a row, different right-hand sides
        f = I.Problem(name, n, L, beta, bc, alpha, seed=seed).rhs()
        d_f = torch.from_numpy(f).cuda()
        # existing path: tpt_solve with the plan's own workspace (the same kernel) ...
        plan.set_fused_small(True)
        d_ref = torch.empty_like(d_f)
        plan.solve(d_f, d_ref)
        torch.cuda.synchronize()
        assert plan.paths() == [tpt.PATH_FUSED_SMALL] * 5
        # ... and the five separate kernels
        plan.set_fused_small(False)
        d_sep = torch.empty_like(d_f)
        plan.solve(d_f, d_sep)
        torch.cuda.synchronize()
        assert plan.launches_last() > 1
        # the new entry point: out of place, then in place
        d_o = torch.full_like(d_f, float("nan"))
        plan.solve_static_scratch(d_f, d_o)
        torch.cuda.synchronize()
        assert plan.launches_last() == 1
        ref, sep, got = d_ref.cpu().numpy(), d_sep.cpu().numpy(), d_o.cpu().numpy()
        assert np.isfinite(got).all()
        assert _rel(got, ref) <= PARITY_TOL and _rel(got, sep) <= PARITY_TOL, (name, call)
        assert np.array_equal(got, ref), (name, call)      # same kernel, same arithmetic: bitwise
        d_g = d_f.clone()
        plan.solve_static_scratch(d_g, d_g)
        torch.cuda.synchronize()
        assert np.array_equal(d_g.cpu().numpy(), ref), (name, call)


def test_static_scratch_on_a_side_stream(tpt, torch):
    name, n, L, beta, bc, alpha = CASES[0]
    P = I.Problem(name, n, L, beta, bc, alpha, seed=77)
    xf, yf, zf = P.faces()
    plan = tpt.plan_create(*n, xf, yf, zf, bc, alpha)
    d_f = torch.from_numpy(P.rhs()).cuda()
    d_ref = torch.empty_like(d_f)
    plan.solve(d_f, d_ref)
    torch.cuda.synchronize()
    st = torch.cuda.Stream()
    d_o = torch.empty_like(d_f)
    with torch.cuda.stream(st):
        for _ in range(3):                      # back to back on one stream: ordered, no race on the shared array
            plan.solve_static_scratch(d_f, d_o, stream=st)
    st.synchronize()
    assert np.array_equal(d_o.cpu().numpy(), d_ref.cpu().numpy())


def test_static_scratch_limits(tpt, torch):
    def plan_of(n, bc=(N_, N_, D_), beta=(1.0, 1.0, 1.0), alpha=0.0, **kw):
        xf, yf, zf = I.Problem("lim", n, (1.0, 1.0, 1.0), beta, bc, alpha, seed=1).faces()
        return tpt.plan_create(*n, xf, yf, zf, bc, alpha, **kw)

    # one point beyond the maximum (16384): a clear error, nothing launched, the output untouched
    big = plan_of((32, 32, 17))
    assert big.points > tpt.STATIC_SCRATCH_POINTS
    d_f = torch.ones(big.points, dtype=torch.float64, device="cuda")
    d_o = torch.full_like(d_f, -7.0)
    with pytest.raises(tpt.TptError) as err:
        big.solve_static_scratch(d_f, d_o)
    assert err.value.status == tpt.ELIMIT
    assert "TPT_STATIC_SCRATCH_POINTS" in tpt.strerror(tpt.ELIMIT)
    torch.cuda.synchronize()
    assert bool((d_o == -7.0).all())
    big.solve(d_f, d_o)                          # the ordinary path still takes that grid
    torch.cuda.synchronize()
    # plans the one-launch kernel does not compute: periodic z, sweep-only (Eq. 2b with x, y explicit: alpha > 0)
    for plan in (plan_of((16, 16, 16), bc=(N_, N_, P_), beta=(1.0, 1.0, 0.0)), plan_of((16, 16, 16), alpha=1e-3, dirs=tpt.DIRS_Z)):
        d_f = torch.ones(plan.points, dtype=torch.float64, device="cuda")
        with pytest.raises(tpt.TptError) as err:
            plan.solve_static_scratch(d_f, torch.empty_like(d_f))
        assert err.value.status == -1            # TPT_EINVAL
