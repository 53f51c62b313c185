"""GPU parity of the tile-blocked mode-space layout (csrc/kernels.cuh): between steps 2.2 and 2.4
the field is stored with the nz rows of every 16-column Thomas tile contiguous.  It is used whenever the TMA GEMM takes
the y transforms and the on-chip sweep takes step 2.3; these cases walk through every launch shape of the sweep
(segment length, tile width, CTAs per SM) and compare with the CPU oracle and with the natural-layout kernels."""
import numpy as np
import pytest

from paper_2603_09528_b200 import inputs as I

pytestmark = pytest.mark.gpu

PARITY_TOL = 1e-10
N_, D_ = I.NEUMANN, I.DIRICHLET


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


def _solve(torch, plan, f):
    d_f = torch.from_numpy(np.ascontiguousarray(f)).cuda()
    d_o = torch.empty_like(d_f)
    plan.solve(d_f, d_o)
    torch.cuda.synchronize()
    return d_o.cpu().numpy()


# nz picks the sweep's launch shape (thomas_onchip.cu, choose_shape): <=128: 8-row segments; <=256: 16 rows, two CTAs per SM;
# 257..800 (blocked): 17 / 19 / 21 / 23 / 25-row segments in 8-column tiles (two CTAs) or — 17 and 19 rows, segment count a
# multiple of 8 — 4-column tiles (four CTAs), with the coefficient table in shared memory where it fits; 801..1008: 21-row
# segments, one CTA per SM; 1009..1056: 17-row segments and 512 threads.  Ragged nz exercises the predicated / zero-filled
# tail rows.
SHAPES = [
    ("nz24", (128, 128, 24), (N_, N_, D_), 0.0),
    ("nz130", (128, 256, 130), (N_, N_, D_), 0.0),
    ("nz256", (256, 128, 256), (N_, D_, N_), 0.0),
    ("nz300", (128, 128, 300), (N_, N_, D_), 2e-3),
    ("nz384", (128, 128, 384), (N_, N_, D_), 0.0),              # 4-column tiles, 24 segments: table through L1
    ("nz500-singular", (128, 128, 500), (N_, N_, N_), 0.0),     # 4-column tiles, table in shared memory; null column from global
    ("nz512", (256, 128, 512), (N_, D_, D_), 1e-3),             # the bench shape (c3, c4)
    ("nz513-singular", (128, 128, 513), (N_, N_, N_), 0.0),
    ("nz576", (128, 128, 576), (D_, N_, N_), 0.0),              # 19-row segments, 4-column tiles
    ("nz616", (128, 128, 616), (N_, N_, D_), 0.0),              # 21-row segments, 8-column tiles, table in shared memory
    ("nz544", (128, 128, 544), (D_, N_, D_), 0.0),
    ("nz545", (128, 128, 545), (N_, N_, D_), 0.0),
    ("nz608", (128, 128, 608), (N_, N_, D_), 1e-3),
    ("nz650", (128, 128, 650), (N_, D_, D_), 0.0),
    ("nz700-singular", (128, 128, 700), (N_, N_, N_), 0.0),
    ("nz768", (128, 128, 768), (N_, N_, D_), 5e-4),
    ("nz800", (128, 128, 800), (D_, D_, N_), 0.0),
    ("nz801", (128, 128, 801), (N_, N_, D_), 0.0),
    ("nz1000", (128, 128, 1000), (N_, N_, D_), 0.0),
    ("nz1008-singular", (128, 128, 1008), (N_, N_, N_), 0.0),
    ("nz1009", (128, 128, 1009), (N_, D_, D_), 0.0),
    ("nz1056", (128, 128, 1056), (N_, D_, N_), 0.0),
]


@pytest.mark.parametrize("case", SHAPES, ids=[c[0] for c in SHAPES])
def test_blocked_layout_parity_across_sweep_shapes(tpt, torch, orc, case):
    name, n, bc, alpha = case
    P = I.Problem(name, n, (1.0, 2.0, 1.0), (2.0, 1.5, 2.5), bc, alpha, seed=77 + n[2])
    xf, yf, zf = P.faces()
    f = P.rhs()
    plan = tpt.plan_create(*P.n, xf, yf, zf, P.bc, P.alpha)
    phi = _solve(torch, plan, f)                    # TMA GEMM + on-chip sweep: blocked mode-space layout
    plan.set_thomas_variant(0)                      # streaming sweep: natural layout, same GEMM kernels
    phi_nat = _solve(torch, plan, f)
    plan.set_thomas_variant(1)
    plan.set_gemm_variant(1)                        # cp.async GEMM: natural layout, on-chip sweep
    phi_nat2 = _solve(torch, plan, f)
    plan.destroy()
    ref = orc.OraclePlan(xf, yf, zf, P.bc, P.alpha).solve(f)
    assert _rel(phi, ref) <= PARITY_TOL
    assert _rel(phi_nat, ref) <= PARITY_TOL and _rel(phi_nat2, ref) <= PARITY_TOL
    assert _rel(phi, phi_nat) <= 1e-11 and _rel(phi, phi_nat2) <= 1e-11
    if plan_singular(bc, alpha):
        V = np.diff(zf)[:, None, None] * np.diff(yf)[None, :, None] * np.diff(xf)[None, None, :]
        assert abs((V * phi).sum()) < 1e-13 * np.abs(phi).max() * V.sum()      # the gauge found column (0,0)


def plan_singular(bc, alpha):
    return alpha == 0.0 and all(b == N_ for b in bc)


def test_blocked_layout_yz_plan_and_batch(tpt, torch, orc):
    # yz plan: rhs -> (2.2, blocked) W -> sweep -> (2.4) out; batched fields keep one blocked field each
    P = I.Problem("blk-yz", (128, 128, 300), (1.0, 1.0, 1.0), (2.0, 2.0, 2.5), (N_, N_, D_), 1e-3, 12)
    xf, yf, zf = P.faces()
    for dirs in (tpt.DIRS_YZ, tpt.DIRS_XYZ):
        plan = tpt.plan_create(*P.n, xf, yf, zf, P.bc, P.alpha, dirs=dirs)
        fs = np.stack([I.uniform_pm1(300 + r, P.points).reshape(P.n[::-1]) for r in range(2)])
        singles = np.stack([_solve(torch, plan, fs[r]) for r in range(2)])
        plan.reserve_batch(2)
        d = torch.from_numpy(fs).cuda()
        plan.solve_batch(d, d)
        torch.cuda.synchronize()
        assert np.array_equal(d.cpu().numpy(), singles)
        ref = orc.OraclePlan(xf, yf, zf, P.bc, P.alpha, dirs=dirs).solve(fs[1])
        assert _rel(singles[1], ref) <= PARITY_TOL
        plan.destroy()
