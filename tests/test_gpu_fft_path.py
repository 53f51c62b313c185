"""GPU parity of the fast-transform path for uniform directions (the paper's FF / FG / GF
variants) against the CPU oracle, which knows nothing of FFTs: it eigen-solves the same operator with
Jacobi and applies dense transforms.  phi is unique, so both must agree whatever basis each side uses.
Grids use power-of-two lengths so that the face coordinates L i / N are exact and "uniform" holds bit for bit."""
import itertools

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


def _solve(torch, plan, f):
    d_f = torch.from_numpy(np.ascontiguousarray(f)).cuda()
    d_o = torch.empty_like(d_f)
    plan.solve(d_f, d_o)
    torch.cuda.synchronize()
    return d_o.cpu().numpy()


def _check(tpt, torch, orc, n, L, beta, bc, alpha, transform, seed=3):
    P = I.Problem("fft", n, L, beta, bc, alpha, seed)
    xf, yf, zf = P.faces()
    f = P.rhs()
    plan = tpt.plan_create(*n, xf, yf, zf, bc, alpha, transform=transform)
    phi = _solve(torch, plan, f)
    ref = orc.OraclePlan(xf, yf, zf, bc, alpha).solve(f)
    assert _rel(phi, ref) <= PARITY_TOL
    r = orc.residual_norms(xf, yf, zf, bc, alpha, f, phi)
    assert r["relL2vol"] <= RESID_TOL
    return plan, phi, (xf, yf, zf)


# every boundary type in each fast direction, both directions, several radix factorizations (16 = 4.4, 32 = 8.4,
# 64 = 8.8, 128 = 8.4.4, 256 = 8.8.4), ragged line counts (ny * nz not a multiple of the lines per CTA)
@pytest.mark.parametrize("bcx,bcy", list(itertools.product((N_, D_, P_), repeat=2)))
def test_ff_all_boundary_types(tpt, torch, orc, bcx, bcy):
    plan, _, _ = _check(tpt, torch, orc, (64, 32, 19), (2.0, 1.0, 1.0), (0.0, 0.0, 2.0), (bcx, bcy, D_), 0.0,
                        (tpt.TRANSFORM_FFT, tpt.TRANSFORM_FFT))
    plan.destroy()


@pytest.mark.parametrize("n,transform", [
    ((16, 128, 21), (1, 1)), ((128, 16, 24), (1, 1)), ((256, 64, 17), (1, 1)),
    ((128, 128, 40), (1, 0)),      # FG: fast x, stretched y through the TMA GEMM and the blocked layout
    ((128, 128, 40), (0, 1)),      # GF: stretched x, fast y
    ((64, 32, 600), (1, 1)),       # long columns: the fast y transform writes / reads the tile-blocked layout
    ((128, 64, 777), (0, 1)),      # the same with a stretched x through the GEMM
    ((40, 64, 33), (0, 1)),        # ragged stretched x (generic GEMM) ... nx % 16 != 0 is rejected below instead
])
def test_sizes_and_mixed_variants(tpt, torch, orc, n, transform):
    if n[0] % 16 and transform[1]:
        with pytest.raises(tpt.TptError):
            tpt.plan_create(*n, *I.Problem("x", n, (1.0, 1.0, 1.0), (2.0, 0.0, 2.0), (N_, N_, D_), 0.0, 1).faces(),
                            (N_, N_, D_), 0.0, transform=transform)
        return
    beta = (0.0 if transform[0] else 2.0, 0.0 if transform[1] else 1.5, 2.5)
    plan, _, _ = _check(tpt, torch, orc, n, (4.0, 1.0, 2.0), beta, (N_, N_, D_), 0.0, transform)
    plan.destroy()


def test_singular_and_helmholtz_and_paper_benchmark_bcs(tpt, torch, orc):
    # all-Neumann Poisson (gauge), Helmholtz (the -1/alpha scale rides in the forward-x scales), and the paper's
    # benchmark BCs: periodic x, Neumann y and z with uniform x, y and a stretched z
    for bc, alpha in (((N_, N_, N_), 0.0), ((N_, D_, N_), 2e-3), ((P_, N_, N_), 0.0)):
        plan, phi, (xf, yf, zf) = _check(tpt, torch, orc, (128, 64, 36), (8.0, 2.0, 1.0), (0.0, 0.0, 2.0), bc, alpha,
                                         (tpt.TRANSFORM_FFT, tpt.TRANSFORM_FFT))
        if alpha == 0.0:
            assert plan.singular
            V = np.diff(zf)[:, None, None] * np.diff(yf)[None, :, None] * np.diff(xf)[None, None, :]
            assert abs((V * phi).sum()) < 1e-13 * np.abs(phi).max() * V.sum()
        plan.destroy()


def test_fast_plan_equals_gemm_plan_and_reports_analytical_eigenvalues(tpt, torch):
    n, L = (256, 128, 48), (8.0, 2.0, 2.0)
    P = I.Problem("c4-like", n, L, (0.0, 0.0, 3.0), (N_, D_, D_), 0.0, 9)
    xf, yf, zf = P.faces()
    f = P.rhs()
    gg = tpt.plan_create(*n, xf, yf, zf, P.bc, 0.0)
    ff = tpt.plan_create(*n, xf, yf, zf, P.bc, 0.0, transform=(tpt.TRANSFORM_FFT, tpt.TRANSFORM_FFT))
    assert _rel(_solve(torch, ff, f), _solve(torch, gg, f)) <= 1e-11
    for d, (m, ln, bc) in enumerate(((n[0], L[0], N_), (n[1], L[1], D_))):
        lam = ff.eigenvalues(d)
        k = np.arange(m) + (1 if bc == D_ else 0)
        closed = -(4.0 / (ln / m) ** 2) * np.sin(np.pi * k / (2 * m)) ** 2          # BJ north_star closed form
        assert np.abs(lam - closed).max() <= 1e-13 * np.abs(closed).max()
        assert np.abs(lam - gg.eigenvalues(d)).max() <= 1e-11 * np.abs(closed).max()   # numerical eigen-solve agrees
        with pytest.raises(tpt.TptError):
            ff.eigen(d)                                                                # the basis is not stored
    # stage-wise: forward then inverse of one direction is the identity
    d_f = torch.from_numpy(f).cuda()
    a, b = torch.empty_like(d_f), torch.empty_like(d_f)
    for fwd, inv in ((tpt.K_FWD_X, tpt.K_INV_X), (tpt.K_FWD_Y, tpt.K_INV_Y)):
        ff.stage(fwd, d_f, a)
        ff.stage(inv, a, b)
        torch.cuda.synchronize()
        assert float((b - d_f).abs().max()) <= 1e-13
    gg.destroy()
    ff.destroy()


def test_fast_transform_is_refused_where_it_does_not_apply(tpt, torch):
    n = (64, 64, 16)
    P = I.Problem("bad", n, (1.0, 1.0, 1.0), (2.0, 0.0, 1.0), (N_, N_, D_), 1e-3, 1)
    xf, yf, zf = P.faces()
    with pytest.raises(tpt.TptError):      # x is stretched
        tpt.plan_create(*n, xf, yf, zf, P.bc, 0.0, transform=(1, 0))
    with pytest.raises(tpt.TptError):      # y is not diagonalised by a z-only plan
        tpt.plan_create(*n, xf, yf, zf, P.bc, 1e-3, dirs=tpt.DIRS_Z, transform=(0, 1))
    Q = I.Problem("bad2", (48, 64, 16), (1.0, 1.0, 1.0), (0.0, 0.0, 1.0), (N_, N_, D_), 0.0, 1)
    with pytest.raises(tpt.TptError):      # 48 is not a power of two
        tpt.plan_create(*Q.n, *Q.faces(), Q.bc, 0.0, transform=(1, 0))
    tpt.plan_create(*Q.n, *Q.faces(), Q.bc, 0.0, transform=(0, 1)).destroy()   # y = 64 uniform: fine


def test_c4_full_size_grids_fg_parity_and_residual(tpt, torch, orc):
    # BASELINE.json configs[3]: x is uniform with 1024 cells — here on the fast path (FG) instead of the GEMM
    P = I.CONFIGS["c4"][0].thin_z(16)
    xf, yf, zf = P.faces()
    f = P.rhs()
    plan = tpt.plan_create(*P.n, xf, yf, zf, P.bc, P.alpha, transform=(tpt.TRANSFORM_FFT, tpt.TRANSFORM_GEMM))
    phi = _solve(torch, plan, f)
    plan.destroy()
    assert _rel(phi, orc.OraclePlan(xf, yf, zf, P.bc, P.alpha).solve(f)) <= PARITY_TOL
    # full size: flux-form residual at round-off
    P = I.CONFIGS["c4"][0]
    xf, yf, zf = P.faces()
    f = P.rhs()
    plan = tpt.plan_create(*P.n, xf, yf, zf, P.bc, P.alpha, transform=(tpt.TRANSFORM_FFT, tpt.TRANSFORM_GEMM))
    phi = _solve(torch, plan, f)
    plan.destroy()
    r = orc.residual_norms(xf, yf, zf, P.bc, P.alpha, f, phi)
    assert r["rel2"] <= RESID_TOL and r["relL2vol"] <= RESID_TOL


@pytest.mark.parametrize("nz", [24, 600])
def test_batched_and_host_solves_on_fast_plans(tpt, torch, nz):
    # three stacked right-hand sides (one launch per x transform, per field on the blocked layout) and the slab-pipelined
    # host path give the same bits as single device solves
    P = I.Problem("ff-batch", (64, 32, nz), (2.0, 1.0, 1.0), (0.0, 0.0, 2.0), (P_, N_, D_), 1e-3, 21)
    xf, yf, zf = P.faces()
    plan = tpt.plan_create(*P.n, xf, yf, zf, P.bc, P.alpha, transform=(tpt.TRANSFORM_FFT, tpt.TRANSFORM_FFT))
    fs = np.stack([I.uniform_pm1(400 + r, P.points).reshape(P.n[::-1]) for r in range(3)])
    singles = np.stack([_solve(torch, plan, fs[r]) for r in range(3)])
    plan.reserve_batch(2)                       # chunks of 2 + 1
    d = torch.from_numpy(fs).cuda()
    plan.solve_batch(d, d)
    torch.cuda.synchronize()
    assert np.array_equal(d.cpu().numpy(), singles)
    out = np.empty_like(fs[0])
    plan.solve_host(fs[1], out)
    assert np.array_equal(out, singles[1])
    plan.destroy()


def test_long_y_lines_use_the_512_thread_tiles(tpt, torch, orc):
    # ny = 1024: 8-column tiles of 8192 samples, 512 threads per CTA (the y grid is c4's x grid, so the oracle's
    # 1024-point eigen-decomposition is shared with the c4 tests)
    P = I.Problem("ylong", (32, 1024, 6), (1.0, 8.0, 1.0), (1.5, 0.0, 2.0), (D_, N_, D_), 0.0, 17)
    xf, yf, zf = P.faces()
    f = P.rhs()
    plan = tpt.plan_create(*P.n, xf, yf, zf, P.bc, 0.0, transform=(tpt.TRANSFORM_GEMM, tpt.TRANSFORM_FFT))
    phi = _solve(torch, plan, f)
    plan.destroy()
    assert _rel(phi, orc.OraclePlan(xf, yf, zf, P.bc, 0.0).solve(f)) <= PARITY_TOL


@pytest.mark.parametrize("direction,bc", [(0, N_), (0, D_), (0, P_), (1, N_), (1, P_)])
def test_longest_lines_against_the_closed_form_basis(tpt, torch, direction, bc):
    # 2048-long lines (radices 8.8.8.4; x: one pair per CTA, y: 4-column tiles with 512 threads).  The oracle's Jacobi
    # would take minutes at this length, so the stage outputs are compared with the closed-form orthonormal bases
    # themselves (BJ north_star: DCT-II for Neumann; sine / Fourier for Dirichlet / periodic): p^ = sqrt(w) Q^T f.
    n = (2048, 16, 3) if direction == 0 else (16, 2048, 3)
    N, L = 2048, 4.0
    bcs = (bc, N_, D_) if direction == 0 else (N_, bc, D_)
    P = I.Problem("long", n, (L, 1.0, 1.0) if direction == 0 else (1.0, L, 1.0), (0.0, 0.0, 1.5), bcs, 0.0, 33)
    xf, yf, zf = P.faces()
    plan = tpt.plan_create(*n, xf, yf, zf, bcs, 0.0, transform=(tpt.TRANSFORM_FFT, tpt.TRANSFORM_FFT))
    i = np.arange(N)[:, None]
    s = np.arange(N)[None, :]
    if bc == N_:
        Q = np.cos(np.pi * s * (2 * i + 1) / (2 * N))
    elif bc == D_:
        Q = np.sin(np.pi * (s + 1) * (2 * i + 1) / (2 * N))
    else:
        j = (s + 1) // 2
        Q = np.where((s == 0) | (s % 2 == 1), np.cos(2 * np.pi * j * i / N), np.sin(2 * np.pi * j * i / N))
    Q = Q / np.linalg.norm(Q, axis=0)
    w = L / N
    f = P.rhs()
    d_f = torch.from_numpy(f).cuda()
    a, b = torch.empty_like(d_f), torch.empty_like(d_f)
    plan.stage(tpt.K_FWD_X if direction == 0 else tpt.K_FWD_Y, d_f, a)
    plan.stage(tpt.K_INV_X if direction == 0 else tpt.K_INV_Y, a, b)
    torch.cuda.synchronize()
    expect = np.sqrt(w) * (np.einsum("im,kji->kjm", Q, f) if direction == 0 else np.einsum("jm,kji->kmi", Q, f))
    assert np.abs(a.cpu().numpy() - expect).max() <= 1e-12 * np.abs(expect).max()
    assert float((b - d_f).abs().max()) <= 1e-12
    lam = plan.eigenvalues(direction)
    k = np.arange(N)
    arg = {N_: np.pi * k / (2 * N), D_: np.pi * (k + 1) / (2 * N), P_: np.pi * ((k + 1) // 2) / N}[bc]
    assert np.abs(lam + 4.0 / w**2 * np.sin(arg) ** 2).max() <= 1e-13 * 4.0 / w**2
    plan.destroy()


# --------------------------------------------------------------------------------------------------
# Slab pipeline of steps 2.2 -> 2.3 -> 2.4 (tpt_plan_set_slab_groups; BASELINE north_star "Fusion"):
# same kernels, same per-column arithmetic, another schedule — bit-for-bit the unslabbed solve.
# --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("case", [
    ("ff-singular", (64, 32, 48), (0.0, 0.0, 2.0), (N_, N_, N_), 0.0, ("f", "f"), 7),
    ("gf-helmholtz", (128, 64, 40), (2.0, 0.0, 2.5), (N_, D_, D_), 1e-3, ("g", "f"), 7),
    ("gg-tma", (256, 128, 24), (2.0, 2.0, 2.0), (N_, N_, D_), 0.0, ("g", "g"), 7),
    ("fg-periodic-x", (64, 96, 33), (0.0, 1.5, 2.0), (P_, N_, N_), 0.0, ("f", "g"), 7),
    ("yz-only", (48, 64, 20), (2.0, 0.0, 2.0), (N_, N_, D_), 5e-3, ("g", "f"), 6),
], ids=lambda c: c[0])
@pytest.mark.parametrize("groups", [1, 3])
def test_slab_pipeline_is_bitwise_the_plain_solve(tpt, torch, orc, case, groups):
    name, n, beta, bc, alpha, tr, dirs = case
    P = I.Problem(name, n, (1.0, 1.0, 1.0), beta, bc, alpha, seed=len(name))
    xf, yf, zf = P.faces()
    f = P.rhs()
    kind = {"g": tpt.TRANSFORM_GEMM, "f": tpt.TRANSFORM_FFT}
    plan = tpt.plan_create(*n, xf, yf, zf, bc, alpha, dirs=dirs, transform=(kind[tr[0]] if dirs & 1 else 0, kind[tr[1]]))
    assert plan.paths()[tpt.K_THOMAS] == tpt.PATH_THOMAS_BLOCKED
    d_f = torch.from_numpy(f).cuda()
    d_ref = torch.empty_like(d_f)
    plan.solve(d_f, d_ref)
    torch.cuda.synchronize()
    plain_launches = plan.launches_last()
    ref = orc.OraclePlan(xf, yf, zf, bc, alpha, dirs=dirs).solve(f)
    assert _rel(d_ref.cpu().numpy(), ref) <= PARITY_TOL
    plan.set_slab_groups(groups)
    nslabs = -(-(n[0] // 16) // groups)
    for inplace in (False, True):
        d_in = d_f.clone()
        d_out = d_in if inplace else torch.empty_like(d_f)
        plan.solve(d_in, d_out)
        torch.cuda.synchronize()
        assert plan.launches_last() == plain_launches - 3 + 3 * nslabs
        assert torch.equal(d_out, d_ref)
    # a batch runs the slabs field by field
    plan.reserve_batch(2)
    d_b = torch.stack([d_f, d_f])
    d_o = torch.empty_like(d_b)
    plan.solve_batch(d_b, d_o)
    torch.cuda.synchronize()
    assert torch.equal(d_o[0], d_ref) and torch.equal(d_o[1], d_ref)
    plan.set_slab_groups(0)
    plan.solve(d_f, d_o[0])
    assert plan.launches_last() == plain_launches
    plan.destroy()


def test_ff512_full_size_parity_in_the_bench_configuration(tpt, torch, orc):
    # the grid bench.py --config ff512 --transform ff times (512^3, uniform x, y, stretched z): every element against a
    # full oracle solve (the oracle knows no fast transform: its own eigen-solver and naive loops), residual and paths
    P = I.CONFIGS["ff512"][0]
    xf, yf, zf = P.faces()
    f = P.rhs()
    plan = tpt.plan_create(*P.n, xf, yf, zf, P.bc, P.alpha, transform=(tpt.TRANSFORM_FFT, tpt.TRANSFORM_FFT))
    assert plan.paths() == [tpt.PATH_FFT, tpt.PATH_FFT, tpt.PATH_THOMAS_BLOCKED, tpt.PATH_FFT, tpt.PATH_FFT]
    d_f = torch.from_numpy(f).cuda()
    d_o = torch.empty_like(d_f)
    plan.solve(d_f, d_o)
    torch.cuda.synchronize()
    phi = d_o.cpu().numpy()
    del d_f, d_o
    plan.destroy()
    r = orc.residual_norms(xf, yf, zf, P.bc, P.alpha, f, phi)
    assert r["rel2"] <= 1e-11 and r["relL2vol"] <= 1e-11
    ref = orc.OraclePlan(xf, yf, zf, P.bc, P.alpha).solve(f)
    assert _rel(phi, ref) <= PARITY_TOL
