"""Sharded solve (include/tpt.h "the solve sharded across the GPUs of one NVLink domain"; Algorithm 1
steps 2, 4, 6, 8 at PAPER.md:235-245) validated with VIRTUAL RANKS: P shards on one device whose peer pointers are plain
device pointers, phases ordered by the stream.  Same kernels, same addressing, same stores as P GPUs; only the
transport (NVLink) and the flag barriers differ — the barrier code is covered separately with P = 1 and with the P
virtual ranks' barriers run as the blocks of one cooperative launch.

Each rank's slab solution is compared element by element with the matching planes of the oracle's full-grid solve."""
import numpy as np
import pytest

from paper_2603_09528_b200 import inputs as I

pytestmark = pytest.mark.gpu

PARITY_TOL = 1e-10
RESID_TOL = 1e-11
N_, D_, PER_ = I.NEUMANN, I.DIRICHLET, I.PERIODIC


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


def _make_shards(tpt, P, nranks, transform_x=0, transform_y=0):
    xf, yf, zf = P.faces()
    shards = [tpt.shard_create(r, nranks, *P.n, xf, yf, zf, P.bc, P.alpha, transform_x, transform_y) for r in range(nranks)]
    syms = [s.sym()[0] for s in shards]
    for s in shards:
        s.set_peers(syms)
    return shards


def _split(torch, shards, f):
    nx, ny, nz = shards[0].nx, shards[0].ny, shards[0].nz
    f3 = f.reshape(nz, ny, nx)
    rhs = [torch.from_numpy(np.ascontiguousarray(f3[s.layout.k0:s.layout.k1])).cuda() for s in shards]
    out = [torch.empty_like(r) for r in rhs]
    return rhs, out


def _gather(shards, out):
    s0 = shards[0]
    return np.concatenate([o.cpu().numpy().reshape(-1) for o in out]).reshape(s0.nz, s0.ny, s0.nx)


CASES = [
    # name, n, L, beta, bc, alpha, ranks
    ("p2", (128, 128, 24), (1.0, 1.0, 1.0), (2.0, 2.0, 2.0), (N_, N_, D_), 0.0, 2),
    ("p2-sing", (128, 128, 40), (1.0, 1.0, 1.0), (2.0, 2.0, 2.0), (N_, N_, N_), 0.0, 2),
    ("p3-ragged", (256, 128, 35), (2.0, 1.0, 1.0), (2.5, 2.0, 3.0), (N_, D_, D_), 0.0, 3),      # 35 planes over 3 ranks, 8 units over 3
    ("p4-helm", (128, 256, 50), (1.0, 1.0, 1.0), (3.0, 3.0, 3.0), (N_, N_, D_), 5e-4, 4),
    ("p4-sing", (256, 256, 130), (1.0, 1.0, 1.0), (2.0, 2.0, 2.0), (N_, N_, N_), 0.0, 4),        # second sweep shape (nz > 128)
    ("p8", (128, 128, 66), (1.0, 2.0, 1.0), (2.0, 2.0, 2.5), (D_, N_, D_), 0.0, 8),              # one 16-row unit per rank
    ("p8-sing-tall", (128, 256, 300), (1.0, 1.0, 1.0), (2.0, 2.0, 3.0), (N_, N_, N_), 0.0, 8),
    ("p4-512", (128, 128, 512), (1.0, 1.0, 1.0), (2.0, 2.0, 2.5), (N_, N_, D_), 0.0, 4),        # 8-column tiles with the table in shared memory
    ("p2-576-sing", (128, 128, 576), (1.0, 1.0, 1.0), (2.0, 2.0, 2.0), (N_, N_, N_), 0.0, 2),   # 19-row segments
    ("p5-periodic", (128, 128, 21), (1.0, 1.0, 1.0), (0.0, 2.0, 2.0), (PER_, N_, D_), 0.0, 5),  # ragged: 21 planes, 5 ranks
    ("p1", (128, 128, 16), (1.0, 1.0, 1.0), (2.0, 2.0, 2.0), (N_, N_, D_), 0.0, 1),
]


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_virtual_rank_parity(tpt, torch, orc, case):
    name, n, L, beta, bc, alpha, nranks = case
    P = I.Problem(name, n, L, beta, bc, alpha, seed=100 + nranks)
    xf, yf, zf = P.faces()
    f = P.rhs()
    shards = _make_shards(tpt, P, nranks)
    # the slabs tile the grid, the mode rows tile ny
    assert [s.layout.k0 for s in shards][0] == 0 and shards[-1].layout.k1 == n[2]
    assert all(a.layout.k1 == b.layout.k0 and a.layout.m1 == b.layout.m0 for a, b in zip(shards, shards[1:]))
    assert shards[0].layout.m0 == 0 and shards[-1].layout.m1 == n[1]
    rhs, out = _split(torch, shards, f)
    tpt.virtual_ranks_solve(shards, rhs, out)
    torch.cuda.synchronize()
    phi = _gather(shards, out)
    ref = orc.OraclePlan(xf, yf, zf, bc, alpha).solve(f)
    assert float(np.abs(phi - ref).max() / np.abs(ref).max()) <= PARITY_TOL
    r = orc.residual_norms(xf, yf, zf, bc, alpha, f, phi)
    assert r["rel2"] <= RESID_TOL and r["relL2vol"] <= RESID_TOL
    # a second solve on the same shards (buffers are reused) gives the same bits, also in place
    tpt.virtual_ranks_solve(shards, rhs, rhs)
    torch.cuda.synchronize()
    assert np.array_equal(_gather(shards, rhs), phi)
    for s in shards:
        s.destroy()


def test_sharded_equals_single_gpu_solve_bitwise(tpt, torch):
    # the sharded path runs the same kernels on the same numbers in the same order per element: identical bits
    P = I.Problem("bits", (256, 128, 48), (1.0, 1.0, 1.0), (2.0, 2.0, 2.0), (N_, N_, N_), 0.0, seed=5)
    xf, yf, zf = P.faces()
    f = P.rhs()
    plan = tpt.plan_create(*P.n, xf, yf, zf, P.bc, P.alpha)
    d_f = torch.from_numpy(f).cuda()
    d_o = torch.empty_like(d_f)
    plan.solve(d_f, d_o)
    torch.cuda.synchronize()
    one = d_o.cpu().numpy()
    shards = _make_shards(tpt, P, 4)
    rhs, out = _split(torch, shards, f)
    tpt.virtual_ranks_solve(shards, rhs, out)
    torch.cuda.synchronize()
    assert np.array_equal(_gather(shards, out).reshape(-1), one.reshape(-1))
    plan.destroy()
    for s in shards:
        s.destroy()


def test_fast_x_transform_in_sharded_solve(tpt, torch, orc):
    # uniform x by the fast cosine transform, y by the GEMM that carries exchange 1
    P = I.Problem("fx", (256, 128, 30), (4.0, 1.0, 1.0), (0.0, 2.0, 2.5), (N_, N_, D_), 0.0, seed=9)
    xf, yf, zf = P.faces()
    f = P.rhs()
    shards = _make_shards(tpt, P, 3, transform_x=tpt.TRANSFORM_FFT)
    rhs, out = _split(torch, shards, f)
    tpt.virtual_ranks_solve(shards, rhs, out)
    torch.cuda.synchronize()
    ref = orc.OraclePlan(xf, yf, zf, P.bc, P.alpha).solve(f)
    phi = _gather(shards, out)
    assert float(np.abs(phi - ref).max() / np.abs(ref).max()) <= PARITY_TOL
    for s in shards:
        s.destroy()


def test_solve_sharded_with_device_barriers(tpt, torch, orc):
    # The flag barrier.  (a) tpt_solve_sharded itself with one rank (its barrier kernels wait on nothing but their own
    # flag).  (b) P = 2, 4, 8 virtual ranks: all ranks' barriers in ONE cooperative launch, block r acting as rank r —
    # kernels that wait on one another must not be separate launches on one GPU — between the phases of the solve, several
    # solves in a row (the epochs keep growing).
    P = I.Problem("bar", (128, 128, 32), (1.0, 1.0, 1.0), (2.0, 2.0, 2.0), (N_, N_, N_), 0.0, seed=3)
    xf, yf, zf = P.faces()
    f = P.rhs()
    ref = orc.OraclePlan(xf, yf, zf, P.bc, P.alpha).solve(f)
    shards = _make_shards(tpt, P, 1)
    rhs, out = _split(torch, shards, f)
    for _ in range(3):
        shards[0].solve(rhs[0], out[0])
    torch.cuda.synchronize()
    assert shards[0].launches() == 7          # 5 compute kernels + 2 barriers
    assert float(np.abs(_gather(shards, out) - ref).max() / np.abs(ref).max()) <= PARITY_TOL
    shards[0].destroy()
    for nranks in (2, 4, 8):
        shards = _make_shards(tpt, P, nranks)
        rhs, out = _split(torch, shards, f)
        for _ in range(3):
            tpt.virtual_ranks_solve(shards, rhs, out, barriers=True)
        torch.cuda.synchronize()
        assert float(np.abs(_gather(shards, out) - ref).max() / np.abs(ref).max()) <= PARITY_TOL
        for s in shards:
            s.destroy()


# The fast y transform carries exchange 1 from its own stores (every mode row written straight into its owner's buffer),
# the inverse reads the slab buffer: the GF and FF variants of PAPER.md:294 sharded — against the oracle, and bit-for-bit
# against the single-plan solve with the same transforms.
@pytest.mark.parametrize("case", [
    ("gf-p3", (128, 64, 30), (1.0, 2.0, 1.0), (2.0, 0.0, 2.5), (N_, D_, D_), 0.0, 3, (0, 1)),
    ("ff-p4-singular", (256, 128, 44), (4.0, 1.0, 1.0), (0.0, 0.0, 2.0), (PER_, N_, N_), 0.0, 4, (1, 1)),
    ("ff-p8-long-y", (128, 1024, 18), (1.0, 3.0, 1.0), (0.0, 0.0, 2.0), (N_, N_, D_), 2e-3, 8, (1, 1)),
    ("gf-p2-small-y", (128, 32, 16), (1.0, 1.0, 1.0), (2.0, 0.0, 1.5), (D_, N_, N_), 0.0, 2, (0, 1)),
], ids=lambda c: c[0])
def test_fast_y_transform_in_sharded_solve(tpt, torch, orc, case):
    name, n, L, beta, bc, alpha, nranks, tr = case
    P = I.Problem(name, n, L, beta, bc, alpha, seed=40 + nranks)
    xf, yf, zf = P.faces()
    f = P.rhs()
    shards = _make_shards(tpt, P, nranks, transform_x=tr[0], transform_y=tr[1])
    rhs, out = _split(torch, shards, f)
    tpt.virtual_ranks_solve(shards, rhs, out)
    torch.cuda.synchronize()
    phi = _gather(shards, out)
    ref = orc.OraclePlan(xf, yf, zf, bc, alpha).solve(f)
    assert float(np.abs(phi - ref).max() / np.abs(ref).max()) <= PARITY_TOL
    plan = tpt.plan_create(*n, xf, yf, zf, bc, alpha, transform=tr)
    d_f = torch.from_numpy(f).cuda()
    d_o = torch.empty_like(d_f)
    plan.solve(d_f, d_o)
    torch.cuda.synchronize()
    assert np.array_equal(d_o.cpu().numpy(), phi)
    plan.destroy()
    # with the device-side flag barriers as well
    tpt.virtual_ranks_solve(shards, rhs, out, barriers=True)
    torch.cuda.synchronize()
    assert np.array_equal(_gather(shards, out), phi)
    for s in shards:
        s.destroy()


def test_shard_argument_errors(tpt, torch):
    P = I.Problem("err", (128, 128, 16), (1.0, 1.0, 1.0), (2.0, 2.0, 2.0), (N_, N_, D_), 0.0, seed=1)
    xf, yf, zf = P.faces()
    with pytest.raises(tpt.TptError):          # nx not a multiple of 128
        tpt.shard_create(0, 2, 96, 128, 16, xf[:97], yf, zf, P.bc)
    with pytest.raises(tpt.TptError):          # more ranks than plane pairs
        tpt.shard_create(0, 8, 128, 128, 12, xf, yf, zf[:13], P.bc)
    with pytest.raises(tpt.TptError):          # periodic z
        tpt.shard_create(0, 2, 128, 128, 16, xf, yf, zf, (N_, N_, PER_))
    with pytest.raises(tpt.TptError):          # a GEMM y transform needs ny % 128 == 0 (a fast one any power of two >= 16)
        tpt.shard_create(0, 2, 128, 64, 16, xf, I.tanh_faces(64, 1.0, 2.0), zf, P.bc)
    s = tpt.shard_create(0, 2, *P.n, xf, yf, zf, P.bc)
    d = torch.zeros(s.slab_points, dtype=torch.float64, device="cuda")
    with pytest.raises(tpt.TptError):          # peers not set yet
        s.solve_phase(0, d, None)
    with pytest.raises(tpt.TptError):          # own entry must be the shard's own allocation
        s.set_peers([s.sym()[0] + 256, s.sym()[0]])
    s.destroy()


def _ipc_worker(rank, world, port, q):
    # One PROCESS per rank, as under torchrun — here both on GPU 0 (the box has one).  The peers' allocations are mapped
    # through CUDA IPC exactly as bench.py --gpus N does it; the phases are ordered by HOST barriers (gloo) after a device
    # synchronise, so no kernel ever waits on another process's kernel.
    import os

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch
    import torch.distributed as dist

    import bench
    from paper_2603_09528_b200 import api

    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    P = I.Problem("ipc", (128, 128, 36), (1.0, 1.0, 1.0), (2.0, 2.0, 2.0), (N_, N_, N_), 0.0, seed=11)
    xf, yf, zf = P.faces()
    sh = api.shard_create(rank, world, *P.n, xf, yf, zf, P.bc, P.alpha)
    handles = bench.exchange_ipc_handles(dist, sh)
    f = P.rhs()
    rhs = torch.from_numpy(bench.shard_slab(f, sh.layout)).cuda()
    out = torch.empty_like(rhs)
    for _ in range(2):
        for ph in range(3):
            sh.solve_phase(ph, rhs if ph == 0 else None, out if ph == 2 else None)
            torch.cuda.synchronize()
            dist.barrier()
    q.put((rank, sh.layout.k0, sh.layout.k1, out.cpu().numpy(), len(set(handles))))
    dist.barrier()
    sh.destroy()
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_solve_across_processes_with_cuda_ipc(tpt, torch, orc, world):
    import os

    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29600 + os.getpid() % 2000 + world
    procs = [ctx.Process(target=_ipc_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=300) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    P = I.Problem("ipc", (128, 128, 36), (1.0, 1.0, 1.0), (2.0, 2.0, 2.0), (N_, N_, N_), 0.0, seed=11)
    xf, yf, zf = P.faces()
    ref = orc.OraclePlan(xf, yf, zf, P.bc, P.alpha).solve(P.rhs())
    assert res[0][1] == 0 and res[-1][2] == P.n[2] and all(a[2] == b[1] for a, b in zip(res, res[1:]))
    assert all(r[4] == world for r in res)                 # every rank saw `world` distinct handles
    phi = np.concatenate([r[3].reshape(-1) for r in res]).reshape(ref.shape)
    assert float(np.abs(phi - ref).max() / np.abs(ref).max()) <= PARITY_TOL
