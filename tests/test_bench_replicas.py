"""Host-side logic of the N > 1 bench path (replicas only, no data-path collective), covered on CPU with
world_size-2 gloo: max-over-ranks timing, whole-job aggregation, per-rank seeds, and the rank-0-only reference arm."""
import json
import os
import subprocess
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2603_09528_b200 import inputs as I

    local_ms = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    total = bench.max_over_ranks(dist, local_ms, "cpu")
    P = I.CONFIGS["c1"][0]
    f = bench.replica_problem(P, rank).rhs()
    q.put((rank, total, bench.whole_job_value(world, P.points, 4, total * 1e-3), float(f.ravel()[0]), int(bench.replica_problem(P, rank).seed)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_replica_seeds_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, t0, v0, f0, s0), (r1, t1, v1, f1, s1) = out
    assert t0 == t1 == 15.0                                   # the slowest rank's time, on every rank
    assert v0 == v1 == 2 * 4096 * 4 / 15e-3 / 1e9            # all ranks' points over that time
    assert s1 == s0 + 1000 and f0 != f1                       # independent replicas: different right-hand sides


def test_single_process_helpers():
    import bench

    assert bench.max_over_ranks(None, 3.5) == 3.5
    assert bench.whole_job_value(1, 10 ** 9, 2, 1.0) == 2.0


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29999", OMP_NUM_THREADS="2")
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "c1",
           "--steps", "2", "--warmup", "1"]
    r1 = subprocess.run(cmd, env=dict(env, RANK="1", LOCAL_RANK="1"), capture_output=True, text=True, timeout=300)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
    r0 = subprocess.run(cmd, env=dict(env, RANK="0", LOCAL_RANK="0"), capture_output=True, text=True, timeout=300)
    assert r0.returncode == 0, r0.stderr
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["unit"] == "Gpts/s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["value"] == line["value"] > 0
    assert line["e2e"] == {"value": line["value"], "unit": "Gpts/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert line["vs_baseline"] is None and np.isfinite(line["ms_per_step"])


class _FakeShard:
    """Stands in for api.Shard on a CPU-only box: the host logic under test is the handle exchange, not CUDA."""

    def __init__(self, rank):
        self.rank, self.imported = rank, None

    def ipc_export(self):
        return bytes([self.rank]) * 64

    def ipc_import(self, handles):
        self.imported = list(handles)


def _shard_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2603_09528_b200 import api, inputs as I

    sh = _FakeShard(rank)
    bench.exchange_ipc_handles(dist, sh)
    nx, ny, nz = 128, 128, 22
    lay = api.shard_layout(world, rank, nx, ny, nz)            # host-only entry point of the library
    f = I.uniform_pm1(3, nx * ny * nz).reshape(nz, ny, nx)
    slab = bench.shard_slab(f, lay)
    q.put((rank, [h[0] for h in sh.imported], lay.k0, lay.k1, slab.shape, float(slab.sum()), float(f.sum()),
           int(lay.nvlink_bytes_per_solve)))
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_host_logic_gloo_world2():
    # SURVEY 8(f).4 host side: IPC handles all-gathered in rank order on every rank; the z-slabs of the ranks tile the
    # field; the byte count that crosses NVLink is 2 * 8 * pts * (P-1)/P over all ranks; strong-scaling value
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    a, b = out
    assert a[1] == b[1] == [0, 1]
    assert a[2] == 0 and a[3] == b[2] and b[3] == 22 and a[3] % 2 == 0
    assert a[4] == (a[3], 128, 128) and b[4] == (22 - a[3], 128, 128)
    assert abs(a[5] + b[5] - a[6]) < 1e-9
    assert a[7] == 2 * 8 * 128 * 64 * (22 - a[3]) and b[7] == 2 * 8 * 128 * 64 * a[3]
    assert a[7] + b[7] == 2 * 8 * 128 * 128 * 22 // 2

    import bench

    assert bench.sharded_strong_value(10 ** 9, 4, 2.0) == 2.0
