#!/usr/bin/env python
"""bench.py — headline benchmark of the tensor-product–Thomas solver on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config c3|c4|c5|c2|c1]

A "step" is one pass of the whole hot path (forward x, forward y, Thomas z, inverse y, inverse x) over one
right-hand side of the workload: BASELINE.json's metric workload, config c3 = FP64 Poisson, 512^3 cells,
tanh beta = 2 in all three directions, all-Neumann (singular), uniform[-1,1] rhs (seed 2) with its
volume-weighted mean removed.  Prints ONE JSON line (rank 0).

  value       whole-job Gpts/s with the rhs already resident in HBM (N>1: N independent replicas, §8(e))
  e2e         the same metric through the C-ABI calls tpt_solve_host_async / tpt_plan_wait with pinned HOST buffers
              (H2D + D2H of every step inside; consecutive steps overlap their copies through two plans)
  roofline    dominant kernel (the slowest of the four DMMA GEMM transforms): algorithmic flops / CUDA-event duration vs FP64 peak
  cpu_baseline the oracle (as it stands) timed on the host cores on a bounded z-slab sample of the workload
  --impl reference  times the oracle alone (rank 0 only)
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2603_09528_b200 import inputs as I  # noqa: E402

METRIC = "FP64 stretched-grid Poisson solve Gpts/s at 512^3 (one tensor-product-Thomas solve per step)"
UNIT = "Gpts/s"
# FP64 peak of one B200: 148 SMs x 64 FP64 FMA/clk/SM x 2 flop x 1.965 GHz; the DMMA and
# DFMA microbenchmarks of the library are reported next to it.
SM_COUNT, FP64_FMA_PER_CLK_SM = 148, 64
# transform type per diagonalised direction (x, y): the paper's GG / FG / GF / FF variants; FFT needs a
# uniform power-of-two direction.  BASELINE.json's metric is quoted on GG.
TRANSFORMS = {"gg": (0, 0), "fg": (1, 0), "gf": (0, 1), "ff": (1, 1)}
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel (gemm_tma_kernel), from the one
# `ncu --set full` capture summarised in profiles/r2_final_round2.md (config c3; bytes), taken with the kernel sources of the
# commit named here (the round's last kernel change).  Other configs: null.
NCU_TRAFFIC = {"commit": "2e93fea", "capture": "profiles/r2_final_round2.md", "bytes": {"c3": 1.075920e9 + 1.030197e9}}


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return json.load(fh), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


def _workload(name: str):
    probs = I.CONFIGS[name]
    return probs


def _config_json(name: str, probs, extra=None):
    P = probs[0]
    cfg = {
        "workload": (f"BASELINE.json configs[{int(name[1]) - 1}] ({name}): " if name[0] == "c" else
                     f"the paper's single-GPU benchmark case, PAPER.md:294 ({name}): ") + ", ".join(p.name for p in probs),
        "grid": list(P.n), "tanh_beta": list(P.beta), "bc": ["N" if b == 0 else "D" for b in P.bc],
        "solves_per_step": len(probs), "helmholtz_alpha": [p.alpha for p in probs],
        "points_per_step": sum(p.points for p in probs),
        "cache": "each array (>= 1 GiB at 512^3) exceeds the 126 MB L2; no flush needed between steps",
    }
    if extra:
        cfg.update(extra)
    return cfg


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    REASONS = {
        0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
        0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
        0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting",
    }

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index = index
        self.stop_flag = threading.Event()
        self.sm, self.power, self.mask, self.sm_max = [], [], 0, None
        self.ok = False

    def run(self):
        try:
            import pynvml as nv

            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.sm_max = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            self.ok = True
            while not self.stop_flag.is_set():
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                try:
                    self.power.append(nv.nvmlDeviceGetPowerUsage(h) / 1000.0)
                    self.mask |= int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                except Exception:
                    pass
                time.sleep(0.02)
        except Exception:
            self.ok = False

    def summary(self):
        if not self.ok or not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": ["unavailable"]}
        reasons = [n for b, n in self.REASONS.items() if self.mask & b and n != "gpu_idle"]
        return {"sm_mhz": float(np.median(self.sm)), "sm_max_mhz": self.sm_max, "reasons": reasons,
                "power_w_max": max(self.power) if self.power else None, "samples": len(self.sm)}


BAD_REASONS = {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"}


def _oracle_time(probs, steps: int, warmup: int, budget_s: float):
    """Times the oracle's solve (plan excluded, like the GPU's) on the workload.  The FULL workload is timed whenever
    (steps + warmup) passes of it fit `budget_s` of host time (configs c1-c4 on the box's 16 cores); otherwise every
    problem is cut to a z-slab of as many planes as fit (same x/y grids, eigenbases and per-point transform work;
    c5: ~3e12 flop per solve), and `sample` says so.  The plane count is chosen from an untimed 8-plane calibration."""
    import oracle   # test infrastructure; allowed here (cpu_baseline / --impl reference)

    passes = steps + warmup
    t_plane = 0.0
    cal = []
    for P in probs:
        C = P.thin_z(min(8, P.n[2]))
        xf, yf, zf = C.faces()
        pl, f = oracle.OraclePlan(xf, yf, zf, C.bc, C.alpha), C.rhs()
        pl.solve(f)
        t0 = time.perf_counter()
        pl.solve(f)
        cal.append((time.perf_counter() - t0) / C.n[2])
        pl.close()
    full_s = sum(c * P.n[2] for c, P in zip(cal, probs)) * passes
    frac = min(1.0, budget_s / max(full_s, 1e-9))
    plans, rhs, pts, planes = [], [], 0, []
    for P in probs:
        nzs = P.n[2] if frac >= 1.0 else max(8, min(P.n[2], int(P.n[2] * frac) // 8 * 8))
        S = P if nzs == P.n[2] else P.thin_z(nzs)
        xf, yf, zf = S.faces()
        plans.append(oracle.OraclePlan(xf, yf, zf, S.bc, S.alpha))
        rhs.append(S.rhs())
        pts += S.points
        planes.append(nzs)
    for _ in range(warmup):
        for pl, f in zip(plans, rhs):
            pl.solve(f)
    t0 = time.perf_counter()
    for _ in range(steps):
        for pl, f in zip(plans, rhs):
            pl.solve(f)
    dt = (time.perf_counter() - t0) / steps
    for pl in plans:
        pl.close()
    P = probs[0]
    if all(n == Q.n[2] for n, Q in zip(planes, probs)):
        sample = (f"the FULL workload ({len(probs)} solve(s) of {P.n[0]}x{P.n[1]}x{P.n[2]} cells per step), {steps} timed step(s) "
                  f"after {warmup} warm-up; plan (eigendecomposition) excluded")
    else:
        sample = (f"oracle solve on a z-slab of each problem: {P.n[0]}x{P.n[1]}x{planes[0]} of {P.n[2]} planes (same x/y grids "
                  f"and eigenbases, per-point transform work identical; the full workload would take ~{full_s:.0f} s for "
                  f"{passes} passes, budget {budget_s:.0f} s), {steps} timed step(s) after {warmup} warm-up; plan excluded")
    return {"value": pts / dt / 1e9, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample,
            "note": "the parity oracle as it stands: naive OpenMP loops, no BLAS, never tuned — a reported baseline, not a "
                    "tuned CPU implementation and not the target",
            "ms_per_sample_step": dt * 1e3, "sample_points": pts}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    probs = _workload(args.config)
    steps, warmup = max(1, args.steps), max(0, args.warmup)      # honoured as given (the driver compares them)
    base = _oracle_time(probs, steps, warmup, budget_s=300.0)
    line = {
        "impl": "reference", "metric": METRIC, "value": base["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warmup, "ms_per_step": base["ms_per_sample_step"],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": _config_json(args.config, probs, {"parallelism": "replicas only" if args.gpus > 1 else "single GPU",
                                                      "transform_xy": args.transform}),
        "cpu_baseline": {k: base[k] for k in ("value", "unit", "cores", "kind", "sample", "note")},
        "e2e": {"value": base["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def replica_problem(P, rank: int):
    """Replicas only: rank r solves its own copy of the workload, rhs seed offset by 1000 r."""
    import dataclasses

    return dataclasses.replace(P, seed=P.seed + 1000 * rank)


def max_over_ranks(dist, value: float, device="cpu") -> float:
    """Timing rule for N > 1: the job takes as long as its slowest rank."""
    if dist is None:
        return float(value)
    import torch

    t = torch.tensor([value], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, pts_step: int, steps: int, seconds: float) -> float:
    """Gpts/s over all replicas: every rank processed pts_step * steps points in `seconds` (max over ranks)."""
    return world * pts_step * steps / seconds / 1e9


def device_rhs(api, torch, P, stream=None):
    """The problem's right-hand side generated on the device: the same counter-based white noise as Problem.rhs()
    (bit-identical, tests/test_gpu_variants.py) and, for singular problems, the volume-weighted mean removed (A8)."""
    nx, ny, nz = P.n
    f = torch.empty((nz, ny, nx), dtype=torch.float64, device="cuda")
    api.fill_uniform(f, P.seed, 0, stream)
    if P.singular:
        wx, wy, wz = (torch.from_numpy(np.diff(a)).cuda() for a in P.faces())
        mean = torch.einsum("k,j,i,kji->", wz, wy, wx, f) / (wx.sum() * wy.sum() * wz.sum())
        f -= mean
    return f


def measure_config(api, torch, name, fp64_peak, hbm_gbs, steps=6, warmup=3):
    """Device-timed numbers of one BASELINE config (GG transforms): ms per step, Gpts/s, the slowest GEMM transform's
    fraction of the FP64 peak and the sweep's fraction of the HBM peak, from `steps` timed steps after `warmup`."""
    probs = I.CONFIGS[name]
    stream = torch.cuda.current_stream()
    plan_cache, plans, rhs, outs = {}, [], [], []
    for P in probs:
        key = (P.n, P.bc, P.alpha, P.beta, P.length)
        if key not in plan_cache:
            plan_cache[key] = api.plan_create(*P.n, *P.faces(), P.bc, P.alpha)
        plans.append(plan_cache[key])
        rhs.append(device_rhs(api, torch, P, stream))
        outs.append(torch.empty_like(rhs[-1]))
    # the small configs fit the 126 MB L2: flush it between steps (outside the per-step events) by rewriting a 256 MB buffer
    small = sum(P.points for P in probs) * 8 * 3 < 256e6
    flush = torch.empty(32 << 20, dtype=torch.float64, device="cuda") if small else None

    def step():
        for pl, r, o in zip(plans, rhs, outs):
            api.solve(pl, r, o, stream)

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    for pl in plan_cache.values():
        pl.set_profiling(True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in ev:
        if flush is not None:
            flush.zero_()
        a.record(stream)
        step()
        b.record(stream)
    torch.cuda.synchronize()
    ms = sorted(a.elapsed_time(b) for a, b in ev)
    ms_step = float(np.mean(ms))
    P0, pl0 = probs[0], plans[0]
    kms, launches, _ = pl0.kernel_times()
    for pl in plan_cache.values():
        pl.set_profiling(False)
    paths = pl0.paths()
    fused = api.PATH_FUSED_SMALL in paths
    back_to_back = None
    if small:      # launch-bound sizes: also the throughput of solves issued back to back (warm L2, no events in between)
        reps = 200
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for _ in range(20):
            step()
        a.record(stream)
        for _ in range(reps):
            step()
        b.record(stream)
        torch.cuda.synchronize()
        back_to_back = a.elapsed_time(b) / reps
    nx, ny, nz = P0.n
    gemm = {"fwd_x": 2.0 * nx, "fwd_y": 2.0 * ny, "inv_y": 2.0 * ny, "inv_x": 2.0 * nx}
    fr = {k: gemm[k] * P0.points / (kms[i] * 1e-3) / 1e12 / fp64_peak for i, k in enumerate(api.KERNEL_NAMES) if k in gemm}
    slow = min(fr, key=fr.get)
    th = kms[api.K_THOMAS]
    out = {
        "workload": ", ".join(P.name for P in probs), "grid": list(P0.n), "solves_per_step": len(probs),
        "ms_per_step": ms_step, "ms_per_step_min": ms[0], "gpts_per_s": sum(P.points for P in probs) / ms_step / 1e6,
        "timed_steps": steps, "warmup": warmup, "l2_flushed_between_steps": bool(small),
        "ms_per_step_back_to_back_warm_l2": back_to_back,
        "paths_first_plan": dict(zip(api.KERNEL_NAMES, paths)),
        "kernel_ms_first_plan": dict(zip(api.KERNEL_NAMES, kms)),
        "gemm_frac_of_fp64_peak": None if fused else {"slowest": slow, "frac": fr[slow], "all": fr},
        "thomas_frac_of_hbm_peak_16B_per_pt": None if fused else 16.0 * P0.points / (th * 1e-3) / 1e9 / hbm_gbs,
        "gpu_launches_first_plan": launches,
    }
    if fused:
        out["note"] = ("small-grid path: the whole solve is ONE cluster launch (fused_small_kernel); its time is reported in the "
                       "fwd_x slot, the other slots are empty event intervals")
    for pl in plan_cache.values():
        pl.destroy()
    del rhs, outs, flush
    torch.cuda.empty_cache()
    return out


def shard_slab(f, lay):
    """This rank's z-slab of the (nz, ny, nx) field f (the field is distributed, each rank holds a part)."""
    return np.ascontiguousarray(f[lay.k0:lay.k1])


def exchange_ipc_handles(dist, shard):
    """Control plane of the sharded solve: all-gather the CUDA IPC handles of the symmetric allocations (64 bytes per rank,
    through torch.distributed's object collective — not a data-path collective) and map the peers."""
    handles = [None] * dist.get_world_size()
    dist.all_gather_object(handles, shard.ipc_export())
    shard.ipc_import(handles)
    return handles


def sharded_strong_value(pts_step: int, steps: int, seconds: float) -> float:
    """Strong scaling: the job is ONE workload whatever the number of ranks."""
    return pts_step * steps / seconds / 1e9


def measure_sharded(api, torch, dist, args, probs, rank, world, stream, barrier):
    """the workload's solves sharded over the `world` GPUs (tpt_solve_sharded: two exchanges fused into the
    forward-y GEMM epilogue and the sweep's TMA store, two flag barriers).  Strong scaling; device-timed, max over ranks.
    Every rank also solves the same right-hand side on its own with the single-GPU plan and compares its slab bit by bit."""
    shards, rhs, out, ok, nvl = [], [], [], True, 0
    cache = {}
    for P in probs:
        key = (P.n, P.bc, P.alpha, P.beta, P.length)
        if key not in cache:
            xf, yf, zf = P.faces()
            sh = api.shard_create(rank, world, *P.n, xf, yf, zf, P.bc, P.alpha, *TRANSFORMS[args.transform])
            exchange_ipc_handles(dist, sh)
            cache[key] = sh
        sh = cache[key]
        shards.append(sh)
        f = P.rhs()
        rhs.append(torch.from_numpy(shard_slab(f, sh.layout)).cuda())
        out.append(torch.empty_like(rhs[-1]))
        nvl += int(sh.layout.nvlink_bytes_per_solve)
        del f
    barrier()

    def step():
        for sh, r, o in zip(shards, rhs, out):
            sh.solve(r, o, stream)

    for _ in range(args.warmup):
        step()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    ms = max_over_ranks(dist, e0.elapsed_time(e1), "cuda")
    # parity of the sharded result with the single-GPU solve of the same right-hand side (first problem), slab by slab
    P = probs[0]
    xf, yf, zf = P.faces()
    plan = api.plan_create(*P.n, xf, yf, zf, P.bc, P.alpha, transform=TRANSFORMS[args.transform])
    full = torch.from_numpy(P.rhs()).cuda()
    api.solve(plan, full, full, stream)
    torch.cuda.synchronize()
    lay = shards[0].layout
    ok = bool(torch.equal(full.view(P.n[2], P.n[1], P.n[0])[lay.k0:lay.k1].reshape(-1), out[0].reshape(-1)))
    flag = torch.tensor([1 if ok else 0], device="cuda")
    dist.all_reduce(flag, op=dist.ReduceOp.MIN)
    plan.destroy()
    del full
    barrier()
    for sh in cache.values():
        sh.destroy()
    pts_step = sum(P.points for P in probs)
    secs = ms * 1e-3
    return {"what": "tpt_solve_sharded: z-slab + y-mode-row ownership, exchanges fused into the GEMM epilogue and the sweep's "
                    "TMA store over NVLink peer memory (PAPER.md:197-207)",
            "scaling": "strong", "ranks": world, "value": sharded_strong_value(pts_step, args.steps, secs), "unit": UNIT,
            "ms_per_step": ms / args.steps, "nvlink_bytes_per_step_per_rank": nvl,
            "nvlink_gbs_per_rank_per_direction": nvl / (ms / args.steps * 1e-3) / 1e9,
            "launches_per_solve": 7, "matches_single_gpu_bitwise": bool(flag.item())}


def measure_sharded_virtual(api, torch, P, nranks, stream, steps=5, warmup=3):
    """One-GPU leg of SURVEY 8(f).4: `nranks` virtual ranks on this device (peer pointers = local pointers), phases ordered
    by the stream.  All ranks' work runs on one GPU, so the time is comparable with one single-plan solve: the difference is
    what the fused exchanges (scattered epilogue rows, per-owner TMA stores) cost on the device."""
    xf, yf, zf = P.faces()
    shards = [api.shard_create(r, nranks, *P.n, xf, yf, zf, P.bc, P.alpha) for r in range(nranks)]
    syms = [sh.sym()[0] for sh in shards]
    for sh in shards:
        sh.set_peers(syms)
    full = device_rhs(api, torch, P, stream).view(P.n[2], P.n[1], P.n[0])
    rhs = [full[sh.layout.k0:sh.layout.k1].reshape(-1) for sh in shards]      # z-slabs are contiguous views
    out = [torch.empty_like(r) for r in rhs]
    for _ in range(warmup):
        api.virtual_ranks_solve(shards, rhs, out, stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        api.virtual_ranks_solve(shards, rhs, out, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    plan = api.plan_create(*P.n, xf, yf, zf, P.bc, P.alpha)
    ref = torch.empty_like(full).reshape(-1)
    api.solve(plan, full.reshape(-1), ref, stream)
    torch.cuda.synchronize()
    same = bool(torch.equal(torch.cat(out), ref))
    e0.record(stream)
    for _ in range(steps):
        api.solve(plan, full.reshape(-1), ref, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_one = e0.elapsed_time(e1) / steps
    plan.destroy()
    for sh in shards:
        sh.destroy()
    return {"what": f"{nranks} virtual ranks of the sharded solve on one device ({P.name}); all ranks' kernels run on this GPU",
            "virtual_ranks": nranks, "ms_per_solve_all_ranks": ms, "ms_single_plan_solve": ms_one,
            "device_overhead_of_fused_exchanges": ms / ms_one - 1.0, "matches_single_plan_bitwise": same,
            "launches": 5 * nranks}


def run_gpu(args):
    import torch

    from paper_2603_09528_b200 import api

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist_mod

        dist = dist_mod
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    else:
        torch.cuda.set_device(0)
    dev_index = torch.cuda.current_device()
    api.lib()   # fails loudly if the CUDA library is missing

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # replicas only (§8(e)): every rank solves its own copy of the workload (seed offset by rank)
    probs = _workload(args.config)
    plans, d_rhs, d_out, h_rhs = [], [], [], []
    plan_cache, probs_by_key, plan_keys = {}, {}, []
    for P in probs:
        xf, yf, zf = P.faces()
        key = (P.n, P.bc, P.alpha, P.beta, P.length)
        if key not in plan_cache:
            plan_cache[key] = api.plan_create(*P.n, xf, yf, zf, P.bc, P.alpha, transform=TRANSFORMS[args.transform])
            probs_by_key[key] = P
        plans.append(plan_cache[key])
        plan_keys.append(key)
        f = replica_problem(P, rank).rhs()
        h_rhs.append(f)
        d_rhs.append(torch.from_numpy(f).cuda())
        d_out.append(torch.empty_like(d_rhs[-1]))
    pts_step = sum(P.points for P in probs)
    stream = torch.cuda.current_stream()

    def step():
        for pl, r, o in zip(plans, d_rhs, d_out):
            api.solve(pl, r, o, stream)

    def timed_region():
        for _ in range(args.warmup):
            step()
        barrier()
        sampler = ClockSampler(dev_index)
        sampler.start()
        for pl in plan_cache.values():
            pl.set_profiling(True)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
        ev[0].record(stream)
        for s in range(args.steps):
            step()
            ev[s + 1].record(stream)
        barrier()
        sampler.stop_flag.set()
        sampler.join()
        total_ms = ev[0].elapsed_time(ev[-1])
        per_step = sorted(ev[s].elapsed_time(ev[s + 1]) for s in range(args.steps))
        kt = {}
        launches = 0
        for key, pl in plan_cache.items():
            ms, n_launch, n_solves = pl.kernel_times()
            pl.set_profiling(False)
            kt[key] = (ms, n_solves)
            launches += n_launch
        return total_ms, per_step, kt, launches, sampler.summary()

    total_ms, per_step, kt, launches, clocks = timed_region()
    if BAD_REASONS & set(clocks["reasons"]):          # rejected: re-measure once
        total_ms, per_step, kt, launches, clocks = timed_region()
        clocks["remeasured"] = True
    total_ms = max_over_ranks(dist, total_ms, "cuda")
    ms_per_step = total_ms / args.steps
    value = whole_job_value(world, pts_step, args.steps, total_ms * 1e-3)

    # ---- e2e: the C-ABI call with pinned HOST buffers, copies inside the timed region.  Every step moves its inputs
    # host -> device and its result device -> host; consecutive steps alternate between two plan sets on two streams
    # (tpt_solve_host_async / tpt_plan_wait), so one step's download overlaps the next one's upload on the full-duplex bus.
    e2e_steps = max(2, min(args.steps, 10))
    pin_in = [torch.from_numpy(f).pin_memory() for f in h_rhs]
    pin_out = [[torch.empty_like(t).pin_memory() for t in pin_in] for _ in range(2)]
    plan_cache2 = {k: api.plan_create(*pl.shape[::-1], *probs_by_key[k].faces(), probs_by_key[k].bc, probs_by_key[k].alpha,
                                      transform=TRANSFORMS[args.transform]) for k, pl in plan_cache.items()}
    slot_plans = [plans, [plan_cache2[k] for k in plan_keys]]
    slot_streams = [torch.cuda.Stream(), torch.cuda.Stream()]

    def e2e_run(nsteps):
        for s in range(nsteps):
            q = s & 1
            for pl, a, b in zip(slot_plans[q], pin_in, pin_out[q]):
                api.solve_host(pl, a, b, slot_streams[q], nowait=True)
        for q in range(2):
            for pl in set(slot_plans[q]):
                api.plan_wait(pl)

    e2e_run(2)
    barrier()
    t0 = time.perf_counter()
    e2e_run(e2e_steps)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(dist, e2e_s, "cuda")
    e2e_val = whole_job_value(world, pts_step, e2e_steps, e2e_s)
    e2e_ok = all(np.array_equal(b.numpy(), o.cpu().numpy()) for q in range(2) for b, o in zip(pin_out[q], d_out))
    for pl in plan_cache2.values():
        api.plan_destroy(pl)
    del pin_out

    # ---- the same workload sharded over the ranks (strong scaling), beside the replica number
    sharded = None
    if world > 1 and not args.no_sharded:
        try:
            sharded = measure_sharded(api, torch, dist, args, probs, rank, world, stream, barrier)
        except api.TptError as exc:      # e.g. a grid the sharded layout does not take: reported, never silently skipped
            sharded = {"unavailable": str(exc)}

    # ---- widened row: one pressure projection (Eq. 2c-2e) = divergence + this solve + correction,
    # timed on the device on the workload's Poisson plan (outside the headline timed region; rank 0 only)
    projection = None
    pois = [(pl, P) for pl, P in zip(plans, probs) if P.alpha == 0.0]
    if rank == 0 and pois and not args.no_projection:
        pl, P = pois[0]
        cu, cv, cw = api.face_counts(pl)
        gen = torch.Generator(device="cuda")
        gen.manual_seed(1234)
        fu, fv, fw = (torch.rand(m, dtype=torch.float64, device="cuda", generator=gen) * 2 - 1 for m in (cu, cv, cw))
        phi, pr = torch.empty(pl.points, dtype=torch.float64, device="cuda"), torch.zeros(pl.points, dtype=torch.float64, device="cuda")

        def timed(fn, reps=10):
            for _ in range(3):
                fn()
            torch.cuda.synchronize()
            e = [torch.cuda.Event(enable_timing=True) for _ in range(reps + 1)]
            e[0].record(stream)
            for q in range(reps):
                fn()
                e[q + 1].record(stream)
            torch.cuda.synchronize()
            return e[0].elapsed_time(e[-1]) / reps

        t_div = timed(lambda: api.divergence(pl, fu, fv, fw, phi, 1.0, stream))
        t_cor = timed(lambda: api.gradient_correct(pl, phi, 1e-9, fu, fv, fw, p=pr, alpha_p=1e-9, dirs=api.DIRS_XYZ, stream=stream))
        t_all = timed(lambda: api.project(pl, fu, fv, fw, 1.0, phi, p=pr, alpha_p=1e-9, dirs=api.DIRS_XYZ, stream=stream))
        hbm = _peaks()[0]["hbm_gbs"]
        projection = {
            "workload": f"tpt_project on {P.name}: white-noise face velocities, pressure update fused (Eq. 2e, L_I = L)",
            "ms_per_projection": t_all, "gpts_per_s": P.points / t_all / 1e6,
            "divergence": {"ms": t_div, "algorithmic_B_per_pt": 32, "frac_of_hbm_peak": 32.0 * P.points / t_div / 1e6 / hbm},
            "correction_with_pressure_update": {"ms": t_cor, "algorithmic_B_per_pt": 72,
                                                "frac_of_hbm_peak": 72.0 * P.points / t_cor / 1e6 / hbm},
        }
        del fu, fv, fw, phi, pr

    if rank == 0:
        peaks, peak_kind = _peaks()
        sm_max = float(peaks.get("sm_max_mhz", 1965.0))
        fp64_peak = SM_COUNT * FP64_FMA_PER_CLK_SM * 2 * sm_max * 1e6 / 1e12
        dmma_meas, dfma_meas = api.fp64_peak(1), api.fp64_peak(0)
        # ---- the other BASELINE configs (device-timed, GG), so that the driver-run record carries all five
        other_configs = None
        if not args.no_other_configs and args.transform == "gg":
            for t in (d_rhs, d_out):
                t.clear()
            torch.cuda.empty_cache()
            other_configs = {n: measure_config(api, torch, n, fp64_peak, peaks["hbm_gbs"])
                             for n in ("c1", "c2", "c3", "c4", "c5") if n != args.config}
        if world == 1 and not args.no_sharded and args.transform == "gg":
            try:
                sharded = measure_sharded_virtual(api, torch, I.CONFIGS["c3"][0], 4, stream)
            except api.TptError as exc:
                sharded = {"unavailable": str(exc)}
        # per-kernel: mean event durations over the timed region (dominant plan = first)
        key0 = next(iter(kt))
        ms0, _ = kt[key0]
        P0 = probs[0]
        nx, ny, nz = P0.n
        pts = P0.points
        flops = {"fwd_x": 2.0 * nx * pts, "fwd_y": 2.0 * ny * pts, "inv_y": 2.0 * ny * pts, "inv_x": 2.0 * nx * pts}
        kernels = {}
        for slot, name in enumerate(api.KERNEL_NAMES):
            entry = {"ms": ms0[slot]}
            fast = (name.endswith("_x") and TRANSFORMS[args.transform][0]) or (name.endswith("_y") and TRANSFORMS[args.transform][1])
            if name == "thomas" or fast:
                gbs = 16.0 * pts / (ms0[slot] * 1e-3) / 1e9
                entry.update({"bound": "hbm", "achieved_gbs_16B_per_pt": gbs, "frac_of_hbm_peak": gbs / peaks["hbm_gbs"]})
            else:
                tf = flops[name] / (ms0[slot] * 1e-3) / 1e12
                entry.update({"bound": "tensor", "achieved_tflops": tf, "frac_of_fp64_peak": tf / fp64_peak})
            kernels[name] = entry
        gemm_slots = [n for n in ("fwd_x", "fwd_y", "inv_y", "inv_x") if kernels[n]["bound"] == "tensor"]
        dom = max(gemm_slots or ("fwd_x", "fwd_y", "inv_y", "inv_x"), key=lambda n: kernels[n]["ms"])
        traffic = NCU_TRAFFIC["bytes"].get(args.config)
        if gemm_slots:
            roofline = {
                "kernel": f"gemm_tma_kernel ({dom})", "bound": "tensor", "achieved": kernels[dom]["achieved_tflops"],
                "peak": fp64_peak, "unit": "TFLOP/s", "frac": kernels[dom]["achieved_tflops"] / fp64_peak, "traffic": traffic,
                "peak_source": f"148 SMs x 64 FP64 FMA/clk x 2 x {sm_max:.0f} MHz ({peak_kind} sm_max_mhz); FP64 is absent from "
                               "MEASURED_PEAKS.json",
                "peak_measured_dmma_loop": dmma_meas, "peak_measured_dfma_loop": dfma_meas,
                "frac_of_measured_dmma_loop": kernels[dom]["achieved_tflops"] / dmma_meas,
                "algorithmic_flops_per_launch": flops[dom], "algorithmic_dram_bytes_per_launch": 16.0 * pts,
            }
            if traffic is not None:
                roofline["traffic_unit"] = (f"bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum; capture "
                                            f"{NCU_TRAFFIC['capture']}, kernel source as of commit {NCU_TRAFFIC['commit']})")
        if not gemm_slots:   # FF: no GEMM left — the dominant kernel is the slowest fast transform, HBM-bound at 16 B/pt
            roofline = {
                "kernel": f"fft kernel ({dom})", "bound": "hbm", "achieved": kernels[dom]["achieved_gbs_16B_per_pt"],
                "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": kernels[dom]["frac_of_hbm_peak"], "traffic": None,
                "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peak_kind})",
                "algorithmic_dram_bytes_per_launch": 16.0 * pts,
            }
        cpu = _oracle_time(probs, 3, 1, budget_s=60.0)
        n20 = per_step[: min(20, len(per_step))]
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": _config_json(args.config, probs, {"parallelism": "replicas only" if world > 1 else "single GPU",
                                                          "transform_xy": args.transform}),
            "clocks": clocks,
            "projection": projection,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": 8 * pts_step, "d2h_bytes_per_step": 8 * pts_step,
                    "steps": e2e_steps, "ms_per_step": e2e_s / e2e_steps * 1e3, "matches_device_result": bool(e2e_ok)},
            "gpu_launches": launches,
            "roofline": roofline,
            "kernels": kernels,
            "cpu_baseline": {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample", "note")},
            "other_configs": other_configs,
            "sharded": sharded,
            "solve_ms_mean_20_fastest": float(np.mean(n20)) / len(probs), "solve_ms_min": per_step[0] / len(probs),
            "hbm_peak_gbs": peaks["hbm_gbs"], "peaks": peak_kind,
        }
        print(json.dumps(line), flush=True)
    for pl in plan_cache.values():
        pl.destroy()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c3", choices=sorted(I.CONFIGS))
    ap.add_argument("--transform", default="gg", choices=sorted(TRANSFORMS),
                    help="transform type in x, y: g = eigenbasis GEMM (BASELINE metric), f = fast transform (uniform directions)")
    ap.add_argument("--no-other-configs", dest="no_other_configs", action="store_true",
                    help="skip the device-timed numbers of the other BASELINE configs (c1, c2, c4, c5)")
    ap.add_argument("--no-sharded", dest="no_sharded", action="store_true",
                    help="skip the sharded-solve leg (N > 1: strong scaling over the ranks; N = 1: four virtual ranks on one GPU)")
    ap.add_argument("--no-projection", dest="no_projection", action="store_true",
                    help="skip the (untimed-region) pressure-projection measurement")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
