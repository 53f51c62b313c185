"""CPU-side checks of the C-ABI library: it builds for sm_100a, loads, exports every symbol the header
declares, and validates arguments without a GPU.  No compute calls."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def tpt():
    from paper_2603_09528_b200 import api, build

    build.build()
    return api


def test_header_symbols_all_exported(tpt):
    hdr = open(os.path.join(ROOT, "include", "tpt.h")).read()
    declared = set(re.findall(r"\b(tpt_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(tpt.SYMBOLS)
    L = tpt.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert "sm_100a" in tpt.version()


def test_header_cites_the_paper_for_each_entry_point():
    hdr = open(os.path.join(ROOT, "include", "tpt.h")).read()
    assert hdr.count("PAPER.md:") >= 10


def test_status_strings(tpt):
    assert tpt.strerror(0) == "ok"
    for s in (-1, -2, -3, -4, -5):
        assert tpt.strerror(s) not in ("ok", "unknown status")
    assert tpt.strerror(-99) == "unknown status"


def test_argument_validation_needs_no_gpu(tpt):
    good = np.linspace(0, 1, 9)
    bad = good.copy()
    bad[3] = bad[2]
    with pytest.raises(tpt.TptError) as e:
        tpt.plan_create(8, 8, 8, bad, good, good, (0, 0, 1), 0.0)
    assert e.value.status == -1
    with pytest.raises(tpt.TptError) as e:
        tpt.plan_create(8, 8, 8, good, good, good, (0, 3, 1), 0.0)
    assert e.value.status == -1
    with pytest.raises(tpt.TptError) as e:
        tpt.plan_create(8, 8, 2, good, good, np.linspace(0, 1, 3), (0, 0, 2), 0.0)      # periodic z needs at least 3 cells
    assert e.value.status == -1
    with pytest.raises(tpt.TptError) as e:
        tpt.plan_create(8, 8, 8, good, good, good, (0, 0, 1), -1.0)
    assert e.value.status == -1
    with pytest.raises(tpt.TptError) as e:
        tpt.plan_create(8, 8, 8, good, good, good, (0, 0, 1), float("nan"))
    assert e.value.status == -1
    with pytest.raises(ValueError):
        tpt.plan_create(8, 8, 8, good[:-1], good, good, (0, 0, 1), 0.0)
    # fast transforms: only for diagonalised, uniform, power-of-two directions
    u16, s16 = np.linspace(0, 1, 17), np.linspace(0, 1, 17) ** 2
    for args, kw in (((16, 16, 16, s16, u16, u16, (0, 0, 1), 0.0), dict(transform=(1, 0))),        # x stretched
                     ((8, 16, 16, good, u16, u16, (0, 0, 1), 0.0), dict(transform=(1, 0))),        # 8 cells: below 16
                     ((16, 16, 16, u16, u16, u16, (0, 0, 1), 1e-3), dict(transform=(0, 1), dirs=tpt.DIRS_Z)),
                     ((16, 16, 16, u16, u16, u16, (0, 0, 1), 0.0), dict(transform=(0, 7)))):
        with pytest.raises(tpt.TptError) as e:
            tpt.plan_create(*args, **kw)
        assert e.value.status == -1
    L = tpt.lib()
    assert L.tpt_project(None, None, None, None, 1.0, None, None, 0.0, 7, None) == -1
    assert L.tpt_divergence(None, None, None, None, 1.0, None, None) == -1
    assert L.tpt_solve(None, None, None, None) == -1
    assert L.tpt_solve_static_scratch(None, None, None, None) == -1
    assert tpt.STATIC_SCRATCH_POINTS == 16384 and "#define TPT_STATIC_SCRATCH_POINTS 16384" in open(os.path.join(ROOT, "include", "tpt.h")).read()
    assert L.tpt_debug_sweep_geometry(512, 1, 0, None) == -1
    assert L.tpt_plan_destroy(None) == 0
    assert L.tpt_plan_is_singular(None) == -1


def test_no_cpu_fallback_without_a_device(tpt):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    good = np.linspace(0, 1, 9)
    with pytest.raises(tpt.TptError) as e:
        tpt.plan_create(8, 8, 8, good, good, good, (0, 0, 1), 0.0)
    assert e.value.status == -3          # TPT_ECUDA: fails loudly, no fallback


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2603_09528_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".hpp", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "tpt_oracle" not in src and "import oracle" not in src and "from oracle" not in src, f
    orc = os.path.join(ROOT, "oracle")
    for f in os.listdir(orc):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(orc, f)).read()
            assert "paper_2603_09528_b200" not in src.replace("under paper_2603_09528_b200/", ""), f
            assert "tpt.h" not in src, f


def test_shard_layout_partitions_planes_and_mode_rows():
    # tpt_shard_layout is host-only: the z-slabs tile [0, nz) with even boundaries, the mode rows tile [0, ny) in units of
    # 16, the symmetric allocation is sized for the largest rank, and the NVLink byte count is what leaves the rank
    # (every element of the mode-space field crosses once per exchange, except the part that stays).
    from paper_2603_09528_b200 import api

    for (nx, ny, nz, P) in [(512, 512, 512, 8), (1024, 256, 512, 8), (128, 128, 21, 5), (256, 128, 35, 3), (128, 256, 300, 8),
                            (128, 128, 16, 1), (768, 768, 768, 7), (1024, 1024, 1024, 8), (128, 64, 30, 3), (256, 32, 16, 2)]:
        lays = [api.shard_layout(P, r, nx, ny, nz) for r in range(P)]
        assert lays[0].k0 == 0 and lays[-1].k1 == nz and lays[0].m0 == 0 and lays[-1].m1 == ny
        sent = 0
        for r, l in enumerate(lays):
            assert (l.rank, l.nranks) == (r, P)
            assert l.k0 % 2 == 0 and l.k1 > l.k0 and l.m0 % 16 == 0 and l.m1 > l.m0 and (l.m1 - l.m0) % 16 == 0
            if r:
                assert l.k0 == lays[r - 1].k1 and l.m0 == lays[r - 1].m1
            assert l.slab_points == nx * ny * (l.k1 - l.k0)
            assert l.mode_bytes == 8 * nx * nz * max(q.m1 - q.m0 for q in lays)
            assert l.slab_bytes == 8 * nx * ny * max(q.k1 - q.k0 for q in lays)
            assert l.sym_bytes >= l.mode_bytes + l.slab_bytes and l.sym_bytes == lays[0].sym_bytes
            assert l.nvlink_bytes_per_solve == 2 * 8 * nx * (l.m1 - l.m0) * (nz - (l.k1 - l.k0))
            sent += l.nvlink_bytes_per_solve
        # balanced to within one unit
        assert max(q.k1 - q.k0 for q in lays) - min(q.k1 - q.k0 for q in lays) <= 2
        assert max(q.m1 - q.m0 for q in lays) - min(q.m1 - q.m0 for q in lays) <= 16
        if P > 1 and nz % (2 * P) == 0 and ny % (16 * P) == 0:
            assert sent == 2 * 8 * nx * ny * nz * (P - 1) // P
    for bad in [(9, 0, 128, 128, 64), (2, 2, 128, 128, 64), (2, 0, 96, 128, 64), (2, 0, 128, 200, 64), (4, 0, 128, 32, 64), (8, 0, 128, 128, 12),
                (2, 0, 128, 128, 2000)]:
        with pytest.raises(api.TptError):
            api.shard_layout(*bad)
