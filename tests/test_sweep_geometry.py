"""Host-side check of the z sweep's launch geometry (csrc/thomas_onchip.cu: choose_shape / thomas_geometry) for EVERY column
length the on-chip kernel takes (step 2.3): the constraints a wrong shape would break on the GPU — TMA box
alignment, shared-memory and register budgets, whole warps, table size — are arithmetic, so they are checked here without
a device, through tpt_debug_sweep_geometry."""
import pytest

SMEM_PER_SM, SMEM_CTA_MAX, CTA_RESERVED = 228 * 1024, 227 * 1024, 1024
TABLE_PAD = 160          # THOMAS_TABLE_PAD (kernels.cuh)
REGS_PER_SM = 65536
REGS_PER_THREAD = 128    # __launch_bounds__ of every instantiation leaves at most this


@pytest.fixture(scope="module")
def tpt():
    from paper_2603_09528_b200 import api

    api.lib()
    return api


def _all(tpt):
    for nz in range(2, 1057):
        for blocked, sharded in ((False, False), (True, False), (True, True)):
            g = tpt.debug_sweep_geometry(nz, blocked, sharded)
            assert g is not None, (nz, blocked, sharded)
            yield nz, blocked, sharded, g


def test_every_column_length_has_a_valid_launch_shape(tpt):
    for nz, blocked, sharded, g in _all(tpt):
        where = (nz, blocked, sharded, g)
        M, tc, S = g["M"], g["cols"], g["S"]
        assert tc in (4, 8, 16) and 16 % tc == 0, where
        assert S * M >= nz and (S - 1) * M < nz + 8 * M, where                 # the segments cover the column
        assert (S * tc) % 32 == 0 and g["threads"] == S * tc <= g["max_threads"] <= 1024, where
        # TMA boxes: at most 256 rows, 128-byte multiples in shared memory, together covering the column, none fully outside
        row_bytes = tc * 8
        assert 1 <= g["box_rows"] <= 256 and (g["box_rows"] * row_bytes) % 128 == 0, where
        assert g["nbox"] * g["box_rows"] >= nz > (g["nbox"] - 1) * g["box_rows"], where
        assert g["buf_rows"] >= g["nbox"] * g["box_rows"] and (g["buf_rows"] * row_bytes) % 128 == 0, where
        if g["ctas_per_sm"] == 1:                                              # no pad-row predicates: all S*M rows exist
            assert g["buf_rows"] >= S * M, where
        # shared memory: ring + scratch (+ table) per CTA, CTAs per SM within the SM's 228 KB
        assert g["nbuf"] in (2, 3), where
        table = ((S + 3) // 4 * 4) * M * 32 if g["table_in_smem"] else 0
        assert g["smem"] == g["nbuf"] * g["buf_rows"] * row_bytes + 6 * S * tc * 8 + 128 + table, where
        assert g["smem"] <= SMEM_CTA_MAX and g["ctas_per_sm"] * (g["smem"] + CTA_RESERVED) <= SMEM_PER_SM, where
        # registers and the tables' padding
        assert g["ctas_per_sm"] * g["threads"] * REGS_PER_THREAD <= REGS_PER_SM, where
        assert ((S + 3) // 4 * 4) * M <= nz + TABLE_PAD, where
        if sharded:                                                            # even slab boundaries: rows of >= 64 bytes
            assert tc >= 8, where
        if tc == 4:
            assert S % 8 == 0 and M in (17, 19) and g["ctas_per_sm"] == 4 and blocked, where


def test_partitions_agree_between_the_plain_and_the_sharded_sweep(tpt):
    # one table per (nz, layout): the 4-column shape of the plain sweep and the 8-column shape of the sharded one must cut
    # the column into the same segments
    for nz in range(2, 1057):
        a, b = tpt.debug_sweep_geometry(nz, True, False), tpt.debug_sweep_geometry(nz, True, True)
        assert (a["M"], a["S"]) == (b["M"], b["S"]), (nz, a, b)


def test_known_shapes(tpt):
    g = tpt.debug_sweep_geometry(512, True)            # the bench shape: 4-column tiles, four CTAs, table in shared memory
    assert (g["M"], g["cols"], g["ctas_per_sm"], g["table_in_smem"], g["S"], g["threads"]) == (17, 4, 4, 1, 32, 128)
    g = tpt.debug_sweep_geometry(512, True, True)      # sharded: 8-column tiles
    assert (g["M"], g["cols"], g["ctas_per_sm"], g["table_in_smem"]) == (17, 8, 2, 1)
    g = tpt.debug_sweep_geometry(768, True)
    assert (g["M"], g["cols"], g["ctas_per_sm"], g["table_in_smem"]) == (25, 8, 2, 0)
    g = tpt.debug_sweep_geometry(1024, True)
    assert (g["M"], g["cols"], g["ctas_per_sm"], g["nbuf"], g["threads"]) == (17, 8, 1, 2, 512)
    g = tpt.debug_sweep_geometry(512, False)           # natural layout (tpt_stage, z-only plans)
    assert (g["M"], g["cols"], g["ctas_per_sm"]) == (16, 16, 1)
    assert tpt.debug_sweep_geometry(1, True) is None and tpt.debug_sweep_geometry(1057, True) is None
    assert tpt.lib().tpt_debug_sweep_geometry(512, 0, 1, (__import__("ctypes").c_int * 12)()) == -1   # sharded needs blocked


def test_every_shape_the_dispatcher_can_choose_is_instantiated(tpt):
    # dispatch() matches the chosen shape against a list of template instantiations (TPT_TRY in thomas_onchip.cu) and fails
    # with cudaErrorInvalidConfiguration on a miss: every reachable (M, columns, thread limit, CTAs, table in shared memory)
    # must be in that list — for the sharded store, outside the `if constexpr (!SH)` block of 4-column shapes
    import os
    import re

    src = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_2603_09528_b200", "csrc",
                            "thomas_onchip.cu")).read()
    body = src[src.index("#define TPT_TRY"):src.index("#undef TPT_TRY")]
    listed = {(int(m), int(tc), int(mt), int(c), ts == "true")
              for m, tc, mt, c, ts in re.findall(r"TPT_TRY\((\d+), (\d+), (\d+), (\d+), (true|false)\)", body)}
    assert len(listed) >= 15
    plain_only = {s for s in listed if s[1] == 4}
    for nz, blocked, sharded, g in _all(tpt):
        shape = (g["M"], g["cols"], g["max_threads"], g["ctas_per_sm"], bool(g["table_in_smem"]))
        assert shape in listed, (nz, blocked, sharded, shape)
        if sharded:
            assert shape not in plain_only, (nz, shape)
