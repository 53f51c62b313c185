"""Pins for the seeded input generators (paper_2603_09528_b200/inputs.py)."""
import math
import os

import numpy as np

from paper_2603_09528_b200 import inputs as I

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as fh:
        return [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]


def test_grading_ratios_match_paper_footnote4():
    # pins Eq. 13 AND the reading that the mapping is applied to cell faces [A2].
    for n, alpha, ratio, tol in _rows("grading_ratios.txt"):
        xf = I.tanh_faces(int(n), 1.0, float(alpha) / 2.0)      # beta = alpha/2 [A15]
        w = np.diff(xf)
        assert abs(w.max() / w.min() - float(ratio)) < float(tol)
        # node-mapped alternative (cell centres on the tanh curve) would NOT give the printed digits
        xi = (np.arange(int(n)) + 0.5) / int(n)
        xc = 0.5 * (1 + np.tanh(float(alpha) * (xi - 0.5)) / math.tanh(float(alpha) / 2))
        dn = np.diff(xc)
        assert abs(dn.max() / dn.min() - float(ratio)) > float(tol)


def test_large_n_ratio_tends_to_cosh2():
    # PAPER.md:276 footnote 1
    for beta in (1.0, 2.0, 3.0):
        w = np.diff(I.tanh_faces(1 << 15, 1.0, beta))
        assert abs(w.max() / w.min() / math.cosh(beta) ** 2 - 1.0) < 2e-3


def test_uniform_limit_and_endpoints():
    xf = I.tanh_faces(10, 8.0, 0.0)
    assert np.array_equal(xf, 8.0 * np.arange(11) / 10)
    xf = I.tanh_faces(37, 2.5, 1.7)
    assert xf[0] == 0.0 and xf[-1] == 2.5 and np.all(np.diff(xf) > 0)
    # symmetric clustering at both ends
    assert np.allclose(np.diff(xf), np.diff(xf)[::-1], rtol=1e-12)


def test_rhs_generator_is_counter_based_and_uniform():
    a = I.uniform_pm1(3, 1000)
    b = np.concatenate([I.uniform_pm1(3, 400), I.uniform_pm1(3, 600, offset=400)])
    assert np.array_equal(a, b)
    assert not np.array_equal(a, I.uniform_pm1(4, 1000))
    u = I.uniform_pm1(2, 1 << 20)
    assert u.min() >= -1.0 and u.max() < 1.0
    assert abs(u.mean()) < 4e-3 and abs((u * u).mean() - 1 / 3) < 4e-3
    # chunking does not change the stream
    assert np.array_equal(I.uniform_pm1(5, 5000, chunk=777), I.uniform_pm1(5, 5000))


def test_weighted_mean_removed_for_singular_configs_only():
    P = I.Problem("t", (12, 10, 8), (1.0, 2.0, 3.0), (2.0, 1.0, 1.5), (0, 0, 0), 0.0, 9)
    xf, yf, zf = P.faces()
    f = P.rhs()
    V = np.diff(zf)[:, None, None] * np.diff(yf)[None, :, None] * np.diff(xf)[None, None, :]
    assert abs((V * f).sum()) < 1e-14 * V.sum()
    assert abs(f.mean()) > 1e-6            # plain mean is NOT what is removed [A8]
    Q = I.Problem("t", (12, 10, 8), (1.0, 2.0, 3.0), (2.0, 1.0, 1.5), (0, 0, 1), 0.0, 9)
    assert np.array_equal(Q.rhs().ravel(), I.uniform_pm1(9, 12 * 10 * 8))


def test_configs_match_baseline_json():
    c = I.CONFIGS
    assert c["c1"][0].n == (16, 16, 16) and c["c1"][0].bc == (0, 0, 1) and c["c1"][0].beta == (1.2, 1.2, 1.5)
    assert c["c2"][0].n == (128, 128, 128) and c["c2"][0].alpha == 1e-3 and c["c2"][0].seed == 1
    assert c["c3"][0].n == (512, 512, 512) and c["c3"][0].singular and c["c3"][0].seed == 2
    assert c["c4"][0].n == (1024, 256, 512) and c["c4"][0].beta[0] == 0.0 and c["c4"][0].length == (8.0, 2.0, 2.0)
    assert [p.seed for p in c["c5"]] == [4, 5, 6, 7] and c["c5"][3].singular and c["c5"][0].alpha == 5e-4
