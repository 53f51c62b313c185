"""Host-side model of the on-chip z sweep's algebra (csrc/thomas_onchip.cu; A13, §5.2): the Thomas elimination of
Eq. 11 re-associated into  (1) a cold forward elimination per segment of M rows that carries the fill-in
towards the previous segment's last unknown,  (2) a tridiagonal system in the S segment-end unknowns solved by parallel
cyclic reduction with an early exit,  (3) back substitution per segment.  The model restates the kernel's formulas line by
line in numpy (test code only: neither the product nor the oracle uses it) and is checked against a dense solve — so the
claims the design rests on are pinned without a GPU: the re-association is exact up to rounding for any segment length and
ragged tail, the padded rows [a, b, c] = [0, -1, 0] are inert, the early exit at 1e-30 cannot change an FP64 result, the
null column's "last unknown = 0" comes out of the replaced last row, and the product a_k c_{k-1} formed from
the previous row's c is the table's entry bit for bit."""
import numpy as np
import pytest


def _operator(nz, rng, stretch=3.0):
    """A stretched-grid 1-D Laplacian in the paper's finite-volume form (Eq. 3-4): rows a_k, b_k, c_k (Neumann ends)."""
    dz = np.diff(np.tanh(stretch * np.linspace(-1, 1, nz + 1)) / np.tanh(stretch))
    dz *= 1.0 + 0.05 * rng.uniform(-1, 1, nz)
    dc = 0.5 * (dz[1:] + dz[:-1])                       # centre spacings at the interior faces
    a = np.zeros(nz); c = np.zeros(nz)
    a[1:] = 1.0 / (dz[1:] * dc)
    c[:-1] = 1.0 / (dz[:-1] * dc)
    return a, -(a + c), c


def partitioned_sweep(a, b, c, p, s, M, null_col=False, exit_below=1e-30, rounds_out=None):
    """x with (T + s I) x = p, the way thomas_onchip_kernel computes it (one 'thread' per segment, same formulas)."""
    nz = len(p)
    S = -(-nz // M)
    rows = S * M
    # tables as thomas_onchip_tables pads them; the null column's last equation becomes "-x = p" with p zeroed
    A_ = np.zeros(rows); B_ = -np.ones(rows); C_ = np.zeros(rows); P_ = np.zeros(rows)
    A_[:nz], B_[:nz], C_[:nz], P_[:nz] = a, b, c, p
    if null_col:
        A_[nz - 1], B_[nz - 1], C_[nz - 1], P_[nz - 1] = 0.0, -1.0, 0.0, 0.0
    AC = np.zeros(rows); AC[1:] = A_[1:] * C_[:-1]
    cp = np.zeros((S, M)); g = np.zeros((S, M)); d = np.zeros((S, M))
    DD = np.zeros(S); GG = np.zeros(S); PI = np.ones(S)
    for seg in range(S):                                 # ---- 1. cold forward elimination
        pi, dd, gg, dprev, rprev = 1.0, 0.0, 0.0, 0.0, 0.0
        for t in range(M):
            k = seg * M + t
            bb = B_[k] + s
            den = bb if t == 0 else bb - AC[k] * rprev
            r = 1.0 / den
            cp[seg, t] = C_[k] * r
            d[seg, t] = (P_[k] if t == 0 else P_[k] - A_[k] * dprev) * r
            g[seg, t] = (A_[k] if t == 0 else -A_[k] * g[seg, t - 1]) * r
            if t < M - 1:
                dd += pi * d[seg, t]
                gg += pi * g[seg, t]
                pi = -pi * cp[seg, t]
            dprev, rprev = d[seg, t], r
        DD[seg], GG[seg], PI[seg] = dd, gg, pi
    # ---- 2. reduced system  X_s + A X_{s-1} + C X_{s+1} = D  in the segments' last unknowns, by parallel cyclic reduction
    A = g[:, M - 1].copy(); C = np.zeros(S); D = d[:, M - 1].copy()
    for seg in range(S):
        Bd = 1.0
        if seg + 1 < S:
            cl = cp[seg, M - 1]
            Bd = 1.0 - cl * GG[seg + 1]
            C[seg] = cl * PI[seg + 1]
            D[seg] = D[seg] - cl * DD[seg + 1]
        A[seg] /= Bd; C[seg] /= Bd; D[seg] /= Bd
    dlt, rounds = 1, 0
    while dlt < S:
        if not (np.maximum(np.abs(A), np.abs(C)) > exit_below).any():
            break
        Al = np.zeros(S); Cl = np.zeros(S); Dl = np.zeros(S); Ah = np.zeros(S); Ch = np.zeros(S); Dh = np.zeros(S)
        Al[dlt:], Cl[dlt:], Dl[dlt:] = A[:-dlt], C[:-dlt], D[:-dlt]
        Ah[:-dlt], Ch[:-dlt], Dh[:-dlt] = A[dlt:], C[dlt:], D[dlt:]
        rB = 1.0 / (1.0 - A * Cl - C * Ah)
        D = (D - A * Dl - C * Dh) * rB
        A, C = -A * Al * rB, -C * Ch * rB
        dlt *= 2; rounds += 1
    if rounds_out is not None:
        rounds_out.append(rounds)
    X = D
    # ---- 3. back substitution
    x = np.zeros(rows)
    for seg in range(S):
        xl = X[seg - 1] if seg > 0 else 0.0
        xk = X[seg]
        x[seg * M + M - 1] = xk
        for t in range(M - 2, -1, -1):
            xk = d[seg, t] - g[seg, t] * xl - cp[seg, t] * xk
            x[seg * M + t] = xk
    return x[:nz], x[nz:]


def _dense(a, b, c, s):
    return np.diag(b + s) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)


@pytest.mark.parametrize("nz,M", [(16, 16), (17, 8), (100, 17), (512, 17), (513, 19), (300, 25), (768, 25), (1000, 21), (37, 8)])
def test_partitioned_sweep_equals_the_dense_solve(nz, M):
    rng = np.random.default_rng(nz * 31 + M)
    a, b, c = _operator(nz, rng)
    scale = np.abs(b).max()
    for s in (-1e-6 * scale, -0.01 * scale, -0.3 * scale, -5.0 * scale):      # low to high (kx, ky) modes: lam_x + lam_y <= 0
        p = rng.uniform(-1, 1, nz)
        x, pad = partitioned_sweep(a, b, c, p, s, M)
        ref = np.linalg.solve(_dense(a, b, c, s), p)
        assert np.abs(x - ref).max() <= 2e-12 * max(np.abs(ref).max(), 1e-300) * max(1.0, abs(scale / s) ** 0.5), (nz, M, s)
        assert np.all(pad == 0.0)                           # decoupled identity rows with p = 0 stay exactly zero


def test_early_exit_of_the_cyclic_reduction_changes_nothing():
    rng = np.random.default_rng(5)
    nz, M = 512, 17
    a, b, c = _operator(nz, rng)
    scale = np.abs(b).max()
    seen = []
    for s in (-1e-7 * scale, -1e-3 * scale, -0.05 * scale, -0.5 * scale, -4.0 * scale):
        p = rng.uniform(-1, 1, nz)
        r_exit, r_full = [], []
        x_exit, _ = partitioned_sweep(a, b, c, p, s, M, exit_below=1e-30, rounds_out=r_exit)
        x_full, _ = partitioned_sweep(a, b, c, p, s, M, exit_below=-1.0, rounds_out=r_full)
        assert np.array_equal(x_exit, x_full), s            # bit for bit
        assert r_full == [5] and r_exit[0] <= 5
        seen.append(r_exit[0])
    assert seen[0] == 5 and seen[-1] < 5 and sorted(seen, reverse=True) == seen     # high modes decouple after fewer rounds


@pytest.mark.parametrize("nz,M", [(64, 17), (512, 17), (130, 16)])
def test_null_column_gets_last_unknown_zero(nz, M):
    # s = 0 on the all-Neumann operator: singular; the replaced last row pins x_{nz-1} = 0 and the other
    # rows are solved exactly — the result differs from any other solution by a constant
    rng = np.random.default_rng(nz)
    a, b, c = _operator(nz, rng)
    x_true = rng.uniform(-1, 1, nz)
    T = _dense(a, b, c, 0.0)
    p = T @ x_true                                         # compatible right-hand side
    x, _ = partitioned_sweep(a, b, c, p, 0.0, M, null_col=True)
    assert x[-1] == 0.0
    shift = x - x_true
    assert np.abs(shift - shift.mean()).max() <= 1e-9 * np.abs(x_true).max()
    assert np.abs((T @ x - p)[:-1]).max() <= 1e-9 * np.abs(p).max()


def test_product_formed_from_the_previous_row_is_the_table_entry():
    # DESIGN.md 5.2 (next step): a_k c_{k-1} computed in the kernel by one rounded multiply equals the host table's entry
    rng = np.random.default_rng(9)
    a, b, c = _operator(777, rng)
    table = np.zeros(777); table[1:] = a[1:] * c[:-1]
    formed = np.array([0.0] + [float(np.float64(a[k]) * np.float64(c[k - 1])) for k in range(1, 777)])
    assert np.array_equal(table, formed)
