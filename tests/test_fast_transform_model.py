"""Host-side model of the fast transforms of a uniform direction (csrc/fft.cu): on a
uniform grid the eigenbasis of the 1-D operator is known in closed form — Neumann: DCT-II vectors, Dirichlet: DST-II
vectors, periodic: the real DFT — so Eq. 10 / 12 can be applied in O(N log N).  The kernel family does it with
  * Makhoul's reordering  v_n = f_{2n}, v_{N-1-n} = f_{2n+1},  C_k = Re(e^{-i pi k / 2N} V_k)  for the cosine transform,
  * sine transform = cosine transform of (-1)^i f_i read backwards,
  * two real lines in the real and imaginary parts of one complex FFT, untangled by
        V1_k = (Z_k + conj Z_{N-k}) / 2,   V2_k = (Z_k - conj Z_{N-k}) / 2i,
  * the inverse as the same steps backwards (Hermitian-symmetrised coefficients -> inverse FFT -> real part).
The steps are restated here in numpy (numpy's FFT standing in for the Stockham passes; test code only) and checked against
the explicit orthonormal bases and — for small N — against the ORACLE's eigen-decomposition of the uniform operator, so the
identities the kernels rely on (signs, index reversal, scaling of the special modes) are pinned without a GPU."""
import numpy as np
import pytest

from paper_2603_09528_b200 import inputs as I

N_, D_, P_ = I.NEUMANN, I.DIRICHLET, I.PERIODIC


def basis(n, bc):
    """Orthonormal eigenvectors Q[i, k] of the uniform 1-D operator, mode 0 smoothest (the plan's order), and -lambda Delta^2."""
    i = np.arange(n)[:, None]
    k = np.arange(n)[None, :]
    if bc == N_:
        Q = np.cos(np.pi * k * (2 * i + 1) / (2 * n)) * np.sqrt(2.0 / n)
        Q[:, 0] = np.sqrt(1.0 / n)
        lam = 4.0 * np.sin(np.pi * np.arange(n) / (2 * n)) ** 2
    elif bc == D_:
        Q = np.sin(np.pi * (k + 1) * (2 * i + 1) / (2 * n)) * np.sqrt(2.0 / n)
        Q[:, n - 1] = np.sqrt(1.0 / n) * (-1.0) ** np.arange(n)
        lam = 4.0 * np.sin(np.pi * (np.arange(n) + 1) / (2 * n)) ** 2
    else:   # periodic: 1, then (cos, sin) pairs of wavenumber 1 .. n/2 - 1, then (-1)^i
        Q = np.zeros((n, n)); lam = np.zeros(n)
        Q[:, 0] = np.sqrt(1.0 / n)
        for m in range(1, n // 2):
            Q[:, 2 * m - 1] = np.cos(2 * np.pi * m * np.arange(n) / n) * np.sqrt(2.0 / n)
            Q[:, 2 * m] = np.sin(2 * np.pi * m * np.arange(n) / n) * np.sqrt(2.0 / n)
            lam[2 * m - 1] = lam[2 * m] = 4.0 * np.sin(np.pi * m / n) ** 2
        Q[:, n - 1] = np.sqrt(1.0 / n) * (-1.0) ** np.arange(n)
        lam[n - 1] = 4.0
    return Q, lam


def untangle(Z):
    """Spectra of the two real lines packed as z = v1 + i v2."""
    Zr = np.conj(np.roll(Z[::-1], 1))                   # conj Z_{N-k}, with Z_N = Z_0
    return (Z + Zr) / 2, (Z - Zr) / 2j


def dct2_pair(f1, f2):
    """Unnormalised DCT-II  C_k = sum_i f_i cos(pi k (2i+1) / 2N)  of two lines by ONE complex FFT (Makhoul)."""
    n = len(f1)
    v = np.empty(n, dtype=complex)
    v[: n // 2] = f1[0::2] + 1j * f2[0::2]
    v[n - 1 : n // 2 - 1 : -1] = f1[1::2] + 1j * f2[1::2]
    V1, V2 = untangle(np.fft.fft(v))
    tw = np.exp(-1j * np.pi * np.arange(n) / (2 * n))
    return (tw * V1).real, (tw * V2).real


def forward_pair(f1, f2, bc):
    """Q^T f for two lines (Eq. 10 on a uniform direction), through the fast path's steps."""
    n = len(f1)
    if bc == N_:
        c1, c2 = dct2_pair(f1, f2)
        s = np.full(n, np.sqrt(2.0 / n)); s[0] = np.sqrt(1.0 / n)
        return c1 * s, c2 * s
    if bc == D_:                                        # S_k = C_{N-1-k} of (-1)^i f_i
        sg = (-1.0) ** np.arange(n)
        c1, c2 = dct2_pair(sg * f1, sg * f2)
        s = np.full(n, np.sqrt(2.0 / n)); s[n - 1] = np.sqrt(1.0 / n)
        return c1[::-1] * s, c2[::-1] * s
    F1, F2 = untangle(np.fft.fft(f1 + 1j * f2))         # periodic: the real DFT itself
    out = []
    for F in (F1, F2):
        o = np.empty(n)
        o[0] = F[0].real * np.sqrt(1.0 / n)
        m = np.arange(1, n // 2)
        o[2 * m - 1] = F[m].real * np.sqrt(2.0 / n)
        o[2 * m] = -F[m].imag * np.sqrt(2.0 / n)
        o[n - 1] = F[n // 2].real * np.sqrt(1.0 / n)
        out.append(o)
    return out[0], out[1]


def inverse_pair(g1, g2, bc):
    """Q g for two lines (Eq. 12): the forward steps backwards."""
    n = len(g1)
    if bc == P_:
        Z = np.zeros(n, dtype=complex)
        for g, unit in ((g1, 1.0), (g2, 1j)):
            F = np.zeros(n, dtype=complex)
            F[0] = g[0] * np.sqrt(n)
            m = np.arange(1, n // 2)
            F[m] = (g[2 * m - 1] - 1j * g[2 * m]) * np.sqrt(n / 2.0)
            F[n - m] = np.conj(F[m])                   # Hermitian symmetry of a real line
            F[n // 2] = g[n - 1] * np.sqrt(n)
            Z += unit * F
        z = np.fft.ifft(Z)
        return z.real, z.imag
    if bc == D_:
        s = np.full(n, np.sqrt(2.0 / n)); s[n - 1] = np.sqrt(1.0 / n)
        c1, c2 = (g1 * s)[::-1], (g2 * s)[::-1]
    else:
        s = np.full(n, np.sqrt(2.0 / n)); s[0] = np.sqrt(1.0 / n)
        c1, c2 = g1 * s, g2 * s
    # f_i = sum_k c_k cos(pi k (2i+1) / 2N): rebuild the spectrum of the (real) Makhoul sequence v — Hermitian by construction,
    # V_k = e^{+i pi k / 2N} (c_k - i c_{N-k}) / 2 for k > 0, V_0 = c_0 — then one inverse FFT and the reordering backwards
    k = np.arange(n)
    tw = np.exp(1j * np.pi * k / (2 * n))
    Z = np.zeros(n, dtype=complex)
    for c, unit in ((c1, 1.0), (c2, 1j)):
        cr = np.concatenate(([0.0], c[:0:-1]))          # c_{N-k}, with c_N := 0
        V = tw * (c - 1j * cr)
        V[0] = c[0]
        Z += unit * V * np.where(k == 0, 1.0, 0.5)
    v = np.fft.ifft(Z) * n                              # v_n = sum_k V_k e^{2 pi i k n / N}
    f = np.empty(n, dtype=complex)
    f[0::2] = v[: n // 2]
    f[1::2] = v[n - 1 : n // 2 - 1 : -1]
    sg = (-1.0) ** np.arange(n) if bc == D_ else 1.0
    return f.real * sg, f.imag * sg


@pytest.mark.parametrize("bc", [N_, D_, P_], ids=["neumann", "dirichlet", "periodic"])
@pytest.mark.parametrize("n", [16, 64, 512, 2048])
def test_fast_path_steps_equal_the_eigenbasis_transforms(n, bc):
    rng = np.random.default_rng(n + 7 * bc)
    Q, _ = basis(n, bc)
    assert np.abs(Q.T @ Q - np.eye(n)).max() < 1e-12
    f1, f2 = rng.uniform(-1, 1, n), rng.uniform(-1, 1, n)
    g1, g2 = forward_pair(f1, f2, bc)
    assert np.abs(g1 - Q.T @ f1).max() < 1e-12 and np.abs(g2 - Q.T @ f2).max() < 1e-12
    h1, h2 = inverse_pair(g1, g2, bc)
    assert np.abs(h1 - f1).max() < 1e-12 and np.abs(h2 - f2).max() < 1e-12
    a1, a2 = inverse_pair(f1, f2, bc)                   # the inverse on arbitrary coefficients is Q itself
    assert np.abs(a1 - Q @ f1).max() < 1e-12 and np.abs(a2 - Q @ f2).max() < 1e-12


@pytest.mark.parametrize("bc", [N_, D_, P_], ids=["neumann", "dirichlet", "periodic"])
def test_closed_form_basis_is_the_oracles_eigenbasis_on_a_uniform_grid(orc, bc):
    # the plan uses the analytical eigenvalues -(4 / Delta^2) sin^2(.) and the closed-form basis for an FFT direction: both
    # must be what the oracle's eigen-solver finds for the uniform operator (eigenvectors up to sign; the periodic cos / sin
    # pairs up to a rotation inside their two-dimensional eigenspaces)
    n, L = 32, 2.0
    xf = np.linspace(0.0, L, n + 1)
    lam, Qo = orc.eig_1d(xf, bc)[:2]
    Q, mu = basis(n, bc)
    delta = L / n
    assert np.abs(np.asarray(lam) - (-mu / delta ** 2)).max() <= 1e-10 * mu.max() / delta ** 2
    Qo = np.asarray(Qo).reshape(n, n)
    if bc == P_:
        for m in range(1, n // 2):                      # projector onto each eigenspace
            Pa = Q[:, 2 * m - 1 : 2 * m + 1] @ Q[:, 2 * m - 1 : 2 * m + 1].T
            Pb = Qo[:, 2 * m - 1 : 2 * m + 1] @ Qo[:, 2 * m - 1 : 2 * m + 1].T
            assert np.abs(Pa - Pb).max() < 1e-10
        assert abs(abs(Q[:, 0] @ Qo[:, 0]) - 1) < 1e-12 and abs(abs(Q[:, n - 1] @ Qo[:, n - 1]) - 1) < 1e-12
    else:
        assert np.abs(np.abs(np.sum(Q * Qo, axis=0)) - 1.0).max() < 1e-10
