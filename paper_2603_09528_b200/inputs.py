"""Seeded synthetic input generators (grids and right-hand sides).

This module is the ONLY code shared by the CUDA path's harness and the CPU oracle's tests.
It holds none of the solver's arithmetic: it produces face coordinates (the paper's tanh
mapping, Eq. 13) and white-noise right-hand sides ("white-noise"
fields), exactly as BASELINE.json `configs` prescribes.  Pure numpy; imports neither the CUDA
binding nor the oracle.

Recipe (also stated in DESIGN.md §Inputs):
  * faces  x_i = L/2 * (1 + tanh(beta*(2 i/N - 1)) / tanh(beta)),  i = 0..N   (Eq. 13 with
    alpha = 2*beta, applied to the cell FACES — reading A2/A15); beta = 0 -> x_i = L*i/N exactly.
  * rhs[idx] = 2*u - 1,  u = top 53 bits of splitmix64-finaliser(idx + (seed+1)*0x9E3779B97F4A7C15 mod 2^64) * 2^-53, a pure
    function of (seed, linear index idx = i + nx*(j + ny*k)), so any consumer reproduces the
    same bits without exchanging files.
  * all-Neumann Poisson configs: the cell-VOLUME-weighted mean is removed from the rhs
    (compatibility, reading A8: the left null vector of T is the cell volume).
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

NEUMANN = 0
DIRICHLET = 1
PERIODIC = 2      # any direction (z: cyclic sweep, A19); the paper's benchmark BCs are periodic x, Neumann y, z

_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def tanh_faces(n: int, length: float, beta: float) -> np.ndarray:
    """n+1 face coordinates on [0, length], clustered at both ends (Eq. 13)."""
    i = np.arange(n + 1, dtype=np.float64)
    if beta == 0.0:
        x = length * (i / n)
    else:
        x = 0.5 * length * (1.0 + np.tanh(beta * (2.0 * i / n - 1.0)) / math.tanh(beta))
    x[0] = 0.0
    x[n] = length
    return x


def uniform_pm1(seed: int, count: int, offset: int = 0, chunk: int = 1 << 24) -> np.ndarray:
    """count i.i.d. uniform[-1,1) doubles: element t is a pure function of (seed, offset+t)."""
    out = np.empty(count, dtype=np.float64)
    base = np.uint64(((int(seed) + 1) * 0x9E3779B97F4A7C15) & 0xFFFFFFFFFFFFFFFF)
    with np.errstate(over="ignore"):
        for s in range(0, count, chunk):
            e = min(count, s + chunk)
            z = np.arange(offset + s, offset + e, dtype=np.uint64) + base
            z ^= z >> np.uint64(30)
            z *= _M1
            z ^= z >> np.uint64(27)
            z *= _M2
            z ^= z >> np.uint64(31)
            z >>= np.uint64(11)
            out[s:e] = z.astype(np.float64) * (2.0 ** -52) - 1.0
    return out


def remove_weighted_mean(f: np.ndarray, xf: np.ndarray, yf: np.ndarray, zf: np.ndarray) -> np.ndarray:
    """f -= sum(V f)/sum(V), V = cell volumes; f has shape (nz, ny, nx). In place; returns f."""
    wx, wy, wz = np.diff(xf), np.diff(yf), np.diff(zf)
    # plane sums first (keeps temporaries small at 768^3)
    s = 0.0
    for k in range(f.shape[0]):
        s += wz[k] * float(wy @ (f[k] @ wx))
    vol = float(wx.sum() * wy.sum() * wz.sum())
    f -= s / vol
    return f


@dataclasses.dataclass(frozen=True)
class Problem:
    """One elliptic problem: grid, BCs, Helmholtz alpha (0 = Poisson) and rhs seed."""
    name: str
    n: tuple            # (nx, ny, nz)
    length: tuple       # (Lx, Ly, Lz)
    beta: tuple         # tanh beta per direction (0 = uniform)
    bc: tuple           # (bc_x, bc_y, bc_z) in {NEUMANN, DIRICHLET, PERIODIC}
    alpha: float        # 0 -> Poisson  L phi = f ; > 0 -> (I - alpha L) u = f
    seed: int

    @property
    def singular(self) -> bool:
        return self.alpha == 0.0 and all(b != DIRICHLET for b in self.bc)

    @property
    def points(self) -> int:
        return self.n[0] * self.n[1] * self.n[2]

    def faces(self):
        return tuple(tanh_faces(self.n[d], self.length[d], self.beta[d]) for d in range(3))

    def rhs(self) -> np.ndarray:
        """rhs with shape (nz, ny, nx), x contiguous; weighted mean removed iff singular."""
        nx, ny, nz = self.n
        f = uniform_pm1(self.seed, nx * ny * nz).reshape(nz, ny, nx)
        if self.singular:
            remove_weighted_mean(f, *self.faces())
        return f

    def thin_z(self, nz: int) -> "Problem":
        """Same x/y grids and BCs, only nz cells in z (same Lz, beta_z): a bounded sample whose
        per-point transform work equals the full problem's."""
        return dataclasses.replace(self, name=f"{self.name}-thinz{nz}", n=(self.n[0], self.n[1], nz))


N_, D_ = NEUMANN, DIRICHLET
_PI = math.pi

# The paper's own single-GPU benchmark case: 1024^3, periodic x, Neumann y and z, GEMM transforms
# in x and y ("GG").  x uniform (the paper's FFT-vs-GEMM comparison needs it), y and z tanh-stretched here (the cost of
# the direct method does not depend on the grading).  Not a BASELINE.json config: context for BASELINE.md.
PAPER_GG = Problem("paper-gg-1024-periodic-x", (1024, 1024, 1024), (1.0, 1.0, 1.0), (0.0, 2.0, 2.0),
                   (PERIODIC, NEUMANN, NEUMANN), 0.0, 8)

# BASELINE.json `configs`, in order.  Config 5 is a step of four solves (3 Helmholtz + 1 Poisson).
CONFIGS = {
    "c1": [Problem("c1-poisson-16", (16, 16, 16), (1.0, 1.0, 1.0), (1.2, 1.2, 1.5), (N_, N_, D_), 0.0, 0)],
    "c2": [Problem("c2-helmholtz-128", (128, 128, 128), (2 * _PI, _PI, 2.0), (2.0, 2.0, 2.5), (N_, N_, D_), 1e-3, 1)],
    "c3": [Problem("c3-poisson-512-neumann", (512, 512, 512), (1.0, 1.0, 1.0), (2.0, 2.0, 2.0), (N_, N_, N_), 0.0, 2)],
    "c4": [Problem("c4-poisson-1024x256x512", (1024, 256, 512), (8.0, 2.0, 2.0), (0.0, 2.5, 3.0), (N_, N_, D_), 0.0, 3)],
    "c5": [Problem(f"c5-helmholtz-768-{s}", (768, 768, 768), (1.0, 1.0, 1.0), (3.0, 3.0, 3.0), (N_, N_, D_), 5e-4, s)
           for s in (4, 5, 6)]
          + [Problem("c5-poisson-768-neumann", (768, 768, 768), (1.0, 1.0, 1.0), (3.0, 3.0, 3.0), (N_, N_, N_), 0.0, 7)],
    "p1024": [PAPER_GG],
    # the same case with y uniform as well, so that all four transform variants FF / FG / GF / GG
    # can be timed on one grid (bench.py --transform)
    # 512^3 with uniform x and y (Neumann) and a stretched z (Dirichlet): the grid on which the FF variant is profiled
    "ff512": [Problem("ff512-poisson-uniform-xy", (512, 512, 512), (8.0, 2.0, 2.0), (0.0, 0.0, 3.0), (N_, N_, D_), 0.0, 9)],
    "p1024u": [dataclasses.replace(PAPER_GG, name="paper-1024-periodic-x-uniform-xy", beta=(0.0, 0.0, 2.0))],
}
