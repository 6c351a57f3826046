"""Seeded synthetic inputs for the five BASELINE.json configs (C1..C5; C4 split into C4a/C4b).

This module is the ONE thing the oracle-side tests and the CUDA-side tests/bench share.  It holds none of the
method's arithmetic: no sphere test, no FFT, no Coulomb kernel.  It describes the cells (lattice vectors, grids,
k-meshes, occupations, kernel parameters — DESIGN.md section 4, the input recipe) and draws the seeded
plane-wave coefficients once the caller tells it how many plane waves each k-point has (the caller gets `npw`
from whichever implementation it is driving).

The workloads stand in for the paper's boron cells (Table I: hR12, hR12x8, hR105, aP107); the
real structures, VASP and PAW data are not available, so shapes/sizes/occupation patterns are synthetic.
"""
import itertools
import math
from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 11110716


def cubic(a):
    return a * np.eye(3)


def rhombohedral(a, alpha_deg):
    """Rows a_i = a (s cos(2 pi i/3), s sin(2 pi i/3), h): |a_i| = a, a_i.a_j = a^2 cos(alpha), 3-fold axis along z."""
    c = math.cos(math.radians(alpha_deg))
    s = math.sqrt(2.0 * (1.0 - c) / 3.0)
    h = math.sqrt((1.0 + 2.0 * c) / 3.0)
    return a * np.array([[s * math.cos(2.0 * math.pi * i / 3.0), s * math.sin(2.0 * math.pi * i / 3.0), h] for i in range(3)])


def monkhorst_pack(n):
    """kappa = (2r - n - 1)/(2n), r = 1..n, per axis; first axis slowest.  n = 2 gives +-1/4 (Gamma-free)."""
    v = [(2.0 * r - n - 1.0) / (2.0 * n) for r in range(1, n + 1)]
    return np.array(list(itertools.product(v, v, v)), dtype=np.float64)


@dataclass
class Workload:
    name: str
    seed: int
    grid: tuple
    lattice: np.ndarray          # rows a_i, bohr
    kfrac: np.ndarray            # (nk, 3) fractional reciprocal coordinates
    kweight: np.ndarray          # (nk,), sums to 1
    ecut: float                  # Hartree
    kernel_kind: int             # 0 bare Coulomb (q+G=0 term := 0), 1 HSE short range (q+G=0 term := pi/mu^2)
    mu: float
    scale: float
    nbands: int
    occ_per_k: np.ndarray        # (nbands,)
    description: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def nk(self):
        return len(self.kweight)

    @property
    def occ(self):
        return np.tile(self.occ_per_k, self.nk).astype(np.float64)

    @property
    def ng(self):
        return int(self.grid[0]) * int(self.grid[1]) * int(self.grid[2])

    @property
    def nocc(self):
        return int(np.count_nonzero(self.occ_per_k))

    @property
    def pair_evals(self):
        """Ordered band-pair exchange evaluations per V_x application: Nk^2 * Nb * Nocc."""
        return self.nk * self.nk * self.nbands * self.nocc

    def coefficients(self, npw):
        """Reading A17: rng = default_rng(seed); for k in order: re = N(0,1)[Nb,Npw_k], then im likewise; c = re + i im;
        each band divided by its 2-norm.  Returns the packed psi array (k-major, band, sphere index), complex128."""
        assert len(npw) == self.nk
        rng = np.random.default_rng(self.seed)
        parts = []
        for k in range(self.nk):
            re = rng.standard_normal((self.nbands, int(npw[k])))
            im = rng.standard_normal((self.nbands, int(npw[k])))
            x = re + 1j * im
            x /= np.sqrt((np.abs(x) ** 2).sum(axis=1))[:, None]
            parts.append(x.reshape(-1))
        return np.concatenate(parts)


def _gamma():
    return np.zeros((1, 3)), np.ones(1)


def _mp2():
    k = monkhorst_pack(2)
    return k, np.full(len(k), 1.0 / len(k))


def make(name):
    """C1, C2, C3, C4a, C4b, C5 — BASELINE.json configs[0..4] (C4's k-set split per DESIGN.md reading A12)."""
    HSE_MU = 0.106
    if name == "C1":
        k, w = _gamma()
        return Workload("C1", SEED_BASE + 1, (16,) * 3, cubic(10.0), k, w, 6.0, 0, 0.0, 1.0, 8, np.ones(8),
                        "tiny exchange check: sc a=10, 16^3, Gamma, 8 bands f=1, bare Coulomb")
    if name == "C2":
        k, w = _mp2()
        return Workload("C2", SEED_BASE + 2, (48,) * 3, rhombohedral(9.55, 58.0), k, w, 15.0, 0, 0.0, 1.0, 24,
                        np.r_[np.ones(18), np.zeros(6)],
                        "alpha-boron-shaped: rh a=9.55 alpha=58, 48^3, 2x2x2 MP, 18 occ + 6 empty, bare Coulomb")
    if name == "C3":
        k, w = _gamma()
        return Workload("C3", SEED_BASE + 3, (64,) * 3, cubic(20.0), k, w, 12.0, 1, HSE_MU, 1.0, 64, np.ones(64),
                        "medium: sc a=20, 64^3, Gamma, 64 bands f=1, HSE mu=0.106")
    if name in ("C4a", "C4b"):
        k, w = _gamma() if name == "C4a" else _mp2()
        return Workload(name, SEED_BASE + 4, (96,) * 3, rhombohedral(19.2, 65.2), k, w, 15.0, 0, 0.0, 1.0, 160,
                        np.r_[np.ones(158), np.full(2, 0.5)],
                        "beta-boron-shaped: rh a=19.2 alpha=65.2, 96^3, %s, 158 occ + 2 half, bare Coulomb"
                        % ("Gamma" if name == "C4a" else "2x2x2 MP"))
    if name == "C5":
        k, w = _gamma()
        return Workload("C5", SEED_BASE + 5, (128,) * 3, cubic(30.0), k, w, 10.0, 1, HSE_MU, 1.0, 256, np.ones(256),
                        "stress: sc a=30, 128^3, Gamma, 256 bands f=1, HSE mu=0.106")
    raise KeyError(name)


def custom(name, seed, grid, lattice, kfrac, kweight, ecut, nbands, occ_per_k, kernel_kind=0, mu=0.0, scale=1.0):
    """A free-form workload with the same seeded-coefficient recipe (used for small parity/edge cases)."""
    return Workload(name, seed, tuple(int(g) for g in grid), np.asarray(lattice, dtype=np.float64),
                    np.asarray(kfrac, dtype=np.float64).reshape(-1, 3), np.asarray(kweight, dtype=np.float64), float(ecut),
                    int(kernel_kind), float(mu), float(scale), int(nbands), np.asarray(occ_per_k, dtype=np.float64))


ALL = ("C1", "C2", "C3", "C4a", "C4b", "C5")
