"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module serves BOTH the oracle-side tests and the CUDA-side tests/bench.  It holds none of the
method's arithmetic: only numpy random draws and the cosine seed patterns the configs name.  The
paper uses no public dataset: its workloads are parameter sets, so these
seeded fields *are* the workload.
"""
from dataclasses import dataclass, field
from itertools import product

import numpy as np

BASE_SEED = 12045434 * 10


@dataclass
class Config:
    name: str
    model: str                      # "external" | "edwards" | "diblock"
    grid: tuple
    cell: tuple
    Ns: int
    fA: float = 0.5
    chiN: float = 10.0
    B: float = 1.0
    C: float = 1.0
    dt: float = 0.0                 # CL time step (configs 4, 5)
    dt_scft: tuple = (5.0, 5.0)     # SCFT pseudo-time steps (reading A-12)
    iters: int = 0
    f0: np.ndarray = field(default=None, repr=False)
    f1: np.ndarray = field(default=None, repr=False)


def _coords(grid, cell):
    ax = [np.arange(n, dtype=np.float64) * (L / n) for n, L in zip(grid, cell)]
    return np.meshgrid(*ax, indexing="ij")


def _rng(config_no, stream=0):
    return np.random.default_rng([BASE_SEED + config_no, stream])


def config1(grid=(16, 16, 16), cell=(4.0, 4.0, 4.0), Ns=64, seed_offset=0):
    """Homopolymer in an external complex field: w = 0.5 + sum over |n|<=2 of seeded amplitudes."""
    rng = _rng(1 + 100 * seed_offset)
    X = _coords(grid, cell)
    reps = [n for n in product(range(-2, 3), repeat=3)
            if 0 < n[0] ** 2 + n[1] ** 2 + n[2] ** 2 <= 4 and n > (0, 0, 0)]     # half-space representatives
    reps.sort()
    wr = np.full(grid, 0.5)
    wi = np.zeros(grid)
    for n in reps:
        a, b, c, d = rng.normal(0.0, 0.1, 4)
        th = 2.0 * np.pi * sum(n[k] * X[k] / cell[k] for k in range(3))
        wr += 2.0 * (a * np.cos(th) - b * np.sin(th))
        wi += 2.0 * (c * np.cos(th) - d * np.sin(th))
    return Config("cfg1_homopolymer_16", "external", tuple(grid), tuple(cell), Ns, f0=(wr + 1j * wi))


def config2(grid=(32, 32, 32), cell=(4.0, 4.0, 4.0), Ns=100, iters=200):
    """Diblock SCFT, hexagonal-cylinder cosine seed along [111] plus N(0, 0.05^2) noise."""
    rng = _rng(2)
    X = _coords(grid, cell)
    wm = np.zeros(grid)
    for n in ((1, -1, 0), (0, 1, -1), (-1, 0, 1)):
        wm += 1.5 * np.cos(2.0 * np.pi * sum(n[k] * X[k] / cell[k] for k in range(3)))
    wm += rng.normal(0.0, 0.05, grid)
    return Config("cfg2_diblock_scft_32", "diblock", tuple(grid), tuple(cell), Ns, fA=0.3, chiN=20.0, C=1.0,
                  iters=iters, f0=np.zeros(grid, np.complex128), f1=wm.astype(np.complex128))


def config3(grid=(64, 64, 64), cell=(8.0, 8.0, 8.0), Ns=200, iters=500):
    """Diblock SCFT, two lamellar periods along x plus noise."""
    rng = _rng(3)
    X = _coords(grid, cell)
    wm = 1.5 * np.cos(2.0 * np.pi * 2.0 * X[0] / cell[0]) + rng.normal(0.0, 0.05, grid)
    return Config("cfg3_diblock_scft_64", "diblock", tuple(grid), tuple(cell), Ns, fA=0.35, chiN=18.0, C=1.0,
                  iters=iters, f0=np.zeros(grid, np.complex128), f1=wm.astype(np.complex128))


def config4(grid=(64, 64, 64), cell=(8.0, 8.0, 8.0), Ns=100, iters=1000):
    """Edwards solution, complex Langevin: Omega_0 = -iC/B + real N(0, 0.05^2)."""
    rng = _rng(4)
    B, Cc = 1.0, 10.0
    om = rng.normal(0.0, 0.05, grid) - 1j * (Cc / B)
    return Config("cfg4_edwards_cl_64", "edwards", tuple(grid), tuple(cell), Ns, B=B, C=Cc, dt=0.01, iters=iters, f0=om)


def config5(n=256, Ns=100, iters=10):
    """Fluctuating diblock melt, complex Langevin, n^3 grid (n = 256; n = 128 is the scaling point)."""
    rng = _rng(5, n)
    grid, cell = (n, n, n), (16.0, 16.0, 16.0)
    x = (np.arange(n, dtype=np.float64) * (cell[0] / n))[:, None, None]
    wm = rng.normal(0.0, 0.05, grid)
    wm += 1.5 * np.cos(2.0 * np.pi * 4.0 * x / cell[0])
    return Config(f"cfg5_diblock_cl_{n}", "diblock", grid, cell, Ns, fA=0.5, chiN=15.0, C=50.0, dt=0.005,
                  iters=iters, f0=np.zeros(grid, np.complex128), f1=wm.astype(np.complex128))


def small_diblock(grid=(8, 16, 32), cell=(3.0, 4.0, 5.0), Ns=20, fA=0.4, chiN=12.0, C=5.0, seed=7, complex_fields=True):
    """A ragged (anisotropic, non-cubic) diblock case for parity tests; complex fields as in CL."""
    rng = _rng(90 + seed)
    X = _coords(grid, cell)
    wm = 0.8 * np.cos(2.0 * np.pi * X[2] / cell[2]) + rng.normal(0.0, 0.2, grid)
    wp = rng.normal(0.0, 0.2, grid)
    if complex_fields:
        wm = wm + 1j * rng.normal(0.0, 0.1, grid)
        wp = wp + 1j * rng.normal(0.0, 0.1, grid)
    return Config("small_diblock", "diblock", tuple(grid), tuple(cell), Ns, fA=fA, chiN=chiN, C=C, dt=0.01,
                  f0=np.asarray(wp, np.complex128), f1=np.asarray(wm, np.complex128))


def random_complex_field(grid, seed, scale=0.3, mean=0.0):
    rng = _rng(50, seed)
    return mean + scale * (rng.normal(size=grid) + 1j * rng.normal(size=grid))


def developed(cfg, seed=0):
    """Seeded fields with the amplitude and roughness of a run that has left its initial condition (stronger
    segregation, a non-zero pressure-like field, complex parts as in CL) — used to compare one solve at a
    'late-time' state without feeding anything produced by the CUDA path to the oracle."""
    rng = _rng(70, seed)
    X = _coords(cfg.grid, cfg.cell)
    smooth = sum(np.cos(2.0 * np.pi * (k + 1) * X[k] / cfg.cell[k]) for k in range(3))
    if cfg.model == "diblock":
        f1 = 2.0 * cfg.f1.real + rng.normal(0.0, 0.1, cfg.grid) + 1j * rng.normal(0.0, 0.05, cfg.grid)
        f0 = 0.4 * smooth + rng.normal(0.0, 0.1, cfg.grid) + 1j * rng.normal(0.0, 0.05, cfg.grid)
        return np.asarray(f0, np.complex128), np.asarray(f1, np.complex128)
    f0 = cfg.f0 + 0.2 * smooth + rng.normal(0.0, 0.3, cfg.grid) + 1j * rng.normal(0.0, 0.2, cfg.grid)
    return np.asarray(f0, np.complex128), None
