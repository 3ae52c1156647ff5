"""Seeded synthetic workloads (inputs only -- none of the method's arithmetic).

The paper validates on the muMAG standard problems #2/#4 and the spin-transfer
torque problem of its ref. [19] and times N x N (x N) grids
(PAPER.md:217-250).  None of those suites' data is used or reproduced here:
these generators make seeded synthetic states with the grid shapes, cell sizes,
material constants and magnetisation structure BASELINE.json `configs` names
(DESIGN.md section "Input recipe").  Both the oracle-side tests and the CUDA
side receive the SAME float32 arrays produced here.

This module imports neither the oracle nor the CUDA binding.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np


@dataclass
class Workload:
    name: str
    grid: tuple            # (Nx, Ny, Nz)
    cell: tuple            # metres
    pbc: tuple             # 0 open, p > 0 periodic with p images each side
    mat: dict              # Ms, Aex, alpha, Ku, anis_u, Bext, T, seed, j, P, xi
    init: str              # "random" | "tilted" | "xnoise" | "vortex" | "uniform"
    seed: int
    method: str = "rk4"
    dt: float = 1e-13
    tol: float = 1e-5
    steps: int = 100
    extra: dict = field(default_factory=dict)


def _gauss(seed: int, shape):
    rng = np.random.Generator(np.random.Philox(key=seed))
    return rng.standard_normal(size=shape)


def initial_m(wl: Workload) -> np.ndarray:
    """float32 unit vectors, shape (3, Nz, Ny, Nx), generated in fp64 and rounded once."""
    Nx, Ny, Nz = wl.grid
    shape = (3, Nz, Ny, Nx)
    g = _gauss(wl.seed, shape)
    if wl.init == "random":                 # uniform on the sphere
        m = g
    elif wl.init == "tilted":               # (1,1,0)/sqrt2 + 0.01 noise
        m = 0.01 * g
        m[0] += 1.0 / math.sqrt(2.0)
        m[1] += 1.0 / math.sqrt(2.0)
    elif wl.init == "xnoise":               # (1,0,0) + 0.1 noise
        m = 0.1 * g
        m[0] += 1.0
    elif wl.init == "uniform":
        m = np.zeros(shape)
        d = np.asarray(wl.extra.get("dir", (1.0, 0.0, 0.0)), dtype=np.float64)
        m += d[:, None, None, None]
    elif wl.init == "vortex":               # in-plane curl + out-of-plane core + 0.05 noise
        dx, dy, _ = wl.cell
        x = (np.arange(Nx) + 0.5 - Nx / 2.0) * dx
        y = (np.arange(Ny) + 0.5 - Ny / 2.0) * dy
        X, Y = np.meshgrid(x, y, indexing="xy")           # (Ny, Nx)
        rho = np.sqrt(X * X + Y * Y)
        rc = float(wl.extra.get("core_radius", 10e-9))
        m = 0.05 * g
        m[0] += (-Y / rho)[None]
        m[1] += (X / rho)[None]
        m[2] += np.exp(-rho * rho / (2.0 * rc * rc))[None]
    else:
        raise ValueError(wl.init)
    m = m / np.sqrt(np.sum(m * m, axis=0, keepdims=True))
    return np.ascontiguousarray(m.astype(np.float32))


def _mat(**kw):
    d = dict(Ms=8e5, Aex=1.3e-11, alpha=0.5, gamma0=2.211e5, Ku=0.0, anis_u=(0.0, 0.0, 1.0),
             Bext=(0.0, 0.0, 0.0), T=0.0, seed=0, j=(0.0, 0.0, 0.0), P=0.0, xi=0.0,
             stt_literal_eq7=False, K1=0.0, K2=0.0, anis_c1=(1.0, 0.0, 0.0), anis_c2=(0.0, 1.0, 0.0),
             exchange_in_kernel=False, geometry=False)
    d.update(kw)
    return d


def config(i: int) -> Workload:
    """BASELINE.json `configs[i]`; i = 5 is the headline 512x512x64 grid the metric is quoted on."""
    if i == 0:
        return Workload("cfg0_32x32x1", (32, 32, 1), (4e-9, 4e-9, 4e-9), (0, 0, 0),
                        _mat(alpha=0.5), "random", 0, "rk4", 1e-13, steps=100)
    if i == 1:
        a = math.radians(170.0)
        return Workload("cfg1_film_256x64x1", (256, 64, 1), (3.90625e-9, 3.90625e-9, 4e-9),
                        (0, 0, 0),
                        _mat(alpha=0.02, Bext=(25e-3 * math.cos(a), 25e-3 * math.sin(a), 0.0)),
                        "tilted", 1, "rkdp", 1e-13, tol=1e-5, steps=100,
                        extra={"t_end": 1e-9})
    if i == 2:
        return Workload("cfg2_cube_128", (128, 128, 128), (5e-9, 5e-9, 5e-9), (0, 0, 0),
                        _mat(Ms=1.1e6, Aex=2e-11, Ku=5e5, anis_u=(0.0, 0.0, 1.0), alpha=1.0),
                        "random", 2, "rkdp", 1e-14, steps=2000)
    if i == 3:
        return Workload("cfg3_pbc_1024x1024x1", (1024, 1024, 1), (4e-9, 4e-9, 2e-9), (10, 10, 0),
                        _mat(alpha=0.1, T=300.0, seed=3, j=(1e12, 0.0, 0.0), P=0.5, xi=0.04),
                        "xnoise", 3, "rk4", 5e-14, steps=10000)
    if i == 4:
        return Workload("cfg4_768x384x64", (768, 384, 64), (3e-9, 3e-9, 3e-9), (0, 0, 0),
                        _mat(alpha=0.02, Ku=1e4, anis_u=(1.0, 0.0, 0.0), Bext=(0.0, 10e-3, 0.0)),
                        "vortex", 4, "rkdp", 1e-14, steps=1000, extra={"core_radius": 10e-9})
    if i == 5:
        return Workload("headline_512x512x64", (512, 512, 64), (3e-9, 3e-9, 3e-9), (0, 0, 0),
                        _mat(alpha=0.02, Ku=1e4, anis_u=(1.0, 0.0, 0.0), Bext=(0.0, 10e-3, 0.0)),
                        "vortex", 5, "rk4", 5e-14, steps=20, extra={"core_radius": 10e-9})
    raise IndexError(i)


def scaled(wl: Workload, grid, name=None, pbc=None) -> Workload:
    """Same material, cell size and initial-state recipe on another grid (parity-test sizes)."""
    import copy
    w = copy.deepcopy(wl)
    w.grid = tuple(int(v) for v in grid)
    if pbc is not None:
        w.pbc = tuple(pbc)
    w.name = name or f"{wl.name}@{'x'.join(map(str, grid))}"
    return w
