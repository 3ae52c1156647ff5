"""oracle/mm_oracle.py -- TEST INFRASTRUCTURE, not product code.

A plain, slow, fp64 CPU statement of what the hot path computes: one effective
field evaluation plus the Landau-Lifshitz torque per Runge-Kutta stage of the
MuMax method (arXiv 1102.3069).  Every function cites the passage of
/root/reference/PAPER.md it restates ("PAPER.md:<line>", section / equation)
and, where the paper is silent, the reading listed in DESIGN.md ("reading A<n>").

Rules this file keeps:
  * SI units, numpy float64 throughout (the demag tensor itself is evaluated in
    __float128 by oracle/demag_tensor.c and handed over as float64).
  * The result of the FFT convolution has a plain definition -- the direct sum
    over all cell pairs -- so `demag_field_direct` IS that definition; the FFT
    route `demag_field_fft` (numpy's FFT as a library step) is a second,
    faster statement of the same sum, pinned to the first.
  * Integrators follow the textbook algorithm stage by stage.
  * No blocking, fusion or reordering beyond that.
  * Shares no code with paper_1102_3069_b200/ and never imports it.  Only
    tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
    reference legs may import this module.

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): tensor closed forms and
symmetries, direct sum == FFT route, sample demagnetising factors, exchange
eigenvalue of a periodic helix, anisotropy special cases, macrospin closed form
(Larmor precession + damping), RK order of convergence, Runge-Kutta order
conditions in exact rationals, Philox known answers, Zhang-Li helix translation.
Parity unpinned (conventions shared with the CUDA path): the
step-controller constants (A10), the periodic image count (A8), one thermal draw
per step (A6), the open-face gradient rule of the Zhang-Li term (A7).

Array layout everywhere: m[c, z, y, x], c = 0,1,2 for x,y,z; shape (3, Nz, Ny, Nx).
`grid` = (Nx, Ny, Nz), `cell` = (dx, dy, dz) in metres, `pbc` = (px, py, pz) with
0 = open and p > 0 = periodic with images -p..p (reading A8).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field
from fractions import Fraction

import numpy as np

MU0 = 4e-7 * np.pi            # T m / A
KB = 1.380649e-23             # J / K
MUB = 9.2740100783e-24        # J / T
QE = 1.602176634e-19          # C
GAMMA0_DEFAULT = 2.211e5      # m / (A s)   (reading A2)

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None


def build_tensor_lib(force: bool = False) -> str:
    """Compile oracle/demag_tensor.c (gcc, libquadmath, OpenMP) next to its source."""
    so = os.path.join(_HERE, "liboracle_tensor.so")
    src = os.path.join(_HERE, "demag_tensor.c")
    if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", so, src,
                               "-lquadmath", "-lm"])
    return so


def _lib():
    global _LIB
    if _LIB is None:
        _LIB = ctypes.CDLL(build_tensor_lib())
    return _LIB


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


# --------------------------------------------------------------------------
# Material / run parameters
# --------------------------------------------------------------------------
@dataclass
class Material:
    """Material and drive parameters in SI units."""
    Ms: float                       # A/m
    Aex: float = 0.0                # J/m        Eq. (3)
    alpha: float = 0.0              # damping    Eq. (1)
    gamma0: float = GAMMA0_DEFAULT  # m/(A s)    reading A2
    Ku: float = 0.0                 # J/m^3      Eq. (4)
    anis_u: tuple = (0.0, 0.0, 1.0)
    Bext: tuple = (0.0, 0.0, 0.0)   # tesla; H = B / mu0
    T: float = 0.0                  # kelvin     Eq. (6)
    seed: int = 0                   # Philox key
    j: tuple = (0.0, 0.0, 0.0)      # A/m^2      Eq. (7)
    P: float = 0.0                  # polarisation, Eq. (8)
    xi: float = 0.0                 # non-adiabaticity, Eq. (7)
    stt_literal_eq7: bool = False   # reading A7
    K1: float = 0.0                 # J/m^3      Eq. (5), cubic anisotropy
    K2: float = 0.0                 # J/m^3      Eq. (5)
    anis_c1: tuple = (1.0, 0.0, 0.0)   # first two cubic axes; the third is c1 x c2 (reading A14)
    anis_c2: tuple = (0.0, 1.0, 0.0)
    exchange_in_kernel: bool = False   # exchange added to the convolution kernel (reading A3')
    geometry: bool = False          # cells with m = 0 are empty (staircase shapes, reading A15)


# --------------------------------------------------------------------------
# Demagnetisation tensor and magnetostatic field  (Eq. (2))
# --------------------------------------------------------------------------
def tensor_at(offsets, cell, nimg=(0, 0, 0), period=(0, 0, 0)) -> np.ndarray:
    """N(xx,yy,zz,xy,xz,yz) at integer cell offsets, float128 inside; shape (n, 6)."""
    off = np.ascontiguousarray(np.asarray(offsets, dtype=np.int64).reshape(-1, 3))
    out = np.zeros((off.shape[0], 6), dtype=np.float64)
    c = np.asarray(cell, dtype=np.float64)
    ni = np.asarray(nimg, dtype=np.int32)
    pe = np.asarray(period, dtype=np.int64)
    _lib().oracle_tensor_at(ctypes.c_long(off.shape[0]), _ptr(off), _ptr(c), _ptr(ni), _ptr(pe),
                            _ptr(out))
    return out


def tensor_octant(n, cell) -> np.ndarray:
    """N on the lattice 0<=i<n[0], 0<=j<n[1], 0<=k<n[2]; shape (6, n2, n1, n0)."""
    out = np.zeros((6, n[2], n[1], n[0]), dtype=np.float64)
    c = np.asarray(cell, dtype=np.float64)
    _lib().oracle_tensor_octant(ctypes.c_long(n[0]), ctypes.c_long(n[1]), ctypes.c_long(n[2]),
                                _ptr(c), _ptr(out))
    return out


def padded_size(grid, pbc):
    """Reading A9: P_a = N_a if periodic, 2 N_a if open and N_a > 1, else 1."""
    return tuple(int(n) if p > 0 else (2 * int(n) if n > 1 else 1) for n, p in zip(grid, pbc))


# parity of each component under reflection of axis a: +1 even, -1 odd
_PARITY = np.array([[1, 1, 1],    # xx
                    [1, 1, 1],    # yy
                    [1, 1, 1],    # zz
                    [-1, -1, 1],  # xy
                    [-1, 1, -1],  # xz
                    [1, -1, -1]])  # yz


def _signed_offsets(n, P, periodic):
    """Offsets d held by slots 0..P-1 of a circular kernel axis, and a validity mask.
    Open axis: d in [-(n-1), n-1] at slot d mod P; slot n (only if P = 2n) is never
    touched by the linear convolution and holds 0 (reading A9).  Periodic axis:
    d folded to (-n/2, n/2] (reading A8)."""
    d = np.arange(P)
    if periodic:
        d = np.where(d > n // 2, d - P, d)
        return d, np.ones(P, dtype=bool)
    if P == 1:
        return d, np.ones(1, dtype=bool)
    valid = d != n
    d = np.where(d > n, d - P, d)
    return d, valid


def demag_kernel(grid, cell, pbc=(0, 0, 0)) -> np.ndarray:
    """The convolution kernel N on the padded circular lattice, shape (6, Pz, Py, Px).

    PAPER.md:73: periodic boundary conditions enter by summing periodic images
    into the kernel; open axes are zero padded.  Reading A8: images
    -p..p around the offset folded to (-N/2, N/2], then symmetrise per axis on the
    circular lattice so that the transform is exactly real."""
    Nx, Ny, Nz = (int(v) for v in grid)
    P = padded_size(grid, pbc)
    per = [p > 0 for p in pbc]
    dx, vx = _signed_offsets(Nx, P[0], per[0])
    dy, vy = _signed_offsets(Ny, P[1], per[1])
    dz, vz = _signed_offsets(Nz, P[2], per[2])
    K = np.zeros((6, P[2], P[1], P[0]))
    if not any(per):
        # all offsets are +-(lattice point of the non-negative octant): use parity
        octv = tensor_octant((Nx, Ny, Nz), cell)
        ax, ay, az = np.abs(dx), np.abs(dy), np.abs(dz)
        for q in range(6):
            s = (np.where(dz < 0, _PARITY[q, 2], 1)[:, None, None]
                 * np.where(dy < 0, _PARITY[q, 1], 1)[None, :, None]
                 * np.where(dx < 0, _PARITY[q, 0], 1)[None, None, :])
            K[q] = octv[q][np.ix_(np.minimum(az, Nz - 1), np.minimum(ay, Ny - 1),
                                  np.minimum(ax, Nx - 1))] * s
    else:
        Z, Y, X = np.meshgrid(dz, dy, dx, indexing="ij")
        off = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)
        nimg = [int(p) if p > 0 else 0 for p in pbc]
        K = tensor_at(off, cell, nimg, (Nx, Ny, Nz)).T.reshape(6, *Z.shape).copy()
        # symmetrise on the circular lattice, axis by axis: K <- (K + sigma_a R_a K)/2 with R_a the
        # circular reflection slot -> (-slot) mod P_a.  With the symmetric image set this is the
        # identity except at slot N_a/2 of an even periodic axis, where components odd in a become 0.
        for q in range(6):
            for arr_ax, a in ((3, 0), (2, 1), (1, 2)):
                if per[a]:
                    refl = np.roll(np.flip(K[q], axis=arr_ax - 1), 1, axis=arr_ax - 1)
                    K[q] = 0.5 * (K[q] + _PARITY[q, a] * refl)
    mask = vz[:, None, None] & vy[None, :, None] & vx[None, None, :]
    K *= mask[None]
    return K


def _sym3(K6):
    """(6, ...) -> nested 3x3 list, order xx,yy,zz,xy,xz,yz."""
    xx, yy, zz, xy, xz, yz = K6
    return [[xx, xy, xz], [xy, yy, yz], [xz, yz, zz]]


def demag_field_direct(m, Ms, grid, cell, pbc=(0, 0, 0)) -> np.ndarray:
    """Path O1: H_ms(i) = -Ms sum_j N(r_i - r_j) . m_j, the plain O(N^2) pair sum
    (discrete Eq. (2)).  Organised offset by offset: for every offset d
    all pairs (i, j = i - d) are accumulated at once.  Tiny grids only."""
    Nx, Ny, Nz = (int(v) for v in grid)
    per = [p > 0 for p in pbc]
    nimg = [int(p) if p > 0 else 0 for p in pbc]
    H = np.zeros_like(m, dtype=np.float64)

    def rng(n, periodic):
        return range(-(n // 2) + (1 if n % 2 == 0 else 0), n // 2 + 1) if periodic \
            else range(-(n - 1), n)

    offs = [(ox, oy, oz) for oz in rng(Nz, per[2]) for oy in rng(Ny, per[1])
            for ox in rng(Nx, per[0])]
    off = np.array(offs, dtype=np.int64)
    self_n = (Nx, Ny, Nz)
    Nd = tensor_at(off, cell, nimg, (Nx, Ny, Nz))
    # reading A8: at offset N_a/2 of an even periodic axis (+N/2 and -N/2 are the same pair of
    # cells) the components odd in a vanish
    for a in range(3):
        if per[a] and self_n[a] % 2 == 0:
            half = off[:, a] == self_n[a] // 2
            Nd[np.ix_(half, _PARITY[:, a] < 0)] = 0.0
    for (ox, oy, oz), n6 in zip(offs, Nd):
        N = _sym3(n6)
        # source field shifted so that src[i] = m[i - d]
        src = m
        sl_dst = [slice(None)] * 3
        sl_src = [slice(None)] * 3
        for ax, (o, n, p) in enumerate(((oz, Nz, per[2]), (oy, Ny, per[1]), (ox, Nx, per[0]))):
            if p:
                src = np.roll(src, o, axis=ax + 1)
            else:
                lo, hi = max(0, o), min(n, n + o)
                sl_dst[ax] = slice(lo, hi)
                sl_src[ax] = slice(lo - o, hi - o)
        d = (slice(None),) + tuple(sl_dst)
        s = (slice(None),) + tuple(sl_src)
        ms = src[s]
        for a in range(3):
            H[d][a] -= Ms * (N[a][0] * ms[0] + N[a][1] * ms[1] + N[a][2] * ms[2])
    return H


def demag_kernel_fft(K) -> np.ndarray:
    """FFT of the placed kernel; real by symmetry, imaginary part is
    returned too so that a test can check it vanishes."""
    return np.fft.rfftn(K, axes=(1, 2, 3))


def demag_field_fft(m, Ms, grid, pbc, Khat) -> np.ndarray:
    """Path O2: zero pad m in the open directions, transform,
    multiply point by point with the transformed kernel, transform back, crop."""
    Nx, Ny, Nz = (int(v) for v in grid)
    P = padded_size(grid, pbc)
    Mh = np.fft.rfftn(np.asarray(m, dtype=np.float64), s=(P[2], P[1], P[0]), axes=(1, 2, 3))
    Kh = _sym3(Khat.real)
    H = np.empty((3, Nz, Ny, Nx))
    for a in range(3):
        Hh = -(Kh[a][0] * Mh[0] + Kh[a][1] * Mh[1] + Kh[a][2] * Mh[2])
        H[a] = np.fft.irfftn(Hh, s=(P[2], P[1], P[0]), axes=(0, 1, 2))[:Nz, :Ny, :Nx]
    return Ms * H


# --------------------------------------------------------------------------
# Local field terms
# --------------------------------------------------------------------------
def exchange_field(m, mat: Material, grid, cell, pbc=(0, 0, 0)) -> np.ndarray:
    """Eq. (3): H_ex = 2A/(mu0 Ms) lap(m), 6-neighbour scheme.  A
    missing neighbour at an open face contributes zero (reading A3); periodic axes
    wrap; an axis with one cell contributes nothing (2D -> 4 neighbours)."""
    H = np.zeros_like(m, dtype=np.float64)
    if mat.Aex == 0.0:
        return H
    pref = 2.0 * mat.Aex / (MU0 * mat.Ms)
    for ax, (n, d, p) in enumerate(((grid[2], cell[2], pbc[2]), (grid[1], cell[1], pbc[1]),
                                    (grid[0], cell[0], pbc[0]))):
        if n == 1:
            continue
        a = ax + 1
        if p > 0:
            H += pref * (np.roll(m, 1, axis=a) + np.roll(m, -1, axis=a) - 2.0 * m) / d ** 2
        else:
            up = [slice(None)] * 4
            dn = [slice(None)] * 4
            up[a] = slice(1, None)
            dn[a] = slice(None, -1)
            diff = (m[tuple(up)] - m[tuple(dn)]) / d ** 2       # m_{i+1} - m_i
            H[tuple(dn)] += pref * diff                          # neighbour i+1 seen from i
            H[tuple(up)] -= pref * diff                          # neighbour i-1 seen from i
    return H


def _shifted(m, a, sgn, n, periodic):
    """m_(i + sgn e_a) with the cell itself where that neighbour does not exist (open face)."""
    if periodic:
        return np.roll(m, -sgn, axis=a)
    idx = np.arange(n)
    return np.take(m, np.clip(idx + sgn, 0, n - 1), axis=a)


def exchange_field_geometry(m, mat: Material, grid, cell, pbc=(0, 0, 0)) -> np.ndarray:
    """Eq. (3) on a staircase shape (reading A15): cells with m = 0 are empty.  An empty
    neighbour counts as a missing one (free boundary, as reading A3: it contributes zero), and an empty
    cell has no exchange field."""
    H = np.zeros_like(m, dtype=np.float64)
    if mat.Aex == 0.0:
        return H
    pref = 2.0 * mat.Aex / (MU0 * mat.Ms)
    full = (np.sum(m * m, axis=0, keepdims=True) > 0.0)
    for a, comp in ((3, 0), (2, 1), (1, 2)):
        n, d = grid[comp], cell[comp]
        if n == 1:
            continue
        for sgn in (1, -1):
            nb = _shifted(m, a, sgn, n, pbc[comp] > 0)
            nb_full = _shifted(full, a, sgn, n, pbc[comp] > 0)
            H += pref * np.where(nb_full & full, nb - m, 0.0) / d ** 2
    return H


def exchange_field_in_kernel(m, mat: Material, grid, cell, pbc=(0, 0, 0)) -> np.ndarray:
    """The paper's own variant (reading A3'): the exchange stencil is added to the
    magnetostatic kernel, so at an open face the zero padding of the convolution makes a missing
    neighbour count as m = 0:  H_ex(i) = 2A/(mu0 Ms) sum_a [ m_(i+a) + m_(i-a) - 2 m_i ] / d_a^2 with
    m = 0 outside the grid.  Written here as exactly that sum (no convolution)."""
    H = np.zeros_like(m, dtype=np.float64)
    if mat.Aex == 0.0:
        return H
    pref = 2.0 * mat.Aex / (MU0 * mat.Ms)
    for ax, (n, d, p) in enumerate(((grid[2], cell[2], pbc[2]), (grid[1], cell[1], pbc[1]),
                                    (grid[0], cell[0], pbc[0]))):
        if n == 1:
            continue
        a = ax + 1
        if p > 0:
            H += pref * (np.roll(m, 1, axis=a) + np.roll(m, -1, axis=a) - 2.0 * m) / d ** 2
        else:
            mp = np.zeros_like(m, dtype=np.float64)      # m_(i+a), zero beyond the last cell
            mm = np.zeros_like(m, dtype=np.float64)      # m_(i-a), zero before the first cell
            up = [slice(None)] * 4
            dn = [slice(None)] * 4
            up[a] = slice(1, None)
            dn[a] = slice(None, -1)
            mp[tuple(dn)] = m[tuple(up)]
            mm[tuple(up)] = m[tuple(dn)]
            H += pref * (mp + mm - 2.0 * m) / d ** 2
    return H


def anisotropy_field(m, mat: Material) -> np.ndarray:
    """From the energy density Eq. (4): E = Ku sin^2(theta) = Ku (1 - (m.u)^2)
    => H = -(1/(mu0 Ms)) dE/dm = 2 Ku/(mu0 Ms) (m.u) u   (reading A5)."""
    if mat.Ku == 0.0:
        return np.zeros_like(m, dtype=np.float64)
    u = np.asarray(mat.anis_u, dtype=np.float64)
    u = u / np.linalg.norm(u)
    mu = np.tensordot(u, m, axes=(0, 0))
    return (2.0 * mat.Ku / (MU0 * mat.Ms)) * u[:, None, None, None] * mu[None]


def cubic_axes(mat: Material):
    """Reading A14 (the paper names "the cubic easy magnetization axes" without saying how they are
    given): c1 normalised, c2 made orthogonal to c1 and normalised, c3 = c1 x c2."""
    c1 = np.asarray(mat.anis_c1, dtype=np.float64)
    c1 = c1 / np.linalg.norm(c1)
    c2 = np.asarray(mat.anis_c2, dtype=np.float64)
    c2 = c2 - np.dot(c2, c1) * c1
    c2 = c2 / np.linalg.norm(c2)
    return c1, c2, np.cross(c1, c2)


def cubic_anisotropy_energy_density(m, mat: Material) -> np.ndarray:
    """Eq. (5): K1 (a1^2 a2^2 + a2^2 a3^2 + a1^2 a3^2) + K2 a1^2 a2^2 a3^2,
    a_i the direction cosines of m on the cubic axes.  J/m^3 per cell."""
    a = [np.tensordot(c, m, axes=(0, 0)) for c in cubic_axes(mat)]
    return mat.K1 * (a[0] ** 2 * a[1] ** 2 + a[1] ** 2 * a[2] ** 2 + a[0] ** 2 * a[2] ** 2) \
        + mat.K2 * a[0] ** 2 * a[1] ** 2 * a[2] ** 2


def cubic_anisotropy_field(m, mat: Material) -> np.ndarray:
    """H = -(1/(mu0 Ms)) dE/dm of Eq. (5): with dE/da1 = 2 K1 a1 (a2^2 + a3^2) + 2 K2 a1 a2^2 a3^2
    (and cyclic), H = -(1/(mu0 Ms)) sum_i (dE/da_i) c_i."""
    if mat.K1 == 0.0 and mat.K2 == 0.0:
        return np.zeros_like(m, dtype=np.float64)
    c = cubic_axes(mat)
    a = [np.tensordot(ci, m, axes=(0, 0)) for ci in c]
    H = np.zeros_like(m, dtype=np.float64)
    for i in range(3):
        j, k = (i + 1) % 3, (i + 2) % 3
        dE = 2.0 * mat.K1 * a[i] * (a[j] ** 2 + a[k] ** 2) + 2.0 * mat.K2 * a[i] * a[j] ** 2 * a[k] ** 2
        H -= c[i][:, None, None, None] * dE[None] / (MU0 * mat.Ms)
    return H


def zeeman_field(m, mat: Material) -> np.ndarray:
    """Applied field: H_ext = B_ext / mu0, uniform."""
    B = np.asarray(mat.Bext, dtype=np.float64)
    return np.broadcast_to((B / MU0)[:, None, None, None], m.shape).copy()


# ---- Philox4x32-10 (counter-based generator; the CUDA path implements the same) ----
_PH_M0 = np.uint64(0xD2511F53)
_PH_M1 = np.uint64(0xCD9E8D57)
_PH_W0 = 0x9E3779B9
_PH_W1 = 0xBB67AE85
_M32 = np.uint64(0xFFFFFFFF)


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Philox4x32 with 10 rounds.  Counter words c0..c3 (arrays or scalars, any
    integer type, taken mod 2^32), key words k0, k1 (ints).  Returns four uint32
    arrays.  Round: (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0));
    then the key is bumped by (W0, W1)."""
    c0, c1, c2, c3 = (np.asarray(c, dtype=np.uint64) & _M32 for c in (c0, c1, c2, c3))
    c0, c1, c2, c3 = np.broadcast_arrays(c0, c1, c2, c3)
    k0 = int(k0) & 0xFFFFFFFF
    k1 = int(k1) & 0xFFFFFFFF
    for _ in range(10):
        p0 = _PH_M0 * c0
        p1 = _PH_M1 * c2
        n0 = (p1 >> np.uint64(32)) ^ c1 ^ np.uint64(k0)
        n1 = p1 & _M32
        n2 = (p0 >> np.uint64(32)) ^ c3 ^ np.uint64(k1)
        n3 = p0 & _M32
        c0, c1, c2, c3 = n0, n1, n2, n3
        k0 = (k0 + _PH_W0) & 0xFFFFFFFF
        k1 = (k1 + _PH_W1) & 0xFFFFFFFF
    return tuple(c.astype(np.uint32) for c in (c0, c1, c2, c3))


def thermal_eta(grid, seed: int, step: int) -> np.ndarray:
    """eta(r, step): three N(0,1) numbers per cell, reading A6:
    key = (seed lo, seed hi), counter = (cell lo, cell hi, step lo, step hi), cell =
    (z*Ny + y)*Nx + x;  u1 = (x0+1) 2^-32, th1 = 2 pi x1 2^-32, u2 = (x2+1) 2^-32,
    th2 = 2 pi x3 2^-32;  eta = (r1 cos th1, r1 sin th1, r2 cos th2), r = sqrt(-2 ln u)."""
    Nx, Ny, Nz = (int(v) for v in grid)
    cellidx = np.arange(Nx * Ny * Nz, dtype=np.uint64)
    x0, x1, x2, x3 = philox4x32_10(cellidx & _M32, cellidx >> np.uint64(32),
                                   step & 0xFFFFFFFF, (step >> 32) & 0xFFFFFFFF,
                                   seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF)
    two32 = 4294967296.0
    u1 = (x0.astype(np.float64) + 1.0) / two32
    u2 = (x2.astype(np.float64) + 1.0) / two32
    th1 = 2.0 * np.pi * x1.astype(np.float64) / two32
    th2 = 2.0 * np.pi * x3.astype(np.float64) / two32
    r1 = np.sqrt(-2.0 * np.log(u1))
    r2 = np.sqrt(-2.0 * np.log(u2))
    eta = np.stack([r1 * np.cos(th1), r1 * np.sin(th1), r2 * np.cos(th2)])
    return eta.reshape(3, Nz, Ny, Nx)


def thermal_sigma(mat: Material, cell, dt: float) -> float:
    """Amplitude of Eq. (6): sqrt(2 alpha kB T / (gamma mu0 Ms V dt)),
    gamma = gamma0 (reading A6)."""
    V = cell[0] * cell[1] * cell[2]
    return float(np.sqrt(2.0 * mat.alpha * KB * mat.T / (mat.gamma0 * MU0 * mat.Ms * V * dt)))


def thermal_field(mat: Material, grid, cell, step: int, dt: float) -> np.ndarray:
    """Eq. (6)."""
    if mat.T == 0.0:
        return np.zeros((3, grid[2], grid[1], grid[0]))
    return thermal_sigma(mat, cell, dt) * thermal_eta(grid, mat.seed, step)


# --------------------------------------------------------------------------
# Effective field, torque
# --------------------------------------------------------------------------
class Problem:
    """Grid + material + the transformed demag kernel (set up once)."""

    def __init__(self, grid, cell, pbc, mat: Material, demag: str = "fft"):
        self.grid = tuple(int(v) for v in grid)
        self.cell = tuple(float(v) for v in cell)
        self.pbc = tuple(int(v) for v in pbc)
        self.mat = mat
        self.demag = demag            # "fft" (O2), "direct" (O1) or "none"
        self.Khat = None
        if demag == "fft":
            Kh = demag_kernel_fft(demag_kernel(self.grid, self.cell, self.pbc))
            self.Khat = Kh

    def demag_field(self, m):
        if self.demag == "none":
            return np.zeros_like(m, dtype=np.float64)
        if self.demag == "direct":
            return demag_field_direct(m, self.mat.Ms, self.grid, self.cell, self.pbc)
        return demag_field_fft(m, self.mat.Ms, self.grid, self.pbc, self.Khat)

    def heff(self, m, step: int = 0, dt_thermal: float = 0.0):
        """H_eff = H_ms + H_ex + H_an + H_ext + H_th, in A/m."""
        m = np.asarray(m, dtype=np.float64)
        H = self.demag_field(m)
        if self.mat.geometry:
            H = H + exchange_field_geometry(m, self.mat, self.grid, self.cell, self.pbc)
        elif self.mat.exchange_in_kernel:
            H = H + exchange_field_in_kernel(m, self.mat, self.grid, self.cell, self.pbc)
        else:
            H = H + exchange_field(m, self.mat, self.grid, self.cell, self.pbc)
        H = H + anisotropy_field(m, self.mat)
        H = H + cubic_anisotropy_field(m, self.mat)
        H = H + zeeman_field(m, self.mat)
        if self.mat.T != 0.0:
            H = H + thermal_field(self.mat, self.grid, self.cell, step, dt_thermal)
        return H

    def torque(self, m, step: int = 0, dt_thermal: float = 0.0):
        """dm/dt in 1/s: Eq. (1) written for m = M/Ms, plus the
        Zhang-Li terms of Eq. (7)-(8) when j != 0."""
        m = np.asarray(m, dtype=np.float64)
        return ll_torque(m, self.heff(m, step, dt_thermal), self.mat, self.grid, self.cell,
                         self.pbc)


def j_dot_grad_m(m, mat: Material, grid, cell, pbc) -> np.ndarray:
    """(j . nabla) m by central differences (m_{i+1} - m_{i-1})/(2 d) per axis with
    j_a != 0; at an open face the missing neighbour is replaced by the cell itself
    (reading A7); periodic axes wrap; one-cell axes contribute nothing."""
    out = np.zeros_like(m, dtype=np.float64)
    for a_m, comp in ((3, 0), (2, 1), (1, 2)):      # array axis, vector component
        ja = mat.j[comp]
        n = grid[comp]
        if ja == 0.0 or n == 1:
            continue
        if pbc[comp] > 0:
            up = np.roll(m, -1, axis=a_m)
            dn = np.roll(m, 1, axis=a_m)
        else:
            idx = np.arange(n)
            up = np.take(m, np.minimum(idx + 1, n - 1), axis=a_m)
            dn = np.take(m, np.maximum(idx - 1, 0), axis=a_m)
        if mat.geometry:          # reading A15: an empty neighbour is replaced by the cell itself
            up = np.where(np.sum(up * up, axis=0, keepdims=True) > 0.0, up, m)
            dn = np.where(np.sum(dn * dn, axis=0, keepdims=True) > 0.0, dn, m)
        out += ja * (up - dn) / (2.0 * cell[comp])
    return out


def ll_torque(m, H, mat: Material, grid=None, cell=None, pbc=None) -> np.ndarray:
    """Eq. (1): dm/dt = -gamma/(1+alpha^2) [ m x H + alpha m x (m x H) ]  (M = Ms m).
    Eq. (7): - c_ad b_j/(1+alpha^2) m x (m x (j.grad) m) - b_j (xi-alpha)/(1+alpha^2) m x (j.grad) m,
    b_j = P muB / (e Ms (1+xi^2)) (Eq. (8)); c_ad = 1 + alpha xi, or 1 when
    stt_literal_eq7 (reading A7)."""
    a = mat.alpha
    mxH = np.cross(m, H, axis=0)
    mxmxH = np.cross(m, mxH, axis=0)
    dmdt = -(mat.gamma0 / (1.0 + a * a)) * (mxH + a * mxmxH)
    if any(v != 0.0 for v in mat.j):
        bj = mat.P * MUB / (QE * mat.Ms * (1.0 + mat.xi ** 2))
        D = bj * j_dot_grad_m(m, mat, grid, cell, pbc)
        c_ad = 1.0 if mat.stt_literal_eq7 else 1.0 + a * mat.xi
        mxD = np.cross(m, D, axis=0)
        mxmxD = np.cross(m, mxD, axis=0)
        dmdt = dmdt - (c_ad / (1.0 + a * a)) * mxmxD - ((mat.xi - a) / (1.0 + a * a)) * mxD
    return dmdt


# --------------------------------------------------------------------------
# Runge-Kutta integrators
# --------------------------------------------------------------------------
def _F(*args):
    return [Fraction(a) if not isinstance(a, tuple) else Fraction(*a) for a in args]


# Butcher tableaux: (c, A rows, b, b* or None).  Exact rationals; tests check the
# order conditions on exactly these objects.
TABLEAUX = {
    # RK1: Euler's method
    "rk1": ([Fraction(0)], [[]], [Fraction(1)], None),
    # RK2: Heun's method
    "rk2": (_F(0, 1), [[], _F(1)], _F((1, 2), (1, 2)), None),
    # RK12: Heun-Euler, adaptive: Heun's solution, Euler's as the embedded one
    "rk12": (_F(0, 1), [[], _F(1)], _F((1, 2), (1, 2)), _F(1, 0)),
    # RK3: Kutta's third-order method
    "rk3": (_F(0, (1, 2), 1), [[], _F((1, 2)), _F(-1, 2)], _F((1, 6), (2, 3), (1, 6)), None),
    # RK23: Bogacki-Shampine 3(2), adaptive, first-same-as-last
    "rk23": (_F(0, (1, 2), (3, 4), 1),
             [[], _F((1, 2)), _F(0, (3, 4)), _F((2, 9), (1, 3), (4, 9))],
             _F((2, 9), (1, 3), (4, 9), 0), _F((7, 24), (1, 4), (1, 3), (1, 8))),
    # RKCK: Cash-Karp 5(4), adaptive
    "rkck": (_F(0, (1, 5), (3, 10), (3, 5), 1, (7, 8)),
             [[],
              _F((1, 5)),
              _F((3, 40), (9, 40)),
              _F((3, 10), (-9, 10), (6, 5)),
              _F((-11, 54), (5, 2), (-70, 27), (35, 27)),
              _F((1631, 55296), (175, 512), (575, 13824), (44275, 110592), (253, 4096))],
             _F((37, 378), 0, (250, 621), (125, 594), 0, (512, 1771)),
             _F((2825, 27648), 0, (18575, 48384), (13525, 55296), (277, 14336), (1, 4))),
    # RK4: classical Runge-Kutta
    "rk4": (_F(0, (1, 2), (1, 2), 1),
            [[], _F((1, 2)), _F(0, (1, 2)), _F(0, 0, 1)],
            _F((1, 6), (1, 3), (1, 3), (1, 6)), None),
    # RKDP: Dormand-Prince 5(4)
    "rkdp": (_F(0, (1, 5), (3, 10), (4, 5), (8, 9), 1, 1),
             [[],
              _F((1, 5)),
              _F((3, 40), (9, 40)),
              _F((44, 45), (-56, 15), (32, 9)),
              _F((19372, 6561), (-25360, 2187), (64448, 6561), (-212, 729)),
              _F((9017, 3168), (-355, 33), (46732, 5247), (49, 176), (-5103, 18656)),
              _F((35, 384), 0, (500, 1113), (125, 192), (-2187, 6784), (11, 84))],
             _F((35, 384), 0, (500, 1113), (125, 192), (-2187, 6784), (11, 84), 0),
             _F((5179, 57600), 0, (7571, 16695), (393, 640), (-92097, 339200), (187, 2100),
                (1, 40))),
}


def _normalise(m):
    """Unit vectors; the zero vector of an empty cell (reading A15) stays zero."""
    n = np.sqrt(np.sum(m * m, axis=0, keepdims=True))
    return np.where(n > 0.0, m / np.where(n > 0.0, n, 1.0), 0.0)


def rk4_step(f, m, dt):
    """Classical RK4; f(m) -> dm/dt.  m <- normalise(m + dt/6 (k1+2k2+2k3+k4));
    no normalisation between stages (reading A10)."""
    k1 = f(m)
    k2 = f(m + 0.5 * dt * k1)
    k3 = f(m + 0.5 * dt * k2)
    k4 = f(m + dt * k3)
    return _normalise(m + (dt / 6.0) * (k1 + 2.0 * k2 + 2.0 * k3 + k4))


def rk1_step(f, m, dt):
    """Euler's method, the step the paper times."""
    return _normalise(m + dt * f(m))


def rkdp_step(f, m, dt, k1=None):
    """One Dormand-Prince 5(4) trial step (reading A10).
    Returns (m_new, err, k7):  m_new = normalise(m + dt sum_{s<=6} b_s k_s);
    k7 = f(m_new) (FSAL on the renormalised state);
    err = dt * max_i || sum_{s=1..7} (b_s - b*_s) k_s(i) ||_2."""
    c, A, b, bs = TABLEAUX["rkdp"]
    k = [f(m) if k1 is None else k1]
    for s in range(1, 6):
        ms = m + dt * sum(float(A[s][j]) * k[j] for j in range(s) if A[s][j] != 0)
        k.append(f(ms))
    m_new = _normalise(m + dt * sum(float(b[j]) * k[j] for j in range(6) if b[j] != 0))
    k.append(f(m_new))
    e = sum(float(b[j] - bs[j]) * k[j] for j in range(7) if b[j] != bs[j])
    err = dt * float(np.max(np.sqrt(np.sum(e * e, axis=0))))
    return m_new, err, k[6]


# order p of the propagated solution: the exponent of the step-size rule is 1/p (reading A10)
ORDER = {"rk1": 1, "rk2": 2, "rk12": 2, "rk3": 3, "rk23": 3, "rk4": 4, "rkck": 5, "rkdp": 5}
FSAL = ("rk23", "rkdp")      # last row of A equals b: the last stage is f(new state)


def rk_step(f, m, dt, name, k1=None):
    """One step of any tableau of TABLEAUX, stage by stage as the textbook states it
    (reading A10).  k_s = f(m + dt sum_j a_sj k_j), no normalisation between
    stages; m_new = normalise(m + dt sum_s b_s k_s).  For the first-same-as-last pairs the last
    stage is evaluated on the renormalised m_new and returned for reuse as the next k_1.
    Embedded pairs: err = dt max_i || sum_s (b_s - b*_s) k_s(i) ||_2, else err = None.
    Returns (m_new, err, k_last)."""
    c, A, b, bs = TABLEAUX[name]
    S = len(b)
    fsal = name in FSAL
    k = [f(m) if k1 is None else k1]
    for s in range(1, S - 1 if fsal else S):
        ms = m + dt * sum(float(A[s][j]) * k[j] for j in range(s) if A[s][j] != 0)
        k.append(f(ms))
    nb = S - 1 if fsal else S
    m_new = _normalise(m + dt * sum(float(b[j]) * k[j] for j in range(nb) if b[j] != 0))
    if fsal:
        k.append(f(m_new))
    err = None
    if bs is not None:
        e = sum(float(b[j] - bs[j]) * k[j] for j in range(S) if b[j] != bs[j])
        err = dt * float(np.max(np.sqrt(np.sum(e * e, axis=0))))
    return m_new, err, k[-1]


def rk_controller(dt, err, tol, name):
    """Reading A10 for any embedded pair: accept iff err <= tol;
    dt <- dt * clamp(0.8 (tol/err)^(1/p), 0.2, 2), p = ORDER[name] (err = 0 => factor 2)."""
    accept = err <= tol
    fac = 2.0 if err == 0.0 else min(2.0, max(0.2, 0.8 * (tol / err) ** (1.0 / ORDER[name])))
    return accept, dt * fac


def max_dm_step_length(f, m, max_dm):
    """PAPER.md:141 "a fixed maximum variation of m per step" for the fixed-step methods:
    dt = max_dm / max_i ||dm/dt(i)||_2, evaluated on the state at the start of the step."""
    k = f(m)
    return max_dm / float(np.max(np.sqrt(np.sum(k * k, axis=0)))), k


def average_m(m):
    """<m> over all cells (PAPER.md:273 output quantity)."""
    return m.reshape(3, -1).mean(axis=1)


def rkdp_controller(dt, err, tol):
    """Reading A10: accept iff err <= tol; dt <- dt * clamp(0.8 (tol/err)^(1/5), 0.2, 2)
    (err = 0 => factor 2)."""
    accept = err <= tol
    fac = 2.0 if err == 0.0 else min(2.0, max(0.2, 0.8 * (tol / err) ** 0.2))
    return accept, dt * fac
