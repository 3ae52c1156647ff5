"""Pins for the oracle's field terms, torque and integrators (oracle/mm_oracle.py).

Each test checks the oracle against something other than itself: a closed form, an
invariant the paper or BASELINE.json names, a textbook special case, or brute force.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import mm_oracle as orc

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rand_m(shape, seed):
    g = np.random.default_rng(seed).standard_normal((3,) + shape)
    return g / np.sqrt((g * g).sum(axis=0, keepdims=True))


# ---------------------------------------------------------------- demag: O1 == O2
@pytest.mark.parametrize("grid,cell,pbc", [
    ((6, 5, 1), (4e-9, 4e-9, 4e-9), (0, 0, 0)),
    ((4, 3, 3), (3e-9, 5e-9, 2e-9), (0, 0, 0)),
    ((5, 4, 2), (1.0, 2.0, 0.5), (0, 0, 0)),
    ((6, 4, 1), (4e-9, 4e-9, 2e-9), (2, 2, 0)),
    ((5, 3, 2), (4e-9, 3e-9, 2e-9), (1, 0, 0)),
    ((4, 4, 3), (2e-9, 2e-9, 2e-9), (0, 1, 2)),
])
def test_fft_route_equals_direct_pair_sum(grid, cell, pbc):
    # BASELINE.json invariant: "The FFT path agrees with the brute-force demag sum"
    Ms = 8e5
    m = _rand_m((grid[2], grid[1], grid[0]), 11)
    K = orc.demag_kernel(grid, cell, pbc)
    Kh = orc.demag_kernel_fft(K)
    assert np.abs(Kh.imag).max() <= 1e-13 * np.abs(Kh.real).max()
    H2 = orc.demag_field_fft(m, Ms, grid, pbc, Kh)
    H1 = orc.demag_field_direct(m, Ms, grid, cell, pbc)
    assert np.abs(H1 - H2).max() <= 1e-12 * np.abs(H1).max()


def test_direct_sum_is_the_textbook_double_loop():
    # demag_field_direct organises the pair sum by offset; this is the literal double loop
    grid, cell, Ms = (3, 2, 2), (1.0, 1.5, 0.5), 2.0
    m = _rand_m((2, 2, 3), 5)
    H = orc.demag_field_direct(m, Ms, grid, cell)
    cells = [(x, y, z) for z in range(2) for y in range(2) for x in range(3)]
    for (x, y, z) in cells:
        h = np.zeros(3)
        for (u, v, w) in cells:
            n = orc.tensor_at([[x - u, y - v, z - w]], cell)[0]
            N = np.array([[n[0], n[3], n[4]], [n[3], n[1], n[5]], [n[4], n[5], n[2]]])
            h -= Ms * N @ m[:, w, v, u]
        assert np.allclose(H[:, z, y, x], h, rtol=1e-12, atol=1e-14)


@pytest.mark.parametrize("grid,cell", [((32, 32, 1), (4.0, 4.0, 4.0)), ((8, 4, 2), (3.0, 3.0, 3.0)),
                                       ((16, 4, 1), (3.90625, 3.90625, 4.0))])
def test_uniform_sample_mean_field_is_sample_demag_factor(grid, cell):
    """Whole-pipeline pin: for uniform m along a, mean(H_a)/Ms over an open sample equals minus the
    self term of ONE cell with the size of the whole sample (coarse graining taken to the limit)."""
    Ms = 8e5
    Kh = orc.demag_kernel_fft(orc.demag_kernel(grid, cell))
    big = orc.tensor_at([[0, 0, 0]], tuple(g * c for g, c in zip(grid, cell)))[0]
    for a in range(3):
        m = np.zeros((3, grid[2], grid[1], grid[0]))
        m[a] = 1.0
        H = orc.demag_field_fft(m, Ms, grid, (0, 0, 0), Kh)
        assert abs(H[a].mean() / Ms + big[a]) < 1e-13
        for b in range(3):
            if b != a:
                assert abs(H[b].mean()) < 1e-10 * Ms


def test_periodic_film_uniform_states():
    # xy-periodic film: uniform in-plane m -> H ~ 0 ; uniform m_z -> H_z -> -Ms as images grow
    grid, cell, Ms = (4, 4, 1), (4e-9, 4e-9, 2e-9), 8e5
    prev = 0.0
    for p in (2, 5, 12):
        Kh = orc.demag_kernel_fft(orc.demag_kernel(grid, cell, (p, p, 0)))
        m = np.zeros((3, 1, 4, 4))
        m[2] = 1.0
        Hz = orc.demag_field_fft(m, Ms, grid, (p, p, 0), Kh)[2]
        assert np.ptp(Hz) < 1e-9 * Ms
        assert prev < -Hz.mean() / Ms < 1.0
        prev = -Hz.mean() / Ms
        m = np.zeros((3, 1, 4, 4))
        m[0] = 1.0
        Hx = orc.demag_field_fft(m, Ms, grid, (p, p, 0), Kh)[0]
        assert 0.0 < -Hx.mean() / Ms < 0.5 * (1.0 - prev) + 1e-12
    assert prev > 0.97


def test_demag_energy_positive_and_reciprocal():
    grid, cell, Ms = (6, 5, 3), (3e-9, 3e-9, 3e-9), 8e5
    Kh = orc.demag_kernel_fft(orc.demag_kernel(grid, cell))
    m1 = _rand_m((3, 5, 6), 1)
    m2 = _rand_m((3, 5, 6), 2)
    H1 = orc.demag_field_fft(m1, Ms, grid, (0, 0, 0), Kh)
    H2 = orc.demag_field_fft(m2, Ms, grid, (0, 0, 0), Kh)
    assert -(m1 * H1).sum() > 0
    assert abs((m1 * H2).sum() - (m2 * H1).sum()) < 1e-12 * abs((m1 * H2).sum())


# ---------------------------------------------------------------- exchange, anisotropy, Zeeman
def test_exchange_zero_for_uniform_m():
    # BASELINE.json invariant; discriminates reading A3 at face cells
    mat = orc.Material(Ms=8e5, Aex=1.3e-11)
    for pbc in ((0, 0, 0), (1, 1, 0), (1, 1, 1)):
        m = np.zeros((3, 3, 4, 5))
        m[0], m[1], m[2] = 0.6, 0.0, 0.8
        H = orc.exchange_field(m, mat, (5, 4, 3), (4e-9, 4e-9, 4e-9), pbc)
        assert np.all(H == 0.0)


def test_exchange_helix_eigenvalue():
    # periodic helix m = (cos qx, sin qx, 0): H_ex = (2A/mu0Ms) * 2(cos(q d) - 1)/d^2 * m   (Eq. (3))
    mat = orc.Material(Ms=8e5, Aex=1.3e-11)
    Nx, d = 16, 4e-9
    q = 2 * math.pi * 3 / (Nx * d)
    x = np.arange(Nx) * d
    m = np.zeros((3, 1, 2, Nx))
    m[0] = np.cos(q * x)[None, None, :]
    m[1] = np.sin(q * x)[None, None, :]
    H = orc.exchange_field(m, mat, (Nx, 2, 1), (d, d, d), (1, 1, 0))
    lam = (2 * mat.Aex / (orc.MU0 * mat.Ms)) * 2 * (math.cos(q * d) - 1) / d ** 2
    assert np.allclose(H, lam * m, rtol=1e-12, atol=1e-6)
    # 2D: a z axis with one cell contributes nothing -- same numbers with pbc z set
    H2 = orc.exchange_field(m, mat, (Nx, 2, 1), (d, d, d), (1, 1, 1))
    assert np.array_equal(H, H2)


def test_exchange_open_boundary_is_neumann_and_matches_brute_force():
    mat = orc.Material(Ms=1.1e6, Aex=2e-11)
    grid, cell = (4, 3, 2), (5e-9, 4e-9, 3e-9)
    m = _rand_m((2, 3, 4), 7)
    H = orc.exchange_field(m, mat, grid, cell)
    pref = 2 * mat.Aex / (orc.MU0 * mat.Ms)
    for z in range(2):
        for y in range(3):
            for x in range(4):
                h = np.zeros(3)
                for (dx, dy, dz, d) in ((1, 0, 0, cell[0]), (-1, 0, 0, cell[0]), (0, 1, 0, cell[1]),
                                        (0, -1, 0, cell[1]), (0, 0, 1, cell[2]), (0, 0, -1, cell[2])):
                    u, v, w = x + dx, y + dy, z + dz
                    if 0 <= u < 4 and 0 <= v < 3 and 0 <= w < 2:
                        h += pref * (m[:, w, v, u] - m[:, z, y, x]) / d ** 2
                assert np.allclose(H[:, z, y, x], h, rtol=1e-12)


def test_exchange_in_kernel_variant_differs_only_at_open_faces_and_gives_the_same_torque():
    """PAPER.md:85 (reading A3').  Pins: (i) interior cells: identical to the free-boundary stencil;
    (ii) a cell with k missing neighbours along axis a differs by exactly -(2A/mu0 Ms d_a^2) k m_i, a field
    parallel to m_i; hence (iii) the torque is the same under both readings; (iv) periodic axes: identical;
    (v) it equals the circular convolution of the zero-padded m with the stencil kernel."""
    rng = np.random.default_rng(8)
    grid, cell = (6, 5, 4), (3e-9, 4e-9, 5e-9)
    mat = orc.Material(Ms=8e5, Aex=1.3e-11, alpha=0.1)
    m = rng.standard_normal((3, grid[2], grid[1], grid[0]))
    m /= np.sqrt((m * m).sum(0))
    Hn = orc.exchange_field(m, mat, grid, cell)
    Hk = orc.exchange_field_in_kernel(m, mat, grid, cell)
    assert np.allclose(Hn[:, 1:-1, 1:-1, 1:-1], Hk[:, 1:-1, 1:-1, 1:-1], rtol=0, atol=1e-6)
    pref = 2 * mat.Aex / (orc.MU0 * mat.Ms)
    miss = np.zeros(m.shape[1:])
    for a, (n, d) in zip((2, 1, 0), zip(grid, cell)):           # array axes z, y, x <-> grid x, y, z reversed
        pass
    for ax_arr, n, d in ((2, grid[0], cell[0]), (1, grid[1], cell[1]), (0, grid[2], cell[2])):
        idx = np.arange(n)
        k = ((idx == 0).astype(float) + (idx == n - 1).astype(float)) / d ** 2
        shape = [1, 1, 1]; shape[ax_arr] = n
        miss = miss + k.reshape(shape)
    assert np.allclose(Hk - Hn, -pref * miss[None] * m, rtol=0, atol=1e-6 * np.abs(Hn).max())
    assert np.allclose(orc.ll_torque(m, Hk, mat), orc.ll_torque(m, Hn, mat), rtol=0, atol=1e-9 * np.abs(orc.ll_torque(m, Hn, mat)).max())
    assert np.allclose(orc.exchange_field(m, mat, grid, cell, (1, 1, 1)), orc.exchange_field_in_kernel(m, mat, grid, cell, (1, 1, 1)))
    # (v) circular convolution of the padded state with the stencil
    P = [2 * n for n in grid]
    ker = np.zeros((P[2], P[1], P[0]))
    for ax_arr, d in ((2, cell[0]), (1, cell[1]), (0, cell[2])):
        ker[0, 0, 0] -= 2 * pref / d ** 2
        for sgn in (1, -1):
            i = [0, 0, 0]; i[ax_arr] = sgn
            ker[tuple(i)] += pref / d ** 2
    mp = np.zeros((3, P[2], P[1], P[0])); mp[:, :grid[2], :grid[1], :grid[0]] = m
    conv = np.fft.ifftn(np.fft.fftn(mp, axes=(1, 2, 3)) * np.fft.fftn(ker)[None], axes=(1, 2, 3)).real
    assert np.allclose(conv[:, :grid[2], :grid[1], :grid[0]], Hk, rtol=0, atol=1e-8 * np.abs(Hk).max())


def test_exchange_on_a_staircase_shape():
    """Reading A15.  Pins: (i) no empty cell: the plain stencil; (ii) an L-shaped sample
    against plain Python loops over cell pairs; (iii) uniform m on any shape: zero; (iv) empty cells get
    no field, and normalisation leaves them empty."""
    rng = np.random.default_rng(4)
    grid, cell = (5, 4, 3), (3e-9, 4e-9, 5e-9)
    mat = orc.Material(Ms=8e5, Aex=1.3e-11, geometry=True)
    m = rng.standard_normal((3, grid[2], grid[1], grid[0]))
    m /= np.sqrt((m * m).sum(0))
    assert np.allclose(orc.exchange_field_geometry(m, mat, grid, cell), orc.exchange_field(m, mat, grid, cell))
    shape = np.ones((grid[2], grid[1], grid[0]), dtype=bool)
    shape[:, 2:, 3:] = False                       # cut a corner out: L shape
    shape[1, 1, 1] = False                         # and a hole
    mg = m * shape[None]
    H = orc.exchange_field_geometry(mg, mat, grid, cell)
    pref = 2 * mat.Aex / (orc.MU0 * mat.Ms)
    ref = np.zeros_like(mg)
    for z in range(grid[2]):
        for y in range(grid[1]):
            for x in range(grid[0]):
                if not shape[z, y, x]:
                    continue
                for dz, dy, dx, d in ((0, 0, 1, cell[0]), (0, 0, -1, cell[0]), (0, 1, 0, cell[1]), (0, -1, 0, cell[1]),
                                      (1, 0, 0, cell[2]), (-1, 0, 0, cell[2])):
                    zz, yy, xx = z + dz, y + dy, x + dx
                    if 0 <= zz < grid[2] and 0 <= yy < grid[1] and 0 <= xx < grid[0] and shape[zz, yy, xx]:
                        ref[:, z, y, x] += pref * (mg[:, zz, yy, xx] - mg[:, z, y, x]) / d ** 2
    assert np.allclose(H, ref, rtol=0, atol=1e-9 * np.abs(ref).max())
    assert np.all(H[:, ~shape] == 0.0)
    mu = np.zeros_like(m); mu[0] = 1.0
    assert np.abs(orc.exchange_field_geometry(mu * shape[None], mat, grid, cell)).max() == 0.0
    nrm = orc._normalise(1.7 * mg)
    assert np.all(nrm[:, ~shape] == 0.0) and np.allclose((nrm * nrm).sum(0)[shape], 1.0)


def test_anisotropy_special_cases():
    mat = orc.Material(Ms=1.1e6, Ku=5e5, anis_u=(0.0, 0.0, 2.0))
    m = np.zeros((3, 1, 1, 2))
    m[2, 0, 0, 0] = 1.0           # parallel
    m[0, 0, 0, 1] = 1.0           # perpendicular
    H = orc.anisotropy_field(m, mat)
    assert np.allclose(H[:, 0, 0, 0], [0, 0, 2 * 5e5 / (orc.MU0 * 1.1e6)], rtol=1e-14)
    assert np.all(H[:, 0, 0, 1] == 0)
    # field = -(1/mu0 Ms) dE/dm of E = Ku (1 - (m.u)^2), by finite differences
    u = np.array([1.0, 2.0, -1.0])
    mat = orc.Material(Ms=8e5, Ku=1e4, anis_u=tuple(u))
    un = u / np.linalg.norm(u)
    m0 = np.array([0.3, -0.5, 0.81])
    E = lambda v: mat.Ku * (1 - (v @ un) ** 2)
    g = np.array([(E(m0 + e) - E(m0 - e)) / 2e-6 for e in 1e-6 * np.eye(3)])
    H = orc.anisotropy_field(m0.reshape(3, 1, 1, 1), mat).ravel()
    assert np.allclose(H, -g / (orc.MU0 * mat.Ms), rtol=1e-8)


def test_cubic_anisotropy_field_is_minus_the_energy_gradient():
    """Eq. (5).  Pins: (i) the field is -(1/mu0 Ms) dE/dm of the printed energy, checked by
    central differences of that energy; (ii) along a cube axis the energy and the field vanish (K1 > 0:
    <100> easy); (iii) along <111> the energy is K1/3 + K2/27; (iv) it is invariant under the cube group
    (a permutation / sign change of the axes)."""
    rng = np.random.default_rng(3)
    mat = orc.Material(Ms=4.8e5, K1=-4.5e3, K2=2.3e3, anis_c1=(1.0, 1.0, 0.0), anis_c2=(-1.0, 1.0, 0.3))
    m = rng.standard_normal((3, 2, 3, 4))
    m /= np.sqrt((m * m).sum(0))
    H = orc.cubic_anisotropy_field(m, mat)
    h = 1e-6
    for c in range(3):
        dm = np.zeros_like(m); dm[c] = h
        dE = (orc.cubic_anisotropy_energy_density(m + dm, mat) - orc.cubic_anisotropy_energy_density(m - dm, mat)) / (2 * h)
        assert np.allclose(H[c], -dE / (orc.MU0 * mat.Ms), rtol=1e-7, atol=1e-6)
    c1, c2, c3 = orc.cubic_axes(mat)
    assert abs(np.dot(c1, c2)) < 1e-15 and abs(np.dot(c1, c3)) < 1e-15 and np.allclose(np.cross(c1, c2), c3)
    for ax in (c1, c2, c3):
        ma = ax.reshape(3, 1, 1, 1)
        assert abs(orc.cubic_anisotropy_energy_density(ma, mat)).max() < 1e-12
        assert np.abs(orc.cubic_anisotropy_field(ma, mat)).max() < 1e-9
    m111 = ((c1 + c2 + c3) / np.sqrt(3.0)).reshape(3, 1, 1, 1)
    assert np.isclose(orc.cubic_anisotropy_energy_density(m111, mat)[0, 0, 0], mat.K1 / 3 + mat.K2 / 27)
    mat2 = orc.Material(Ms=4.8e5, K1=-4.5e3, K2=2.3e3, anis_c1=tuple(-c3), anis_c2=tuple(c1))
    assert np.allclose(orc.cubic_anisotropy_field(m, mat2), H, rtol=0, atol=1e-9)
    # and it enters H_eff
    pb = orc.Problem((4, 3, 2), (3e-9, 3e-9, 3e-9), (0, 0, 0), mat, demag="none")
    assert np.allclose(pb.heff(m), H + orc.exchange_field(m, mat, (4, 3, 2), (3e-9,) * 3) + orc.zeeman_field(m, mat))


def test_zeeman():
    mat = orc.Material(Ms=8e5, Bext=(0.0, 10e-3, 0.0))
    H = orc.zeeman_field(np.zeros((3, 2, 2, 2)), mat)
    assert np.allclose(H[1], 10e-3 / orc.MU0) and np.all(H[0] == 0) and np.all(H[2] == 0)


# ---------------------------------------------------------------- torque and integrators
def test_torque_is_perpendicular_to_m():
    # BASELINE.json invariant "|M| = Ms is conserved by the torque"
    mat = orc.Material(Ms=8e5, Aex=1.3e-11, alpha=0.1, j=(1e12, 0, 0), P=0.5, xi=0.04)
    grid, cell = (6, 4, 2), (4e-9, 4e-9, 2e-9)
    m = _rand_m((2, 4, 6), 3)
    H = 1e5 * np.random.default_rng(4).standard_normal(m.shape)
    t = orc.ll_torque(m, H, mat, grid, cell, (0, 0, 0))
    assert np.abs((m * t).sum(axis=0)).max() < 1e-15 * np.abs(t).max() * 10


def _macrospin(alpha, Hz, gamma0=orc.GAMMA0_DEFAULT):
    # single cubic cell: N = I/3 -> demag field parallel to m, no torque
    mat = orc.Material(Ms=8e5, alpha=alpha, gamma0=gamma0, Bext=(0.0, 0.0, orc.MU0 * Hz))
    return orc.Problem((1, 1, 1), (5e-9, 5e-9, 5e-9), (0, 0, 0), mat, demag="fft")


def _macrospin_exact(m0, alpha, Hz, gamma0, t):
    # from Eq. (1): m_z = tanh(alpha g' H t + atanh m_z0), phi = phi0 + g' H t, g' = gamma0/(1+alpha^2)
    gp = gamma0 / (1 + alpha ** 2)
    mz = math.tanh(alpha * gp * Hz * t + math.atanh(m0[2]))
    phi = math.atan2(m0[1], m0[0]) + gp * Hz * t
    s = math.sqrt(1 - mz * mz)
    return np.array([s * math.cos(phi), s * math.sin(phi), mz])


@pytest.mark.parametrize("alpha,gamma0", [(0.0, orc.GAMMA0_DEFAULT), (0.1, orc.GAMMA0_DEFAULT),
                                          (0.5, 1.76e5)])
def test_macrospin_larmor_and_damping_closed_form(alpha, gamma0):
    Hz = 1e5
    pb = _macrospin(alpha, Hz, gamma0)
    m0 = np.array([0.6, 0.0, 0.8])
    m = m0.reshape(3, 1, 1, 1).copy()
    T = 2 * math.pi / (gamma0 * Hz)          # ~ one Larmor period
    n = 400
    dt = T / n
    for _ in range(n):
        m = orc.rk4_step(pb.torque, m, dt)
    assert np.allclose(m.ravel(), _macrospin_exact(m0, alpha, Hz, gamma0, T), atol=2e-8)
    # Dormand-Prince, fixed steps
    m = m0.reshape(3, 1, 1, 1).copy()
    k1 = None
    for _ in range(100):
        m, err, k1 = orc.rkdp_step(pb.torque, m, T / 100, k1)
    assert np.allclose(m.ravel(), _macrospin_exact(m0, alpha, Hz, gamma0, T), atol=2e-8)


def test_convergence_orders():
    alpha, Hz = 0.3, 2e5
    pb = _macrospin(alpha, Hz)
    m0 = np.array([0.8, 0.0, 0.6])
    T0 = 1.0 / (orc.GAMMA0_DEFAULT * Hz)

    def run(stepper, n, T):
        m = m0.reshape(3, 1, 1, 1).copy()
        k1 = None
        for _ in range(n):
            if stepper == "rk4":
                m = orc.rk4_step(pb.torque, m, T / n)
            elif stepper == "rk1":
                m = orc.rk1_step(pb.torque, m, T / n)
            else:
                m, _, k1 = orc.rkdp_step(pb.torque, m, T / n, k1)
        return np.abs(m.ravel() - _macrospin_exact(m0, alpha, Hz, orc.GAMMA0_DEFAULT, T)).max()

    for stepper, order, ns, T in (("rk1", 1, (40, 80), 3 * T0), ("rk4", 4, (6, 12), 3 * T0),
                                  ("rkdp", 5, (16, 32), 2 * T0)):
        e1, e2 = run(stepper, ns[0], T), run(stepper, ns[1], T)
        assert abs(math.log2(e1 / e2) - order) < 0.45, (stepper, e1, e2)


def _order_conditions(c, A, b, order):
    s = len(b)
    A = [list(r) + [Fraction(0)] * (s - len(r)) for r in A]
    Ac = [sum(A[i][j] * c[j] for j in range(s)) for i in range(s)]
    Ac2 = [sum(A[i][j] * c[j] ** 2 for j in range(s)) for i in range(s)]
    Ac3 = [sum(A[i][j] * c[j] ** 3 for j in range(s)) for i in range(s)]
    AAc = [sum(A[i][j] * Ac[j] for j in range(s)) for i in range(s)]
    AAc2 = [sum(A[i][j] * Ac2[j] for j in range(s)) for i in range(s)]
    AAAc = [sum(A[i][j] * AAc[j] for j in range(s)) for i in range(s)]
    AcAc = [sum(A[i][j] * c[j] * Ac[j] for j in range(s)) for i in range(s)]
    dot = lambda *vs: sum(b[i] * math.prod(v[i] for v in vs) for i in range(s))
    one = [Fraction(1)] * s
    conds = [(1, dot(one), Fraction(1)),
             (2, dot(c), Fraction(1, 2)),
             (3, dot(c, c), Fraction(1, 3)), (3, dot(Ac), Fraction(1, 6)),
             (4, dot(c, c, c), Fraction(1, 4)), (4, dot(c, Ac), Fraction(1, 8)),
             (4, dot(Ac2), Fraction(1, 12)), (4, dot(AAc), Fraction(1, 24)),
             (5, dot(c, c, c, c), Fraction(1, 5)), (5, dot(c, c, Ac), Fraction(1, 10)),
             (5, dot(Ac, Ac), Fraction(1, 20)), (5, dot(c, Ac2), Fraction(1, 15)),
             (5, dot(Ac3), Fraction(1, 20)), (5, dot(c, AAc), Fraction(1, 30)),
             (5, dot(AcAc), Fraction(1, 40)), (5, dot(AAc2), Fraction(1, 60)),
             (5, dot(AAAc), Fraction(1, 120))]
    return all(v == t for (o, v, t) in conds if o <= order)


def test_butcher_tableaux_satisfy_order_conditions_exactly():
    for name, order, order_star in (("rk1", 1, None), ("rk2", 2, None), ("rk12", 2, 1), ("rk3", 3, None),
                                    ("rk23", 3, 2), ("rk4", 4, None), ("rkck", 5, 4), ("rkdp", 5, 4)):
        assert orc.ORDER[name] == order
        c, A, b, bs = orc.TABLEAUX[name]
        for i, row in enumerate(A):
            assert sum(row, Fraction(0)) == c[i]
        assert _order_conditions(c, A, b, order)
        if order < 5:          # the condition list above stops at order 5
            assert not _order_conditions(c, A, b, order + 1)
        if bs is not None:
            assert _order_conditions(c, A, bs, order_star)
            assert not _order_conditions(c, A, bs, order_star + 1)


def test_generic_stepper_reduces_to_the_written_out_ones_and_converges_at_its_order():
    """rk_step from the tableau == the hand-written rk1 / rk4 / rkdp steps; every other tableau
    converges on the macrospin closed form (pin P14) at its nominal order (pin P15)."""
    alpha, Hz = 0.3, 2e5
    pb = _macrospin(alpha, Hz)
    m0 = np.array([0.8, 0.0, 0.6])
    T0 = 1.0 / (orc.GAMMA0_DEFAULT * Hz)
    ms = m0.reshape(3, 1, 1, 1)
    dt = 0.2 * T0
    assert np.allclose(orc.rk_step(pb.torque, ms, dt, "rk1")[0], orc.rk1_step(pb.torque, ms, dt), rtol=0, atol=1e-15)
    assert np.allclose(orc.rk_step(pb.torque, ms, dt, "rk4")[0], orc.rk4_step(pb.torque, ms, dt), rtol=0, atol=1e-15)
    a, ea, ka = orc.rk_step(pb.torque, ms, dt, "rkdp")
    b, eb, kb = orc.rkdp_step(pb.torque, ms, dt)
    assert np.allclose(a, b, rtol=0, atol=1e-15) and math.isclose(ea, eb, rel_tol=1e-12) and np.allclose(ka, kb)

    def run(name, n, T):
        m, k1 = ms.copy(), None
        for _ in range(n):
            m, _, kl = orc.rk_step(pb.torque, m, T / n, name, k1)
            k1 = kl if name in orc.FSAL else None
        return np.abs(m.ravel() - _macrospin_exact(m0, alpha, Hz, orc.GAMMA0_DEFAULT, T)).max()

    for name, ns, T in (("rk2", (20, 40), 3 * T0), ("rk12", (20, 40), 3 * T0), ("rk3", (10, 20), 3 * T0),
                        ("rk23", (10, 20), 3 * T0), ("rkck", (12, 24), 2 * T0)):
        e1, e2 = run(name, ns[0], T), run(name, ns[1], T)
        assert abs(math.log2(e1 / e2) - orc.ORDER[name]) < 0.45, (name, e1, e2)
    # embedded error estimates scale with the order of the lower solution + 1
    for name, lo in (("rk12", 2), ("rk23", 3), ("rkck", 5)):
        _, e1, _ = orc.rk_step(pb.torque, ms, T0, name)
        _, e2, _ = orc.rk_step(pb.torque, ms, T0 / 2, name)
        assert abs(math.log2(e1 / e2) - lo) < 0.7, (name, e1, e2)
    # controller and the maximum-variation step length
    ok, dtn = orc.rk_controller(1e-13, 1e-5, 1e-5, "rk23")
    assert ok and math.isclose(dtn, 0.8e-13)
    ok, dtn = orc.rk_controller(1e-13, 8e-5, 1e-5, "rk23")
    assert (not ok) and math.isclose(dtn, 0.4e-13)
    dtm, k = orc.max_dm_step_length(pb.torque, ms, 0.01)
    assert math.isclose(dtm * np.sqrt((k * k).sum()), 0.01, rel_tol=1e-12)
    assert np.allclose(orc.average_m(np.concatenate([ms, -ms], axis=3)), 0.0)


def test_dormand_prince_tableau_matches_published_coefficients():
    rows = {}
    with open(os.path.join(GOLD, "dormand_prince_tableau.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            rows[k] = [Fraction(s) for s in v]
    c, A, b, bs = orc.TABLEAUX["rkdp"]
    assert rows["c"] == c and rows["b"] == b and rows["bstar"] == bs
    for i in range(1, 7):
        assert rows[f"a{i + 1}"] == A[i]


def test_rkdp_error_estimate_and_controller():
    pb = _macrospin(0.3, 2e5)
    m0 = np.array([0.8, 0.0, 0.6]).reshape(3, 1, 1, 1)
    T = 1.0 / (orc.GAMMA0_DEFAULT * 2e5)
    _, e1, _ = orc.rkdp_step(pb.torque, m0, T)
    _, e2, _ = orc.rkdp_step(pb.torque, m0, T / 2)
    assert 4.3 < math.log2(e1 / e2) < 5.7           # local error of the 4th-order solution ~ dt^5
    ok, dt = orc.rkdp_controller(1e-13, 1e-5, 1e-5)
    assert ok and math.isclose(dt, 0.8e-13)
    ok, dt = orc.rkdp_controller(1e-13, 1.0, 1e-5)
    assert (not ok) and math.isclose(dt, 0.2e-13)
    ok, dt = orc.rkdp_controller(1e-13, 0.0, 1e-5)
    assert ok and math.isclose(dt, 2e-13)


# ---------------------------------------------------------------- spin-transfer torque
def test_zhang_li_uniform_is_zero_and_helix_translates():
    Ms, A, d, Nx = 8e5, 1.3e-11, 4e-9, 32
    alpha = 0.1
    grid, cell, pbc = (Nx, 1, 1), (d, d, d), (1, 0, 0)
    j = 1e12
    P, xi = 0.5, alpha                       # xi = alpha: the (xi - alpha) term vanishes
    q = 2 * math.pi * 2 / (Nx * d)
    x = np.arange(Nx) * d
    m = np.zeros((3, 1, 1, Nx))
    m[0], m[1] = np.cos(q * x), np.sin(q * x)
    bj = P * orc.MUB / (orc.QE * Ms * (1 + xi ** 2))
    for literal, cad in ((False, 1 + alpha * xi), (True, 1.0)):
        mat = orc.Material(Ms=Ms, Aex=A, alpha=alpha, j=(j, 0, 0), P=P, xi=xi, stt_literal_eq7=literal)
        mu = np.zeros_like(m)
        mu[2] = 1.0
        assert np.all(orc.ll_torque(mu, np.zeros_like(m), mat, grid, cell, pbc) == 0.0)
        # exchange field of the helix is parallel to m -> only the STT moves it:
        Hex = orc.exchange_field(m, mat, grid, cell, pbc)
        t = orc.ll_torque(m, Hex, mat, grid, cell, pbc)
        # m x (m x D) = -D for D perpendicular to m  =>  dm/dt = cad/(1+alpha^2) D,
        # D = bj j sin(q d)/d * dm/dphi: rigid rotation at omega, pattern moves against j
        omega = cad / (1 + alpha ** 2) * bj * j * math.sin(q * d) / d
        dmdphi = np.stack([-m[1], m[0], m[2] * 0])
        assert np.allclose(t, omega * dmdphi, rtol=1e-10, atol=1e-10 * omega)
        assert omega > 0


def test_open_face_gradient_rule():
    mat = orc.Material(Ms=8e5, j=(0.0, 2.0, 0.0), P=0.5)
    m = _rand_m((1, 4, 3), 9)
    D = orc.j_dot_grad_m(m, mat, (3, 4, 1), (1.0, 0.5, 1.0), (0, 0, 0))
    assert np.allclose(D[:, 0, 0, :], 2.0 * (m[:, 0, 1, :] - m[:, 0, 0, :]) / (2 * 0.5))
    assert np.allclose(D[:, 0, 2, :], 2.0 * (m[:, 0, 3, :] - m[:, 0, 1, :]) / (2 * 0.5))
    assert np.allclose(D[:, 0, 3, :], 2.0 * (m[:, 0, 3, :] - m[:, 0, 2, :]) / (2 * 0.5))


# ---------------------------------------------------------------- thermal field
def test_philox_known_answers():
    with open(os.path.join(GOLD, "philox4x32_10_kat.txt")) as fh:
        rows = [l.split() for l in fh if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(s, 16) for s in r]
        out = orc.philox4x32_10(*v[:4], v[4], v[5])
        assert [int(o) for o in out] == v[6:]


def test_thermal_field_moments_and_amplitude():
    grid = (64, 64, 4)
    e0 = orc.thermal_eta(grid, seed=3, step=0)
    e1 = orc.thermal_eta(grid, seed=3, step=1)
    n = e0.size
    assert abs(e0.mean()) < 4 / math.sqrt(n)
    assert abs(e0.var() - 1) < 4 * math.sqrt(2 / n)
    assert abs(np.mean(e0 ** 4) - 3) < 0.15                      # Gaussian kurtosis
    assert abs(np.mean(e0 * e1)) < 4 / math.sqrt(n)              # uncorrelated in time
    assert abs(np.mean(e0[:, :, :, 1:] * e0[:, :, :, :-1])) < 4 / math.sqrt(n)   # and in space
    assert abs(np.mean(e0[0] * e0[1])) < 4 / math.sqrt(n / 3)    # and between components
    assert not np.array_equal(e0, orc.thermal_eta(grid, seed=4, step=0))
    # amplitude of Eq. (6) by hand for config 3 (4x4x2 nm, alpha 0.1, 300 K, dt 5e-14)
    mat = orc.Material(Ms=8e5, alpha=0.1, T=300.0)
    s = orc.thermal_sigma(mat, (4e-9, 4e-9, 2e-9), 5e-14)
    by_hand = math.sqrt(2 * 0.1 * 1.380649e-23 * 300 /
                        (2.211e5 * 4e-7 * math.pi * 8e5 * 32e-27 * 5e-14))
    assert math.isclose(s, by_hand, rel_tol=1e-12) and 1.5e6 < s < 1.55e6


def test_heff_is_the_sum_of_its_terms():
    mat = orc.Material(Ms=8e5, Aex=1.3e-11, alpha=0.1, Ku=1e4, anis_u=(1, 0, 0), Bext=(0, 1e-2, 0),
                       T=300.0, seed=7)
    grid, cell = (5, 4, 2), (3e-9, 3e-9, 3e-9)
    pb = orc.Problem(grid, cell, (0, 0, 0), mat)
    m = _rand_m((2, 4, 5), 2)
    H = pb.heff(m, step=3, dt_thermal=1e-13)
    parts = (orc.demag_field_direct(m, mat.Ms, grid, cell) + orc.exchange_field(m, mat, grid, cell)
             + orc.anisotropy_field(m, mat) + orc.zeeman_field(m, mat)
             + orc.thermal_field(mat, grid, cell, 3, 1e-13))
    assert np.allclose(H, parts, rtol=1e-12, atol=1e-6)


# ---------------------------------------------------------------- round-2 pins ("parity unpinned")
def test_current_gradient_on_a_staircase_shape():
    """j_dot_grad_m with geometry=True (reading A15): an empty or missing neighbour is
    replaced by the cell itself.  Pinned against plain Python loops on the L shape with a hole of
    test_exchange_on_a_staircase_shape; `zero instead of the cell itself` or a wrong axis fails."""
    rng = np.random.default_rng(11)
    grid, cell = (5, 4, 3), (3e-9, 4e-9, 5e-9)
    shape = np.ones((grid[2], grid[1], grid[0]), dtype=bool)
    shape[:, 2:, 3:] = False
    shape[1, 1, 1] = False
    m = rng.standard_normal((3, grid[2], grid[1], grid[0]))
    m /= np.sqrt((m * m).sum(0))
    mg = m * shape[None]
    j = (1.5e12, -0.7e12, 0.4e12)
    mat = orc.Material(Ms=8e5, j=j, P=0.5, xi=0.04, geometry=True)
    D = orc.j_dot_grad_m(mg, mat, grid, cell, (0, 0, 0))
    ref = np.zeros_like(mg)
    steps = ((0, 0, 1), (0, 1, 0), (1, 0, 0))            # (dz, dy, dx) of axis x, y, z
    for z in range(grid[2]):
        for y in range(grid[1]):
            for x in range(grid[0]):
                if not shape[z, y, x]:
                    continue
                for a, (dz, dy, dx) in enumerate(steps):
                    def at(s):
                        zz, yy, xx = z + s * dz, y + s * dy, x + s * dx
                        inside = 0 <= zz < grid[2] and 0 <= yy < grid[1] and 0 <= xx < grid[0]
                        return mg[:, zz, yy, xx] if inside and shape[zz, yy, xx] else mg[:, z, y, x]
                    ref[:, z, y, x] += j[a] * (at(+1) - at(-1)) / (2.0 * cell[a])
    occupied = np.broadcast_to(shape[None], mg.shape)
    assert np.allclose(D[occupied], ref[occupied], rtol=0, atol=1e-12 * np.abs(ref).max())
    # without empty cells the geometry branch is the plain rule
    mat0 = orc.Material(Ms=8e5, j=j, P=0.5, xi=0.04)
    assert np.allclose(orc.j_dot_grad_m(m, mat, grid, cell, (0, 0, 0)), orc.j_dot_grad_m(m, mat0, grid, cell, (0, 0, 0)))


def test_average_m_against_a_hand_sum():
    """<m> is the arithmetic mean per component over cells: `sum` instead of `mean`, or an
    average over the wrong axis, fails on this non-symmetric 2 x 1 x 3 state."""
    m = np.zeros((3, 3, 1, 2))
    vals = [(1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.6, 0.0, 0.8), (0.0, -0.6, 0.8), (0.0, 0.0, -1.0), (1.0, 0.0, 0.0)]
    for i, v in enumerate(vals):
        m[:, i // 2, 0, i % 2] = v
    want = (np.array([2.6, 0.4, 0.6]) / 6.0)
    assert np.allclose(orc.average_m(m), want, rtol=0, atol=1e-15)


def test_max_dm_step_length_takes_the_largest_cell():
    """dt = max_dm / max_i |dm/dt(i)|: with two uncoupled cells of different torque the larger
    one sets the step (a mean, a minimum or a per-component maximum fails)."""
    def f(m):
        k = np.zeros_like(m)
        k[:, 0, 0, 0] = (3.0, 4.0, 0.0)          # |k| = 5
        k[:, 0, 0, 1] = (1.0, 2.0, 2.0)          # |k| = 3
        k[:, 0, 0, 2] = (0.0, 0.0, 4.5)          # largest single component, |k| = 4.5
        return k
    m = np.zeros((3, 1, 1, 3)); m[2] = 1.0
    dt, k = orc.max_dm_step_length(f, m, 0.02)
    assert math.isclose(dt, 0.02 / 5.0, rel_tol=1e-15) and np.array_equal(k, f(m))


def test_thermal_eta_word_to_component_map_is_the_documented_convention():
    """Any map from the four Philox words to three N(0,1) numbers is a correct thermal field; which word
    feeds which component is a convention (reading A6).  This pins the documented one on one cell:
    eta = (r1 cos th1, r1 sin th1, r2 cos th2), u1 from word 0, th1 from word 1, u2 from word 2, th2 from
    word 3, counter = (cell, 0, step, 0)."""
    grid, seed, step = (3, 2, 2), 0x1234567, 7
    eta = orc.thermal_eta(grid, seed, step)
    cellidx = (1 * 2 + 1) * 3 + 2                  # z = 1, y = 1, x = 2
    w = [int(v) for v in orc.philox4x32_10(cellidx, 0, step, 0, seed & 0xFFFFFFFF, seed >> 32)]
    r1 = math.sqrt(-2.0 * math.log((w[0] + 1) / 2 ** 32)); th1 = 2 * math.pi * w[1] / 2 ** 32
    r2 = math.sqrt(-2.0 * math.log((w[2] + 1) / 2 ** 32)); th2 = 2 * math.pi * w[3] / 2 ** 32
    want = (r1 * math.cos(th1), r1 * math.sin(th1), r2 * math.cos(th2))
    assert np.allclose(eta[:, 1, 1, 2], want, rtol=1e-13, atol=1e-15)
