"""Pins for the oracle's demagnetisation tensor (oracle/demag_tensor.c).

The paper gives only Eq. (2) and states that the kernel matrices are
"completely symmetrical"; reading A1 fixes the closed
form.  None of these checks re-types that closed form: they use what the
mathematics fixes (self terms of a cube, trace, parity, the point-dipole limit,
the coarse-graining identity, a direct numerical quadrature of Eq. (2)).
"""
import itertools

import numpy as np
import pytest

from oracle import mm_oracle as orc


def test_cube_self_terms_are_one_third():
    # BASELINE.json invariant: "Newell tensor self-terms of a cube equal 1/3 each"
    n = orc.tensor_at([[0, 0, 0]], (1.0, 1.0, 1.0))[0]
    assert np.allclose(n[:3], 1.0 / 3.0, rtol=0, atol=1e-15)
    assert np.allclose(n[3:], 0.0, atol=1e-30)
    n = orc.tensor_at([[0, 0, 0]], (5e-9, 5e-9, 5e-9))[0]
    assert np.allclose(n[:3], 1.0 / 3.0, rtol=0, atol=1e-15)


@pytest.mark.parametrize("cell", [(1, 1, 1), (4, 4, 2), (3.90625, 3.90625, 4), (1, 2, 5),
                                  (3e-9, 3e-9, 3e-9)])
def test_trace_is_one_at_origin_and_zero_elsewhere(cell):
    # trace N(0) = 1 (BASELINE.json invariant); div H = -div M => trace N(R != 0) = 0
    n0 = orc.tensor_at([[0, 0, 0]], cell)[0]
    assert abs(n0[:3].sum() - 1.0) < 1e-15
    offs = [(1, 0, 0), (0, 1, 0), (0, 0, 1), (1, 1, 0), (1, 1, 1), (2, -3, 1), (7, 5, -3),
            (40, 25, -13), (300, 200, 31), (1000, 700, 63)]
    n = orc.tensor_at(offs, cell)
    scale = np.abs(n[:, :3]).max(axis=1)
    assert np.all(np.abs(n[:, :3].sum(axis=1)) <= 1e-14 * scale + 1e-30)


def test_parity_of_components():
    # N_xx even in X,Y,Z; N_xy odd in X and Y, even in Z; cyclic for xz, yz
    cell = (1.0, 2.0, 0.5)
    base = np.array([3, 2, 5])
    ref = orc.tensor_at([base], cell)[0]
    for sx, sy, sz in itertools.product((1, -1), repeat=3):
        n = orc.tensor_at([base * np.array([sx, sy, sz])], cell)[0]
        expect = ref * np.array([1, 1, 1, sx * sy, sx * sz, sy * sz])
        assert np.allclose(n, expect, rtol=1e-14, atol=0)
    # components vanish on their odd planes
    n = orc.tensor_at([[0, 4, 3], [4, 0, 3], [4, 3, 0]], cell)
    assert n[0, 3] == 0 and n[0, 4] == 0
    assert n[1, 3] == 0 and n[1, 5] == 0
    assert n[2, 4] == 0 and n[2, 5] == 0


def _dipole(R, V):
    R = np.asarray(R, dtype=np.float64)
    r = np.linalg.norm(R)
    T = (np.eye(3) / r ** 3 - 3.0 * np.outer(R, R) / r ** 5) * V / (4.0 * np.pi)
    return np.array([T[0, 0], T[1, 1], T[2, 2], T[0, 1], T[0, 2], T[1, 2]])


def test_far_field_is_point_dipole():
    # H of a point dipole: H = (1/4pi)(3 R (R.mu)/R^5 - mu/R^3), mu = M V  =>  N -> V/(4pi)(I/R^3 - 3RR/R^5)
    for off, tol in (((40, 25, -13), 1e-6), ((100, -60, 13), 3e-8), ((1000, 700, 63), 1e-9)):
        n = orc.tensor_at([off], (1, 1, 1))[0]
        d = _dipole(off, 1.0)
        assert np.allclose(n, d, rtol=tol, atol=tol * np.abs(d).max())
    # non-cubic cell, physical units
    cell = np.array([4e-9, 4e-9, 2e-9])
    off = np.array([60, -45, 80])
    n = orc.tensor_at([off], cell)[0]
    d = _dipole(off * cell, cell.prod())
    assert np.allclose(n, d, rtol=0, atol=2e-4 * np.abs(d).max())


def test_coarse_graining_identity():
    """The tensor between two block cells equals the average over all pairs of their
    fine cells (linearity of Eq. (2)): checks f and g at many offsets at once."""
    fine = (1.0, 1.0, 1.0)
    for blk, boff in (((2, 1, 1), (0, 0, 0)), ((2, 2, 1), (1, 1, 0)), ((1, 2, 3), (2, -1, 1)),
                      ((3, 2, 2), (0, 1, 0))):
        big = orc.tensor_at([boff], tuple(float(b) for b in blk))[0]
        cells = list(itertools.product(range(blk[0]), range(blk[1]), range(blk[2])))
        acc = np.zeros(6)
        for a in cells:
            for b in cells:
                d = [boff[i] * blk[i] + a[i] - b[i] for i in range(3)]
                acc += orc.tensor_at([d], fine)[0]
        acc /= len(cells)
        assert np.allclose(big, acc, rtol=1e-13, atol=1e-15), (blk, boff)


def test_against_numerical_quadrature_of_eq2():
    """Eq. (2) for two separated cells: N_ij = (1/V) int_cell int_cell' T_ij(r - r') with the
    point kernel T = (1/4pi)(delta_ij/R^3 - 3 R_i R_j/R^5).  6-fold Gauss-Legendre quadrature."""
    cell = np.array([1.0, 1.5, 0.75])
    x, w = np.polynomial.legendre.leggauss(8)
    x = 0.5 * x
    w = 0.5 * w                                     # nodes / weights on [-1/2, 1/2]
    # difference of two uniform variables on [-1/2,1/2]: integrate pairwise
    U = (x[:, None] - x[None, :]).ravel()
    Wt = (w[:, None] * w[None, :]).ravel()
    for off in ((3, -2, 1), (2, 0, 0), (0, 2, -2), (2, 2, 3)):
        Rx = (off[0] + U) * cell[0]
        Ry = (off[1] + U) * cell[1]
        Rz = (off[2] + U) * cell[2]
        X, Y, Z = np.meshgrid(Rx, Ry, Rz, indexing="ij")
        W3 = Wt[:, None, None] * Wt[None, :, None] * Wt[None, None, :]
        r2 = X * X + Y * Y + Z * Z
        r5 = r2 ** 2.5
        V = cell.prod()
        q = []
        for (A, B, diag) in ((X, X, True), (Y, Y, True), (Z, Z, True), (X, Y, False),
                             (X, Z, False), (Y, Z, False)):
            T = ((r2 if diag else 0.0) - 3.0 * A * B) / r5 / (4.0 * np.pi)
            q.append(np.sum(W3 * T) * V)
        n = orc.tensor_at([off], cell)[0]
        assert np.allclose(n, q, rtol=0, atol=2e-8 * np.abs(n).max()), off


def test_octant_table_equals_pointwise_evaluation():
    cell = (3.90625, 3.90625, 4.0)
    n = (7, 5, 3)
    o = orc.tensor_octant(n, cell)
    offs = [(i, j, k) for k in range(n[2]) for j in range(n[1]) for i in range(n[0])]
    p = orc.tensor_at(offs, cell).T.reshape(6, n[2], n[1], n[0])
    assert np.allclose(o, p, rtol=1e-15, atol=1e-30)


def test_float128_beats_fp64_cancellation():
    # reading A1: at 1000 cells the 27-point sum cancels ~ 25 digits; the result must still
    # match the dipole limit to 1e-9 relative (test_far_field) -- here: the value is finite,
    # non-zero and of dipole magnitude, which plain fp64 evaluation does not deliver.
    n = orc.tensor_at([(1000, 700, 63)], (1, 1, 1))[0]
    d = _dipole((1000, 700, 63), 1.0)
    assert np.all(np.abs(n - d) < 1e-8 * np.abs(d).max())


def test_thin_film_limit_nzz_tends_to_one():
    # BASELINE.json invariant: "The thin-film N_zz limit tends to 1": sum of N_zz over an
    # L x L x 1 film of cubes seen from the centre cell grows towards 1 with L
    prev = 0.0
    for L in (9, 17, 33):
        h = L // 2
        offs = [(i, j, 0) for i in range(-h, h + 1) for j in range(-h, h + 1)]
        s = orc.tensor_at(offs, (1, 1, 1))[:, 2].sum()
        assert prev < s < 1.0
        prev = s
    assert s > 0.97
    # and the self term of a very flat cell
    n = orc.tensor_at([[0, 0, 0]], (1000.0, 1000.0, 1.0))[0]
    assert n[2] > 0.995 and n[0] < 0.0025


def _golden_rows():
    import os
    rows = []
    with open(os.path.join(os.path.dirname(__file__), "golden", "tensor_near_field_survey.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            w = line.split()
            rows.append((w[0], tuple(float(v) for v in w[1:4]), tuple(int(v) for v in w[4:7]),
                         [None if v == "-" else float(v) for v in w[7:13]]))
    return rows


def test_printed_near_field_and_self_term_values():
    """SURVEY.md:443-444 pins P5 (near field of unit cubes) and P6 (self terms of the configs' cells),
    "[survey-computed]" there, stored in tests/golden/tensor_near_field_survey.txt.  The values are
    printed to 12-15 digits; a wrong sign, a swapped component or a dropped term of f or g fails here."""
    rows = _golden_rows()
    assert sum(r[0] == "P5" for r in rows) == 5 and sum(r[0] == "P6" for r in rows) == 3
    for kind, cell, off, want in rows:
        got = orc.tensor_at([list(off)], cell)[0]
        for c in range(6):
            if want[c] is None:
                assert abs(got[c]) <= 1e-15          # off-diagonal self terms vanish by symmetry
            else:
                assert abs(got[c] - want[c]) <= 2e-12, (kind, cell, off, c)   # printed to >= 12 digits
