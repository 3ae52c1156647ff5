"""Batch of independent films in one context: every film must come out as
if it had a context of its own -- against the oracle per film, and against B separate contexts."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import mm_oracle as orc                      # noqa: E402
from paper_1102_3069_b200 import workloads as wlm        # noqa: E402
import mmtest_util as util                               # noqa: E402

TOL_H = 2e-5
TOL_M = 1e-4


def _films(wl, B):
    ms = []
    for b in range(B):
        w = wlm.scaled(wl, wl.grid)
        w.seed = 100 + b
        ms.append(wlm.initial_m(w)[:, 0])                 # (3, Ny, Nx)
    return np.ascontiguousarray(np.stack(ms, axis=1))      # (3, B, Ny, Nx)


@pytest.mark.parametrize("grid,pbc,B", [((64, 16, 1), (0, 0, 0), 5), ((32, 32, 1), (0, 0, 0), 3),
                                        ((64, 32, 1), (2, 2, 0), 4)])
def test_each_film_of_a_batch_matches_the_oracle_and_its_own_context(grid, pbc, B):
    import paper_1102_3069_b200 as mm
    wl = util.small(grid, (4e-9, 4e-9, 3e-9), pbc, init="tilted", alpha=0.1, j=(1e12, -5e11, 0.0), P=0.5, xi=0.04)
    m = _films(wl, B)
    Bs = np.array([[0.01 * b, -0.02 + 0.005 * b, 0.003 * b] for b in range(B)])
    sim = mm.Sim(wl.grid, wl.cell, wl.pbc, wl.mat, nfilms=B)
    sim.batch_set_field(Bs)
    md = util.to_dev(m)
    H = sim.heff(md).double().cpu().numpy()
    T = sim.torque(md).double().cpu().numpy()
    dt, n = 5e-14, 20
    sim.steps_fixed(md, "rk4", dt, n)
    mb = md.double().cpu().numpy()
    sim.close()
    for b in range(B):
        wb = wlm.scaled(wl, wl.grid)
        wb.mat = dict(wl.mat, Bext=tuple(Bs[b]))
        pb = util.oracle_problem(wb)
        m64 = m[:, b:b + 1].astype(np.float64)
        Href, Tref = pb.heff(m64), pb.torque(m64)
        assert np.abs(H[:, b:b + 1] - Href).max() <= TOL_H * np.abs(Href).max()
        assert np.abs(T[:, b:b + 1] - Tref).max() <= TOL_H * np.abs(Tref).max()
        one = util.gpu_sim(wb)                              # the same film in a context of its own
        m1 = util.to_dev(m[:, b:b + 1])
        one.steps_fixed(m1, "rk4", dt, n)
        assert np.abs(m1.double().cpu().numpy() - mb[:, b:b + 1]).max() <= 2e-6
        one.close()
        if b == 0:
            mo = m64
            for _ in range(n):
                mo = orc.rk4_step(pb.torque, mo, dt)
            assert np.abs(mb[:, b:b + 1] - mo).max() <= TOL_M


def test_batch_refuses_what_it_cannot_run():
    import paper_1102_3069_b200 as mm
    wl = util.small((64, 16, 1), (4e-9, 4e-9, 3e-9))
    with pytest.raises(mm.mm.MMError):
        mm.Sim((64, 16, 2), wl.cell, wl.pbc, wl.mat, nfilms=3)          # members must be films
    with pytest.raises(mm.mm.MMError):
        mm.Sim((24, 16, 1), wl.cell, wl.pbc, wl.mat, nfilms=3)          # padded 48: no size-specialised kernel
    sim = mm.Sim(wl.grid, wl.cell, wl.pbc, wl.mat, nfilms=3)
    with pytest.raises(mm.mm.MMError):
        sim.set_fast_path(0)
    sim.close()
