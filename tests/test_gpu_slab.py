"""Multi-GPU slab decomposition on ONE GPU: R contexts of one process stand for R ranks,
the two all-to-alls and the halo exchange are device-to-device copies of exactly the segments the NCCL transport
would send (paper_1102_3069_b200/dist.py).  Ranks run one after the other, phase by phase.  The gathered field
must match the oracle (north_star tolerance) and the single-context result."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_1102_3069_b200 import workloads as wlm        # noqa: E402
import mmtest_util as util                               # noqa: E402

TOL_H = 2e-5


def _slab_eval(wl, m, R, what, **kw):
    import torch
    from paper_1102_3069_b200 import dist as mmd
    ranks = [mmd.SlabRank(wl.grid, wl.cell, wl.pbc, wl.mat, r, R) for r in range(R)]
    ms = [util.to_dev(m[:, r.slab.z0:r.slab.z1]) for r in ranks]
    outs = mmd.evaluate_local(ranks, ms, what, **kw)
    full = torch.cat(outs, dim=1).double().cpu().numpy()
    for r in ranks:
        r.close()
    return full


@pytest.mark.parametrize("grid,R", [((64, 32, 64), 2), ((64, 32, 64), 3), ((128, 32, 32), 4)])
def test_slab_decomposition_matches_the_oracle(grid, R):
    wl = util.small(grid, (3e-9, 4e-9, 2e-9), (0, 0, 0), T=300.0, seed=77, j=(1e12, -5e11, 2e11), P=0.5, xi=0.04)
    m = wlm.initial_m(wl)
    m64 = m.astype(np.float64)
    pb = util.oracle_problem(wl)
    for what, ref in (("demag", pb.demag_field(m64)), ("heff", pb.heff(m64, 3, 5e-14)),
                      ("torque", pb.torque(m64, 3, 5e-14))):
        got = _slab_eval(wl, m, R, what, step=3, dt_thermal=5e-14)
        err = np.abs(got - ref).max()
        assert err <= TOL_H * np.abs(ref).max(), (what, err, np.abs(ref).max())


@pytest.mark.parametrize("pbc,R", [((0, 0, 1), 2), ((1, 0, 1), 3), ((0, 0, 0), 1)])
def test_slab_decomposition_matches_the_single_context_result(pbc, R):
    """Periodic z (the ring neighbours' planes are the halos) and one-rank degenerate case against mm_heff /
    mm_torque of an ordinary context: same kernels apart from the z pass variant, so agreement to fp32 rounding."""
    wl = util.small((64, 32, 64), (3e-9, 3e-9, 3e-9), pbc, T=300.0, seed=5, j=(2e11, 1e12, -7e11), P=0.5, xi=0.04)
    m = wlm.initial_m(wl)
    sim = util.gpu_sim(wl)
    md = util.to_dev(m)
    ref_h = sim.heff(md, step=2, dt_thermal=5e-14).double().cpu().numpy()
    ref_t = sim.torque(md, step=2, dt_thermal=5e-14).double().cpu().numpy()
    sim.close()
    got_h = _slab_eval(wl, m, R, "heff", step=2, dt_thermal=5e-14)
    got_t = _slab_eval(wl, m, R, "torque", step=2, dt_thermal=5e-14)
    assert np.abs(got_h - ref_h).max() <= 2e-6 * np.abs(ref_h).max()
    assert np.abs(got_t - ref_t).max() <= 2e-6 * np.abs(ref_t).max()


@pytest.mark.parametrize("method,R,T", [("rk4", 2, 0.0), ("rk4", 3, 300.0), ("rk2", 2, 0.0), ("rk1", 2, 300.0),
                                        ("rk3", 4, 0.0)])
def test_slab_time_stepping_follows_the_oracle_and_the_single_context(method, R, T):
    """Ten fixed steps on R slabs (stage by stage: forward, all-to-all, mid, all-to-all, halo planes of the STAGE
    state, backward with the a9 combine): the gathered state against the oracle's textbook stepper (north_star
    tolerance in m) and against mm_steps_fixed of one ordinary context (fp32 rounding of the z pass variant)."""
    import torch
    from oracle import mm_oracle as orc
    from paper_1102_3069_b200 import dist as mmd
    wl = util.small((64, 32, 64), (3e-9, 4e-9, 2e-9), (0, 0, 0), T=T, seed=21, j=(1e12, -5e11, 2e11), P=0.5, xi=0.04)
    m = wlm.initial_m(wl)
    dt, n = 5e-14, 10
    pb = util.oracle_problem(wl)
    mo = m.astype(np.float64)
    for s in range(n):
        mo = orc.rk_step(lambda x: pb.torque(x, s, dt), mo, dt, method)[0]
    sim = util.gpu_sim(wl)
    md = util.to_dev(m)
    sim.steps_fixed(md, method, dt, n)
    one = md.double().cpu().numpy()
    sim.close()
    ranks = [mmd.SlabRank(wl.grid, wl.cell, wl.pbc, wl.mat, r, R) for r in range(R)]
    ms = [util.to_dev(m[:, r.slab.z0:r.slab.z1]) for r in ranks]
    mmd.steps_fixed_local(ranks, ms, method, dt, n)
    got = torch.cat(ms, dim=1).double().cpu().numpy()
    for r in ranks:
        r.close()
    assert np.abs(got - mo).max() <= 1e-4, np.abs(got - mo).max()
    assert np.abs(got - one).max() <= 5e-6, np.abs(got - one).max()
    assert np.abs(np.sqrt((got * got).sum(0)) - 1.0).max() <= 1e-6


def test_slab_stepping_refuses_the_step_controlled_methods():
    import paper_1102_3069_b200 as mm
    from paper_1102_3069_b200 import dist as mmd
    wl = util.small((64, 32, 64), (3e-9, 3e-9, 3e-9))
    r = mmd.SlabRank(wl.grid, wl.cell, wl.pbc, wl.mat, 0, 2)
    m = util.to_dev(wlm.initial_m(wl)[:, r.slab.z0:r.slab.z1])
    for method, stage in (("rkdp", 0), ("rk23", 1), ("rk4", 4), ("rk2", -1)):
        with pytest.raises(mm.mm.MMError):
            r.stage_input(m, method, stage)
        with pytest.raises(mm.mm.MMError):
            r.backward_stage(m, method, stage, 1e-14, 0, None, None)
    r.close()


def test_slab_context_refuses_the_single_gpu_entry_points_and_bad_grids():
    import paper_1102_3069_b200 as mm
    from paper_1102_3069_b200 import dist as mmd
    wl = util.small((64, 32, 64), (3e-9, 3e-9, 3e-9))
    r = mmd.SlabRank(wl.grid, wl.cell, wl.pbc, wl.mat, 0, 2)
    st = r.L.mm_heff(r.ctx, None, None, 0.0, 0, 0.0)
    assert mm.mm.STATUS[st] == "MM_ESTATE"
    r.close()
    with pytest.raises(mm.mm.MMError):          # 24 -> padded 48: no size-specialised kernel for that length
        mmd.SlabRank((24, 32, 64), wl.cell, wl.pbc, wl.mat, 0, 2)
