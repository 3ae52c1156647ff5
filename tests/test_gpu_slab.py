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
