"""GPU parity: the CUDA path (through the C-ABI) against the fp64 oracle, element by element.

Tolerances (BASELINE.json north_star): per H_eff evaluation 2e-5 of max|H| (fp32 against fp64); after
100 fixed-step RK4 steps 1e-4 in m.  Reading A12: the magnetostatic field is also checked on its own
scale so that a demag error cannot hide under the exchange field.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import mm_oracle as orc                      # noqa: E402
from paper_1102_3069_b200 import workloads as wlm        # noqa: E402
import mmtest_util as util                               # noqa: E402

TOL_H = 2e-5
TOL_M = 1e-4

GRIDS = [
    # grid, cell, pbc                       what it exercises
    ((32, 32, 1), (4e-9, 4e-9, 4e-9), (0, 0, 0)),        # config 1 shape
    ((24, 10, 6), (3e-9, 4e-9, 5e-9), (0, 0, 0)),        # radix 3 and 5 (48, 20, 12)
    ((15, 9, 5), (3e-9, 3e-9, 3e-9), (0, 0, 0)),         # odd sizes, ragged pair tail (30, 18, 10)
    ((40, 6, 3), (2e-9, 2e-9, 4e-9), (0, 0, 0)),         # 80 = 16 * 5
    ((16, 12, 1), (4e-9, 4e-9, 2e-9), (2, 2, 0)),        # periodic film, no padding in x, y
    ((8, 6, 4), (4e-9, 3e-9, 2e-9), (0, 1, 2)),          # mixed periodic / open 3D
    ((16, 1, 1), (2e-9, 3e-9, 4e-9), (0, 0, 0)),         # 1D chain: multiply without y / z pass
    ((1, 1, 1), (5e-9, 5e-9, 5e-9), (0, 0, 0)),          # macrospin
    ((1, 8, 2), (5e-9, 4e-9, 3e-9), (0, 0, 0)),          # one cell along x
    ((64, 48, 2), (3e-9, 3e-9, 3e-9), (0, 0, 0)),        # several tiles per pass
    ((28, 14, 7), (3e-9, 4e-9, 5e-9), (0, 0, 0)),        # radix 7 (56, 28, 14)
    ((49, 7, 1), (3e-9, 3e-9, 3e-9), (1, 1, 0)),         # 49 = 7 * 7 periodic, no padding
]


def _cmp(a_gpu, b_ref, tol, scale=None):
    a = a_gpu.double().cpu().numpy()
    s = np.abs(b_ref).max() if scale is None else scale
    err = np.abs(a - b_ref).max()
    assert err <= tol * s, f"max err {err:.3e} > {tol:.1e} * {s:.3e}"
    return err / s if s > 0 else 0.0


@pytest.mark.parametrize("fast", [False, True])
@pytest.mark.parametrize("grid,cell,pbc", GRIDS)
def test_demag_field_matches_direct_pair_sum(grid, cell, pbc, fast):
    wl = util.small(grid, cell, pbc)
    m = wlm.initial_m(wl)
    sim = util.gpu_sim(wl, fast=fast)
    H = sim.demag_field(util.to_dev(m))
    ncell = grid[0] * grid[1] * grid[2]
    if ncell <= 2048:
        ref = orc.demag_field_direct(m.astype(np.float64), wl.mat["Ms"], grid, cell, pbc)
    else:
        ref = util.oracle_problem(wl).demag_field(m.astype(np.float64))
    _cmp(H, ref, TOL_H, scale=max(np.abs(ref).max(), 1e-3 * wl.mat["Ms"]))
    sim.close()


@pytest.mark.parametrize("fast", [False, True])
@pytest.mark.parametrize("grid,cell,pbc", GRIDS)
def test_heff_and_torque_match_oracle(grid, cell, pbc, fast):
    wl = util.small(grid, cell, pbc, T=300.0, seed=12345678901234, j=(1e12, -5e11, 2e11), P=0.5, xi=0.04)
    m = wlm.initial_m(wl)
    pb = util.oracle_problem(wl)
    sim = util.gpu_sim(wl, fast=fast)
    md = util.to_dev(m)
    m64 = m.astype(np.float64)
    step, dt = (1 << 33) + 5, 5e-14
    Href = pb.heff(m64, step, dt)
    _cmp(sim.heff(md, step=step, dt_thermal=dt), Href, TOL_H)
    Tref = pb.torque(m64, step, dt)
    _cmp(sim.torque(md, step=step, dt_thermal=dt), Tref, TOL_H)
    # without the thermal field (which dominates the scale at these cell sizes)
    wl2 = util.small(grid, cell, pbc, j=(1e12, -5e11, 2e11), P=0.5, xi=0.04)
    pb2 = util.oracle_problem(wl2)
    sim.set_material(wl2.mat)
    _cmp(sim.heff(md), pb2.heff(m64), TOL_H)
    _cmp(sim.torque(md), pb2.torque(m64), TOL_H)
    sim.close()


def test_local_terms_alone_demag_off():
    wl = util.small((24, 10, 6), Aex=1.3e-11)
    m = wlm.initial_m(wl)
    pb = util.oracle_problem(wl, demag="none")
    sim = util.gpu_sim(wl, demag=False)
    _cmp(sim.heff(util.to_dev(m)), pb.heff(m.astype(np.float64)), 2e-6)
    sim.close()


def test_config1_heff_then_100_rk4_steps():
    """BASELINE.json configs[0]: 32x32x1, one H_eff against the direct O(N^2) sum, then 100 RK4 steps."""
    wl = wlm.config(0)
    m = wlm.initial_m(wl)
    m64 = m.astype(np.float64)
    sim = util.gpu_sim(wl)
    md = util.to_dev(m)
    pb1 = util.oracle_problem(wl, demag="direct")
    _cmp(sim.heff(md), pb1.heff(m64), TOL_H)
    pb = util.oracle_problem(wl)
    mo = m64.copy()
    for _ in range(wl.steps):
        mo = orc.rk4_step(pb.torque, mo, wl.dt)
    t, _ = sim.steps_fixed(md, "rk4", wl.dt, wl.steps)
    assert abs(t - wl.steps * wl.dt) < 1e-20
    err = np.abs(md.double().cpu().numpy() - mo).max()
    assert err <= TOL_M, err
    # same through mm_step, one call per step
    md2 = util.to_dev(m)
    sim.reset_stepper(0)
    for _ in range(wl.steps):
        acc, _, dtn, _ = sim.step(md2, "rk4", wl.dt)
        assert acc and dtn == wl.dt
    assert np.abs(md2.double().cpu().numpy() - mo).max() <= TOL_M
    sim.close()


@pytest.mark.parametrize("grid,cell,pbc", [((24, 10, 6), (3e-9, 4e-9, 5e-9), (0, 0, 0)),
                                           ((16, 12, 1), (4e-9, 4e-9, 2e-9), (2, 2, 0))])
def test_rk4_with_thermal_and_stt_trajectory(grid, cell, pbc):
    wl = util.small(grid, cell, pbc, init="xnoise", alpha=0.1, T=300.0, seed=3, j=(1e12, 0, 0), P=0.5,
                    xi=0.04)
    m = wlm.initial_m(wl)
    pb = util.oracle_problem(wl)
    dt, n = 5e-14, 10
    mo = m.astype(np.float64)
    for s in range(n):
        mo = orc.rk4_step(lambda x: pb.torque(x, s, dt), mo, dt)
    sim = util.gpu_sim(wl)
    md = util.to_dev(m)
    sim.steps_fixed(md, "rk4", dt, n)
    assert np.abs(md.double().cpu().numpy() - mo).max() <= TOL_M
    sim.close()


def test_rk1_steps():
    wl = util.small((15, 9, 5), alpha=0.5)
    m = wlm.initial_m(wl)
    pb = util.oracle_problem(wl)
    mo = m.astype(np.float64)
    for _ in range(20):
        mo = orc.rk1_step(pb.torque, mo, 2e-14)
    sim = util.gpu_sim(wl)
    md = util.to_dev(m)
    sim.steps_fixed(md, "rk1", 2e-14, 20)
    assert np.abs(md.double().cpu().numpy() - mo).max() <= TOL_M
    sim.close()


def test_rkdp_replay_of_oracle_step_sequence_and_free_run():
    """Reading A10: adaptive runs are compared by replaying the oracle's accepted dt sequence."""
    wl = util.small((24, 10, 6), init="tilted", alpha=0.02, Bext=(-0.0246, 0.0043, 0.0), Ku=0.0)
    m = wlm.initial_m(wl)
    pb = util.oracle_problem(wl)
    tol, dt = 1e-5, 1e-13
    mo = m.astype(np.float64)
    k1, seq, errs, trials = None, [], [], 0
    while len(seq) < 30:
        mn, err, k7 = orc.rkdp_step(pb.torque, mo, dt, k1)
        ok, dtn = orc.rkdp_controller(dt, err, tol)
        trials += 1
        if ok:
            seq.append(dt); errs.append(err); mo, k1 = mn, k7
        dt = dtn
    sim = util.gpu_sim(wl)
    md = util.to_dev(m)
    for d, e in zip(seq, errs):
        _, ge = sim.steps_fixed(md, "rkdp", d, 1)
        assert abs(ge - e) <= 0.02 * e + 1e-9, (ge, e)
    assert np.abs(md.double().cpu().numpy() - mo).max() <= TOL_M
    # free run with the library's own controller: same number of trials, same end time (to a few %)
    md = util.to_dev(m)
    sim.reset_stepper(0)
    dt, t, nacc, ntr = 1e-13, 0.0, 0, 0
    while nacc < 30:
        acc, err, dt, t = sim.step(md, "rkdp", dt, tol, t)
        ntr += 1
        nacc += int(acc)
    assert abs(ntr - trials) <= 2
    assert abs(t - sum(seq)) <= 0.05 * sum(seq)
    assert np.abs(md.double().cpu().numpy() - mo).max() <= 1e-3
    sim.close()


def test_thermal_with_adaptive_method_is_refused():
    import paper_1102_3069_b200 as mm
    wl = util.small((8, 6, 4), T=300.0)
    sim = util.gpu_sim(wl)
    md = util.to_dev(wlm.initial_m(wl))
    with pytest.raises(mm.MMError) as e:
        sim.step(md, "rkdp", 1e-13)
    assert e.value.status == 5
    sim.close()


def test_call_order_and_nan_are_reported():
    import paper_1102_3069_b200 as mm
    wl = util.small((8, 6, 4))
    sim = mm.Sim(wl.grid, wl.cell, wl.pbc, None, demag_init=False)
    md = util.to_dev(wlm.initial_m(wl))
    with pytest.raises(mm.MMError) as e:
        sim.heff(md)
    assert e.value.status == 4
    sim.set_material(wl.mat)
    with pytest.raises(mm.MMError) as e:
        sim.heff(md)
    assert e.value.status == 4
    sim.demag_init()
    sim.heff(md)
    md[0, 1, 2, 3] = float("nan")
    with pytest.raises(mm.MMError) as e:
        sim.step(md, "rk4", 1e-13)
    assert e.value.status == 6
    sim.close()


def test_uniform_state_mean_field_is_sample_demag_factor():
    """Pin P7 on the GPU alone: mean of H_a/Ms over a uniformly magnetised sample = -N_aa of one cell
    the size of the sample (coarse-graining identity); the latter comes from the oracle tensor."""
    grid, cell = (32, 32, 1), (4e-9, 4e-9, 4e-9)
    for a in range(3):
        d = [0.0, 0.0, 0.0]; d[a] = 1.0
        wl = wlm.Workload("u", grid, cell, (0, 0, 0), wlm._mat(), "uniform", 0, extra={"dir": d})
        sim = util.gpu_sim(wl)
        H = sim.demag_field(util.to_dev(wlm.initial_m(wl))).double().cpu().numpy()
        big = orc.tensor_at([[0, 0, 0]], tuple(c * n for c, n in zip(cell, grid)))[0]
        assert abs(H[a].mean() / wl.mat["Ms"] + big[a]) <= 2e-6
        sim.close()


def test_reciprocity_and_positive_energy_on_gpu():
    """Pin P18: sum m1.H[m2] = sum m2.H[m1]; demag energy >= 0."""
    wl = util.small((64, 48, 2), (3e-9, 3e-9, 3e-9))
    sim = util.gpu_sim(wl)
    m1 = util.to_dev(wlm.initial_m(wl))
    wl.seed = 99
    m2 = util.to_dev(wlm.initial_m(wl))
    H1 = sim.demag_field(m1).double()
    H2 = sim.demag_field(m2).double()
    a = float((m1.double() * H2).sum()); b = float((m2.double() * H1).sum())
    assert abs(a - b) <= 1e-5 * max(abs(a), abs(b))
    assert float((m1.double() * H1).sum()) < 0.0
    sim.close()


# ---- size-specialised register FFT passes (fft_fast*.cuh): padded lengths 64..1024 ----
FAST_GRIDS = [
    # grid, cell, pbc                                     padded          passes with a fast kernel
    ((32, 32, 32), (3e-9, 3e-9, 3e-9), (0, 0, 0)),      # 64^3            all
    ((64, 32, 64), (3e-9, 4e-9, 2e-9), (0, 0, 0)),      # 128 x 64 x 128  all
    ((128, 64, 6), (3e-9, 3e-9, 3e-9), (0, 0, 0)),      # 256 x 128 x 12  x, y fast; z generic
    ((256, 64, 1), (3.90625e-9, 3.90625e-9, 4e-9), (0, 0, 0)),   # config 2 shape: 512 x 128, 2D
    ((512, 45, 3), (3e-9, 3e-9, 3e-9), (0, 0, 0)),      # 1024 along x, odd Ny (ragged pair), generic y/z
    ((16, 512, 1), (3e-9, 3e-9, 3e-9), (0, 0, 0)),      # 1024 along y, 2D
    ((64, 128, 1), (4e-9, 4e-9, 2e-9), (2, 2, 0)),      # periodic film: no padding in x, y
    ((64, 32, 64), (3e-9, 3e-9, 3e-9), (1, 0, 1)),      # periodic x, z; open y
    ((36, 32, 128), (3e-9, 3e-9, 3e-9), (0, 0, 0)),     # x generic (72), y 64, z 256; ragged kx tiles
    ((192, 96, 32), (3e-9, 3e-9, 3e-9), (0, 0, 0)),     # one factor 3: 384 x 192 x 64, all fast
    ((384, 192, 4), (3e-9, 4e-9, 5e-9), (0, 0, 0)),     # 768 x 384 x 8 (z generic)
    ((384, 192, 1), (4e-9, 4e-9, 2e-9), (1, 1, 0)),     # periodic film 384 x 192, 2D
    ((768, 24, 2), (3e-9, 3e-9, 3e-9), (0, 0, 0)),      # x = 1536 through the half-length real transform
    ((1024, 16, 2), (3e-9, 3e-9, 3e-9), (0, 0, 0)),     # x = 2048, same
    ((1536, 8, 1), (3e-9, 3e-9, 3e-9), (1, 0, 0)),      # x = 1536 periodic (no padding)
    ((32, 40, 128), (3e-9, 3e-9, 3e-9), (0, 0, 1)),     # periodic z of length 128 (no padding), ragged kx tile
    ((16, 16, 8), (3e-9, 3e-9, 3e-9), (0, 0, 0)),       # 32 x 32 x 16: the shortest size-specialised lines (x, y)
    ((64, 16, 1), (4e-9, 4e-9, 3e-9), (0, 0, 0)),       # film 128 x 32 (the batch-of-films shape)
    ((16, 1024, 1), (3e-9, 3e-9, 3e-9), (0, 0, 0)),     # y = 2048: two interleaved 1024-point transforms + combine
    ((8, 2048, 1), (3e-9, 3e-9, 3e-9), (0, 0, 0)),      # y = 4096: four
    ((16, 2048, 1), (3e-9, 3e-9, 3e-9), (0, 1, 0)),     # y = 2048 periodic (no padding)
    ((32, 1024, 2), (3e-9, 3e-9, 3e-9), (0, 0, 0)),     # y = 2048 in a 3D grid (z generic), ragged kx tile
    ((2048, 8, 1), (3e-9, 3e-9, 3e-9), (0, 0, 0)),      # x = 4096: even / odd samples through the 2048-point real transform
    ((4096, 4, 1), (3e-9, 3e-9, 3e-9), (1, 0, 0)),      # x = 4096 periodic (no padding)
    ((2048, 6, 2), (3e-9, 3e-9, 3e-9), (0, 0, 0)),      # x = 4096 in a 3D grid
    ((32, 16, 256), (3e-9, 3e-9, 3e-9), (0, 0, 0)),     # z = 512: unfused z pass through the z-padded buffer
    ((16, 20, 192), (3e-9, 3e-9, 3e-9), (0, 0, 0)),     # z = 384 (one factor 3), y generic (40)
    ((32, 16, 512), (3e-9, 3e-9, 3e-9), (0, 0, 1)),     # z = 512 periodic (no padding)
    # lengths 2^n * {5, 7, 9} and 3 * 2^n beyond the kernels' own: R interleaved transforms + combine
    ((16, 960, 1), (3e-9, 3e-9, 3e-9), (0, 0, 0)),      # y = 1920 = 5 * 384
    ((16, 448, 1), (3e-9, 3e-9, 3e-9), (0, 0, 0)),      # y = 896 = 7 * 128
    ((16, 576, 2), (3e-9, 3e-9, 3e-9), (0, 0, 0)),      # y = 1152 = 9 * 128, 3D
    ((960, 16, 1), (3e-9, 3e-9, 3e-9), (0, 0, 0)),      # x = 1920 = 5 * 384 (pair-packed sub-rows)
    ((448, 8, 1), (3e-9, 3e-9, 3e-9), (0, 0, 0)),       # x = 896 = 7 * 128
    ((640, 8, 1), (3e-9, 3e-9, 3e-9), (1, 0, 0)),       # x = 640 = 5 * 128 periodic
    ((1536, 8, 1), (3e-9, 3e-9, 3e-9), (0, 0, 0)),      # x = 3072 = 2 * 1536 (half-length sub-transform)
    ((16, 16, 80), (3e-9, 3e-9, 3e-9), (0, 0, 0)),      # z = 160 = 5 * 32, unfused z pass
    ((320, 160, 1), (3e-9, 3e-9, 3e-9), (0, 0, 0)),     # 640 x 320 = 5 * 128, 5 * 64: both axes split
]


# (x lines of 4096 have no generic counterpart -- the line does not fit its shared-memory tile -- and meet the oracle only)
@pytest.mark.parametrize("grid,cell,pbc", [g for g in FAST_GRIDS if g[0][0] * (1 if g[2][0] else 2) < 4096])
def test_fast_passes_match_generic_pass_by_pass(grid, cell, pbc):
    """Both kernel families use the same layouts: switch the fast kernels on one pass at a time."""
    wl = util.small(grid, cell, pbc, j=(1e12, -5e11, 2e11), P=0.5, xi=0.04)
    m = wlm.initial_m(wl)
    sim = util.gpu_sim(wl, fast=0)
    md = util.to_dev(m)
    Hg = sim.demag_field(md).double()
    Tg = sim.torque(md).double()
    sH, sT = float(Hg.abs().max()), float(Tg.abs().max())
    for mask in (1, 2, 4, 8, 16, 15, 31, 63):
        sim.set_fast_path(mask)
        eh = float((sim.demag_field(md).double() - Hg).abs().max()) / sH
        et = float((sim.torque(md).double() - Tg).abs().max()) / sT
        assert eh <= 2e-6 and et <= 2e-6, (mask, eh, et)
    sim.close()


# Every size-specialised kernel family meets the oracle itself (not only the generic kernels): all of FAST_GRIDS
# except the two 3D grids with a periodic axis, whose float128 image sums take up to a minute each -- those are in
# tests/test_gpu_configs.py::test_periodic_3d_fast_grids_against_the_oracle (MM_SLOW=1).
@pytest.mark.parametrize("grid,cell,pbc", [g for g in FAST_GRIDS if not (g[0][2] > 1 and any(g[2]))])
def test_fast_path_matches_oracle(grid, cell, pbc):
    wl = util.small(grid, cell, pbc, T=300.0, seed=77, j=(1e12, -5e11, 2e11), P=0.5, xi=0.04)
    m = wlm.initial_m(wl)
    m64 = m.astype(np.float64)
    pb = util.oracle_problem(wl)
    sim = util.gpu_sim(wl)
    md = util.to_dev(m)
    ref = pb.demag_field(m64)
    _cmp(sim.demag_field(md), ref, TOL_H)
    _cmp(sim.heff(md, step=3, dt_thermal=5e-14), pb.heff(m64, 3, 5e-14), TOL_H)
    _cmp(sim.torque(md, step=3, dt_thermal=5e-14), pb.torque(m64, 3, 5e-14), TOL_H)
    sim.close()


def test_fast_path_rk4_and_rkdp_steps_match_generic():
    wl = util.small((64, 32, 64), (3e-9, 3e-9, 3e-9), init="xnoise", alpha=0.1)
    m = wlm.initial_m(wl)
    out = {}
    for fast in (0, 15, 31):
        sim = util.gpu_sim(wl, fast=fast)
        md = util.to_dev(m)
        sim.steps_fixed(md, "rk4", 5e-14, 5)
        _, err = sim.steps_fixed(md, "rkdp", 5e-14, 3)
        out[fast] = (md.double().cpu().numpy(), err)
        sim.close()
    for f in (15, 31):
        assert np.abs(out[0][0] - out[f][0]).max() <= 1e-5
        assert abs(out[0][1] - out[f][1]) <= 0.02 * out[0][1] + 1e-9


@pytest.mark.parametrize("grid,pbc", [((64, 32, 64), (0, 0, 0)), ((128, 32, 32), (0, 0, 1))])
def test_chunked_l2_resident_passes_match_whole_array_passes(grid, pbc):
    """a2-a4 in kx chunks through a compact buffer (several streams) against the whole-array passes."""
    wl = util.small(grid, (3e-9, 3e-9, 3e-9), pbc)
    m = wlm.initial_m(wl)
    # mid_pipe = 1: the whole-array z pass runs the same cp.async kernel as the chunks (the TMA / packed kernel
    # orders its additions differently), so that the comparison is bit for bit
    sim = util.gpu_sim(wl, fast=31, options={"chunk_w": 16, "chunk_streams": 3, "mid_pipe": 1})
    md = util.to_dev(m)
    H0 = sim.demag_field(md).double()
    T0 = sim.torque(md).double()
    sim.set_fast_path(63)
    for _ in range(3):
        H1 = sim.demag_field(md).double()
        T1 = sim.torque(md).double()
        assert float((H1 - H0).abs().max()) == 0.0
        assert float((T1 - T0).abs().max()) == 0.0
    if tuple(pbc) == (0, 0, 0):              # (the periodic oracle tensor in float128 takes minutes)
        ref = util.oracle_problem(wl).demag_field(m.astype(np.float64))
        _cmp(H1.float(), ref, TOL_H)
    sim.close()


@pytest.mark.parametrize("grid,pbc", [((64, 32, 64), (0, 0, 0)), ((200, 48, 64), (0, 0, 0)), ((64, 64, 128), (0, 1, 1))])
def test_panel_layout_of_the_spectrum_changes_no_bit(grid, pbc):
    """Option spec_panel: the y-transformed spectrum in 16-column panels (a2, a3, a4 with pk::k_mid_t as the z pass)
    against plain rows -- same arithmetic, another address map: bit for bit, also with a ragged last panel."""
    wl = util.small(grid, (3e-9, 4e-9, 2e-9), pbc, j=(1e12, -5e11, 2e11), P=0.5, xi=0.04)
    md = util.to_dev(wlm.initial_m(wl))
    out = {}
    for flag in (1, 0):
        sim = util.gpu_sim(wl, options={"spec_panel": flag})
        out[flag] = (sim.demag_field(md).clone(), sim.torque(md).clone())
        sim.close()
    assert float((out[0][0] - out[1][0]).abs().max()) == 0.0
    assert float((out[0][1] - out[1][1]).abs().max()) == 0.0
    assert float(out[1][0].abs().max()) > 0.0


@pytest.mark.parametrize("grid,pbc", [((64, 512, 64), (0, 0, 0)), ((36, 512, 64), (0, 0, 0)), ((64, 1024, 64), (0, 1, 0))])
def test_tma_tile_loads_of_the_y_passes_change_no_bit(grid, pbc):
    """Option y_tma: the y-pass tiles of 1024-long lines arrive by cp.async.bulk.tensor instead of cp.async (1), and
    leave through a staging tile and TMA tile stores in the forward pass (2) or in both (3); whole-array passes in
    the panel form; 36 columns: a ragged last tile whose missing columns the tensor map fills with zeros / clips."""
    wl = util.small(grid, (3e-9, 4e-9, 5e-9), pbc, seed=3)
    md = util.to_dev(wlm.initial_m(wl))
    out = {}
    for flag in (0, 1, 2, 3):
        sim = util.gpu_sim(wl, options={"y_tma": flag})
        out[flag] = (sim.demag_field(md).clone(), sim.torque(md).clone())
        sim.close()
    for flag in (1, 2, 3):
        assert float((out[0][0] - out[flag][0]).abs().max()) == 0.0
        assert float((out[0][1] - out[flag][1]).abs().max()) == 0.0
    assert float(out[2][0].abs().max()) > 0.0


@pytest.mark.parametrize("grid,pbc,kw", [
    ((512, 16, 8), (0, 0, 0), {}),
    ((512, 15, 4), (0, 0, 0), dict(T=300.0, j=(1e12, -5e11, 2e11), P=0.5, xi=0.04)),     # odd Ny: a last single row
    ((1024, 8, 4), (1, 0, 0), dict(K1=4.8e4, K2=-1.0e4)),                                   # periodic x, cubic anisotropy
    ((512, 32, 2), (0, 1, 1), dict(T=300.0)),
    ((256, 6, 3), (0, 0, 0), {}),                          # x lines of 512: two row pairs per block, 9 pairs (ragged)
    ((512, 10, 2), (1, 0, 0), dict(T=300.0, j=(1e12, -5e11, 2e11), P=0.5, xi=0.04)),
    ((128, 32, 5), (0, 0, 0), {}),                         # x lines of 256 (config 3's)
    ((256, 7, 3), (1, 0, 0), dict(K1=4.8e4, K2=-1.0e4))])
def test_one_kernel_last_pass_gives_the_bits_of_the_split_one(grid, pbc, kw):
    """Option last_fused: inverse x transform and per-cell tail of a row pair in one block (k_inv_x_q, H_ms through
    shared memory) against k_inv_x_h + k_epi4 (H_ms through HBM): the same arithmetic on the same values, so H_eff,
    torque, fixed steps and controlled steps agree bit for bit; and the field meets the oracle."""
    wl = util.small(grid, (3e-9, 4e-9, 5e-9), pbc, seed=3, **kw)
    m = wlm.initial_m(wl)
    res = {}
    for flag in (0, 1):
        sim = util.gpu_sim(wl, options={"last_fused": flag})
        md = util.to_dev(m)
        H = sim.heff(md, step=2, dt_thermal=5e-14).clone()
        Tq = sim.torque(md, step=2, dt_thermal=5e-14).clone()
        l0 = sim.launch_count()
        sim.torque(md)
        nl = sim.launch_count() - l0
        sim.steps_fixed(md, "rk4", 5e-14, 3)
        out = [H, Tq, md.clone(), nl]
        if not kw.get("T"):
            md2 = util.to_dev(m)
            _, err = sim.steps_fixed(md2, "rkdp", 5e-14, 2)
            out += [md2.clone(), err]
        res[flag] = out
        sim.close()
    assert res[1][3] == res[0][3] - 1                     # one launch fewer per evaluation
    for a, b in zip(res[0][:3], res[1][:3]):
        assert float((a - b).abs().max()) == 0.0
    if not kw.get("T"):
        assert float((res[0][4] - res[1][4]).abs().max()) == 0.0 and res[0][5] == res[1][5]
    if not any(pbc):                                       # (periodic float128 image sums take too long here)
        ref = util.oracle_problem(wl).heff(m.astype(np.float64), 2, 5e-14)
        _cmp(res[1][0], ref, TOL_H)


def test_full_size_headline_grid_sampled_against_the_definition():
    """BASELINE.json's metric size (512x512x64, the launch configuration bench.py times).  The oracle
    cannot evaluate a dense state at this size in test time, so: (a) a sparse state of a few source
    cells -- H_ms is linear, so every output is a sum of a few tensor values the oracle computes one by
    one from the definition; (b) pin P7: uniform states give the sample's demagnetising factors;
    (c) pin P18: reciprocity and positive energy for two dense random states (no oracle needed)."""
    import torch
    wl = wlm.config(5)
    Nx, Ny, Nz = wl.grid
    Ms = wl.mat["Ms"]
    sim = util.gpu_sim(wl)
    # (a) sparse sources, incl. the corners that exercise the padding and every sign of the offsets
    src = [((0, 0, 0), (1.0, 0.0, 0.0)), ((Nx - 1, Ny - 1, Nz - 1), (0.0, 1.0, 0.0)),
           ((Nx // 2, Ny // 2, Nz // 2), (0.3, -0.5, 0.8)), ((Nx - 1, 0, 5), (0.0, 0.0, 1.0)),
           ((17, Ny - 3, Nz - 1), (-0.6, 0.6, 0.5)), ((300, 100, 20), (0.2, 0.9, -0.4))]
    m = torch.zeros((3, Nz, Ny, Nx), dtype=torch.float32, device="cuda")
    for (x, y, z), vec in src:
        for c in range(3):
            m[c, z, y, x] = vec[c]
    H = sim.demag_field(m)
    rng = np.random.default_rng(11)
    obs = []
    for (x, y, z), _ in src:                       # the sources themselves and their neighbourhoods
        for d in [(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -2, 0), (0, 0, 1), (0, 0, -1), (3, -2, 1),
                  (-7, 5, -3), (25, 14, 6)]:
            p = (x + d[0], y + d[1], z + d[2])
            if 0 <= p[0] < Nx and 0 <= p[1] < Ny and 0 <= p[2] < Nz:
                obs.append(p)
    obs += [(0, Ny - 1, 0), (Nx - 1, 0, Nz - 1), (Nx - 1, Ny - 1, 0), (0, 0, Nz - 1)]
    obs += [tuple(int(v) for v in (rng.integers(0, Nx), rng.integers(0, Ny), rng.integers(0, Nz))) for _ in range(20)]
    offs = np.array([[o[0] - s[0][0], o[1] - s[0][1], o[2] - s[0][2]] for o in obs for s in src])
    N6 = orc.tensor_at(offs, wl.cell).reshape(len(obs), len(src), 6)
    ref = np.zeros((len(obs), 3))
    for i in range(len(obs)):
        for k, (_, vec) in enumerate(src):
            xx, yy, zz, xy, xz, yz = N6[i, k]
            Nm = np.array([[xx, xy, xz], [xy, yy, yz], [xz, yz, zz]])
            ref[i] -= Ms * Nm @ np.array(vec)
    got = np.array([[float(H[c, o[2], o[1], o[0]]) for c in range(3)] for o in obs])
    scale = float(H.abs().max())
    assert np.abs(got - ref).max() <= TOL_H * scale, (np.abs(got - ref).max(), scale)
    big = np.abs(ref) > 1e-4 * scale               # mid-range values must be right on their own scale too
    assert big.sum() > 30
    assert (np.abs(got - ref)[big] <= 2e-3 * np.abs(ref)[big] + 2e-7 * scale).all()
    # (b) uniform states: mean field = - (demagnetising factor of the whole sample) Ms
    big_cell = tuple(c * n for c, n in zip(wl.cell, wl.grid))
    Nbig = orc.tensor_at([[0, 0, 0]], big_cell)[0]
    for a in range(3):
        m.zero_()
        m[a] = 1.0
        Hu = sim.demag_field(m)
        assert abs(float(Hu[a].double().mean()) / Ms + Nbig[a]) <= 2e-6
    # (c) reciprocity and positive energy, dense random states
    g = torch.Generator(device="cuda").manual_seed(5)
    m1 = torch.nn.functional.normalize(torch.randn((3, Nz, Ny, Nx), device="cuda", generator=g), dim=0)
    m2 = torch.nn.functional.normalize(torch.randn((3, Nz, Ny, Nx), device="cuda", generator=g), dim=0)
    H1 = sim.demag_field(m1).double()
    H2 = sim.demag_field(m2).double()
    a_, b_ = float((m1.double() * H2).sum()), float((m2.double() * H1).sum())
    assert abs(a_ - b_) <= 1e-5 * float((m1.double() * H1).sum().abs())
    assert float((m1.double() * H1).sum()) < 0.0
    sim.close()


def test_full_size_headline_grid_local_terms_and_torque():
    """Same size: the per-cell tail.  The local field terms (exchange, anisotropy, Zeeman) have no
    magnetostatic part, so the oracle evaluates them densely; the torque kernel is then checked by
    feeding the oracle's Landau-Lifshitz formula with the H_eff the GPU returned."""
    wl = wlm.config(5)
    m = wlm.initial_m(wl)
    m64 = m.astype(np.float64)
    md = util.to_dev(m)
    mat = util.oracle_material(wl.mat)
    Hloc = orc.exchange_field(m64, mat, wl.grid, wl.cell, wl.pbc) + orc.anisotropy_field(m64, mat) \
        + orc.zeeman_field(m64, mat)
    sim = util.gpu_sim(wl)
    Hms = sim.demag_field(md).double().cpu().numpy()
    Heff = sim.heff(md).double().cpu().numpy()
    s = np.abs(Heff).max()
    assert np.abs(Heff - (Hms + Hloc)).max() <= TOL_H * s
    Tref = orc.ll_torque(m64, Heff, mat, wl.grid, wl.cell, wl.pbc)
    _cmp(sim.torque(md), Tref, TOL_H)
    sim.close()


@pytest.mark.parametrize("method", ["rk1", "rk4"])
def test_graph_replayed_steps_equal_plain_launches(method):
    """mm_steps_fixed replays a captured step for the fixed-step, non-FSAL methods: same bits as plain launches."""
    wl = util.small((32, 32, 1), (4e-9, 4e-9, 4e-9), alpha=0.5)
    m = wlm.initial_m(wl)
    out = []
    for flag in (1, 0):
        sim = util.gpu_sim(wl, options={"graph": flag})
        md = util.to_dev(m)
        t, _ = sim.steps_fixed(md, method, 1e-13, 25)
        l0 = sim.launch_count()
        t, _ = sim.steps_fixed(md, method, 1e-13, 3)         # below the replay threshold
        assert abs(t - 3e-13) < 1e-25 and sim.launch_count() > l0
        out.append(md.cpu().numpy().copy())
        sim.close()
    assert np.array_equal(out[0], out[1])


@pytest.mark.parametrize("method", ["rkdp", "rk23"])
def test_device_side_step_controller_follows_the_host_controlled_run(method):
    """Step a11: mm_steps_adaptive keeps error norm, accept / reject, dt and t on the device; it must
    take the same decisions as mm_step (one host sync per step) and end in the same state."""
    wl = util.small((24, 12, 8), init="tilted", alpha=0.02, Bext=(-0.0246, 0.0043, 0.0), Ku=0.0)
    m = wlm.initial_m(wl)
    tol, ntr = 1e-5, 40
    sim = util.gpu_sim(wl)
    md = util.to_dev(m)
    dt, t, nacc = 4e-13, 0.0, 0              # starts too long: the first trials are rejected
    for _ in range(ntr):
        acc, err, dt, t = sim.step(md, method, dt, tol, t)
        nacc += int(acc)
    ref = md.double().cpu().numpy()
    assert 0 < nacc < ntr
    sim2 = util.gpu_sim(wl)
    md2 = util.to_dev(m)
    nacc2, err2, dt2, t2 = sim2.steps_adaptive(md2, method, ntr, 4e-13, tol, 0.0)
    assert nacc2 == nacc
    # the tableau is scaled by dt in fp32 on the device and in fp64 on the host: the error estimates, hence
    # the step lengths, agree to a few 1e-5
    assert abs(t2 - t) <= 1e-4 * t and abs(dt2 - dt) <= 2e-3 * dt
    assert abs(err2 - err) <= 0.02 * err + 1e-12
    assert np.abs(md2.double().cpu().numpy() - ref).max() <= 1e-5
    # split into two calls: the FSAL stage and the device scalars carry over
    sim3 = util.gpu_sim(wl)
    md3 = util.to_dev(m)
    n1, _, dt3, t3 = sim3.steps_adaptive(md3, method, 15, 4e-13, tol, 0.0)
    n2, _, dt3, t3 = sim3.steps_adaptive(md3, method, ntr - 15, dt3, tol, t3)
    assert n1 + n2 == nacc and abs(t3 - t) <= 1e-4 * t
    assert np.abs(md3.double().cpu().numpy() - ref).max() <= 1e-5
    for s_ in (sim, sim2, sim3):
        s_.close()


# ---- the remaining Runge-Kutta tableaux, the maximum-variation step, <m> ----
@pytest.mark.parametrize("method", ["rk2", "rk3", "rk12", "rk23", "rkck"])
def test_remaining_tableaux_follow_the_oracle(method):
    wl = util.small((24, 10, 6), init="tilted", alpha=0.05, Bext=(-0.0246, 0.0043, 0.0))
    m = wlm.initial_m(wl)
    pb = util.oracle_problem(wl)
    dt, n = 4e-14, 12
    mo, k1, errs = m.astype(np.float64), None, []
    for _ in range(n):
        mo, err, kl = orc.rk_step(pb.torque, mo, dt, method, k1)
        k1 = kl if method in orc.FSAL else None
        errs.append(err)
    sim = util.gpu_sim(wl)
    md = util.to_dev(m)
    for i in range(n):
        _, ge = sim.steps_fixed(md, method, dt, 1)
        if errs[i] is not None:
            # fp32 floor of the embedded difference: a few 1e-10 (dimensionless), far below any tolerance in use
            assert abs(ge - errs[i]) <= 0.02 * errs[i] + 1e-9, (i, ge, errs[i])
    assert np.abs(md.double().cpu().numpy() - mo).max() <= TOL_M
    md2 = util.to_dev(m)                       # the same in one call
    sim.reset_stepper(0)
    sim.steps_fixed(md2, method, dt, n)
    assert np.abs(md2.double().cpu().numpy() - mo).max() <= TOL_M
    sim.close()


@pytest.mark.parametrize("fsal", ["rkdp", "rk23"])
def test_saved_first_stage_is_dropped_when_another_method_runs_in_between(fsal):
    """FSAL step, then fixed steps of a method that overwrites the first-stage buffer, then FSAL again: the
    saved k_1 belongs to an older state and must not be reused (the oracle evaluates k_1 afresh)."""
    wl = util.small((24, 10, 6), init="tilted", alpha=0.05, Bext=(-0.0246, 0.0043, 0.0))
    m = wlm.initial_m(wl)
    pb = util.oracle_problem(wl)
    dt = 6e-14
    mo = m.astype(np.float64)
    mo, _, _ = orc.rk_step(pb.torque, mo, dt, fsal)
    for _ in range(3):
        mo = orc.rk4_step(pb.torque, mo, dt)
    mo, err_o, _ = orc.rk_step(pb.torque, mo, dt, fsal)          # k_1 evaluated on the current state
    for inner in ("fixed", "step"):
        sim = util.gpu_sim(wl)
        md = util.to_dev(m)
        sim.steps_fixed(md, fsal, dt, 1)
        if inner == "fixed":
            sim.steps_fixed(md, "rk4", dt, 3)
        else:
            for _ in range(3):
                sim.step(md, "rk4", dt)
        _, err_g = sim.steps_fixed(md, fsal, dt, 1)
        assert np.abs(md.double().cpu().numpy() - mo).max() <= 2e-6
        assert abs(err_g - err_o) <= 0.02 * err_o + 1e-9
        sim.close()


def test_fixed_step_fsal_method_with_thermal_field_redraws_per_step():
    """Reading A6: one draw per step, held over that step's own stages -- the first stage of step n+1 is
    evaluated with draw n+1, so the last stage of step n (draw n) cannot be reused when T > 0."""
    wl = util.small((16, 12, 1), (4e-9, 4e-9, 2e-9), (2, 2, 0), init="xnoise", alpha=0.1, T=300.0, seed=3)
    m = wlm.initial_m(wl)
    pb = util.oracle_problem(wl)
    dt, n = 5e-14, 4
    mo = m.astype(np.float64)
    for i in range(n):
        mo, _, _ = orc.rk_step(lambda x: pb.torque(x, step=i, dt_thermal=dt), mo, dt, "rk23")
    sim = util.gpu_sim(wl)
    md = util.to_dev(m)
    sim.steps_fixed(md, "rk23", dt, n)
    assert np.abs(md.double().cpu().numpy() - mo).max() <= TOL_M
    sim.close()


def test_cash_karp_adaptive_run_matches_the_oracle_controller():
    wl = util.small((24, 10, 6), init="tilted", alpha=0.02, Bext=(-0.0246, 0.0043, 0.0), Ku=0.0)
    m = wlm.initial_m(wl)
    pb = util.oracle_problem(wl)
    tol, dt, mo, seq, trials = 1e-5, 3e-13, m.astype(np.float64), [], 0
    while len(seq) < 20:
        mn, err, _ = orc.rk_step(pb.torque, mo, dt, "rkck")
        ok, dtn = orc.rk_controller(dt, err, tol, "rkck")
        trials += 1
        if ok:
            seq.append(dt); mo = mn
        dt = dtn
    sim = util.gpu_sim(wl)
    md = util.to_dev(m)
    dt, t, nacc, ntr = 3e-13, 0.0, 0, 0
    while nacc < 20:
        acc, err, dt, t = sim.step(md, "rkck", dt, tol, t)
        ntr += 1; nacc += int(acc)
    assert abs(ntr - trials) <= 1 and abs(t - sum(seq)) <= 0.02 * sum(seq)
    assert np.abs(md.double().cpu().numpy() - mo).max() <= 1e-3
    md2 = util.to_dev(m)                       # controller on the device
    sim.reset_stepper(0)
    n2, _, _, t2 = sim.steps_adaptive(md2, "rkck", ntr, 3e-13, tol, 0.0)
    assert n2 == 20 and abs(t2 - t) <= 1e-3 * t
    sim.close()


@pytest.mark.parametrize("method", ["rk1", "rk2", "rk4"])
def test_maximum_variation_step_length(method):
    """the fixed-step methods with 'a fixed maximum variation of m per step'."""
    wl = util.small((24, 10, 6), init="tilted", alpha=0.1, Bext=(-0.0246, 0.0043, 0.0))
    m = wlm.initial_m(wl)
    pb = util.oracle_problem(wl)
    max_dm, n = 2e-3, 10
    mo, t_ref, dt_ref = m.astype(np.float64), 0.0, 0.0
    for _ in range(n):
        dt_ref, k1 = orc.max_dm_step_length(pb.torque, mo, max_dm)
        mo, _, _ = orc.rk_step(pb.torque, mo, dt_ref, method, k1)
        t_ref += dt_ref
    sim = util.gpu_sim(wl)
    md = util.to_dev(m)
    t, last_dt = sim.steps_maxdm(md, method, max_dm, n)
    assert abs(t - t_ref) <= 1e-4 * t_ref and abs(last_dt - dt_ref) <= 1e-4 * dt_ref
    assert np.abs(md.double().cpu().numpy() - mo).max() <= TOL_M
    sim.close()


def test_average_magnetisation():
    wl = util.small((40, 6, 3), (2e-9, 2e-9, 4e-9))
    m = wlm.initial_m(wl)
    sim = util.gpu_sim(wl)
    avg = sim.average(util.to_dev(m))
    assert np.abs(avg - orc.average_m(m.astype(np.float64))).max() <= 1e-7
    sim.close()


def test_graph_replay_with_thermal_field_draws_per_step():
    """With a thermal field the step index that selects the draw is advanced on the device during the
    replay: same bits as plain launches, and as the oracle's per-step draws (reading A6)."""
    wl = util.small((16, 12, 1), (4e-9, 4e-9, 2e-9), (2, 2, 0), init="xnoise", alpha=0.1, T=300.0, seed=3)
    m = wlm.initial_m(wl)
    out = []
    for flag in (1, 0):
        sim = util.gpu_sim(wl, options={"graph": flag})
        md = util.to_dev(m)
        sim.steps_fixed(md, "rk4", 5e-14, 8)
        sim.steps_fixed(md, "rk4", 5e-14, 6)          # continues at step index 8
        out.append(md.cpu().numpy().copy())
        sim.close()
    assert np.array_equal(out[0], out[1])
    pb = util.oracle_problem(wl)
    mo = m.astype(np.float64)
    for s_ in range(14):
        mo = orc.rk4_step(lambda x: pb.torque(x, s_, 5e-14), mo, 5e-14)
    assert np.abs(out[0].astype(np.float64) - mo).max() <= TOL_M


@pytest.mark.parametrize("grid,fast", [((24, 10, 6), 0), ((64, 32, 32), 63), ((15, 9, 5), 0)])
def test_cubic_anisotropy_matches_oracle(grid, fast):
    """Eq. (5) with tilted axes, next to every other field term."""
    wl = util.small(grid, (3e-9, 4e-9, 5e-9), K1=-4.5e4, K2=2.3e4, anis_c1=(1.0, 1.0, 0.0), anis_c2=(-1.0, 1.0, 0.3),
                    j=(1e12, 0, 0), P=0.5, xi=0.04)
    m = wlm.initial_m(wl)
    m64 = m.astype(np.float64)
    pb = util.oracle_problem(wl)
    sim = util.gpu_sim(wl, fast=fast)
    md = util.to_dev(m)
    _cmp(sim.heff(md), pb.heff(m64), TOL_H)
    _cmp(sim.torque(md), pb.torque(m64), TOL_H)
    # the cubic term on its own scale: switch everything else off
    wl2 = util.small(grid, (3e-9, 4e-9, 5e-9), K1=-4.5e4, K2=2.3e4, anis_c1=(1.0, 1.0, 0.0), anis_c2=(-1.0, 1.0, 0.3),
                     Aex=0.0, Ku=0.0, Bext=(0.0, 0.0, 0.0))
    sim2 = util.gpu_sim(wl2, demag=False)
    ref = orc.cubic_anisotropy_field(m64, util.oracle_material(wl2.mat))
    _cmp(sim2.heff(md), ref, 2e-6)
    mo = m64.copy()
    for _ in range(5):
        mo = orc.rk4_step(pb.torque, mo, 5e-14)
    sim.steps_fixed(md, "rk4", 5e-14, 5)
    assert np.abs(md.double().cpu().numpy() - mo).max() <= TOL_M
    sim.close(); sim2.close()


@pytest.mark.parametrize("grid,pbc,fast", [((24, 10, 6), (0, 0, 0), 0), ((64, 32, 32), (0, 0, 0), 63),
                                           ((16, 12, 1), (2, 2, 0), 0), ((32, 32, 32), (0, 1, 0), 63)])
def test_exchange_inside_the_kernel_variant(grid, pbc, fast):
    """SURVEY 8(f) row f-2, PAPER.md:85 (reading A3'): the exchange stencil rides on the convolution
    kernel; H_eff changes only at open faces (by a field parallel to m), the torque not at all."""
    wl = util.small(grid, (3e-9, 4e-9, 5e-9), pbc, exchange_in_kernel=True)
    wl0 = util.small(grid, (3e-9, 4e-9, 5e-9), pbc)
    m = wlm.initial_m(wl)
    m64 = m.astype(np.float64)
    pb = util.oracle_problem(wl)
    sim = util.gpu_sim(wl, fast=fast)
    md = util.to_dev(m)
    H = sim.heff(md)
    _cmp(H, pb.heff(m64), TOL_H)
    _cmp(sim.torque(md), pb.torque(m64), TOL_H)
    _cmp(sim.demag_field(md), pb.demag_field(m64), TOL_H)          # the pure magnetostatic field is unchanged
    sim0 = util.gpu_sim(wl0, fast=fast)
    T0, T1 = sim0.torque(md).double(), sim.torque(md).double()
    assert float((T0 - T1).abs().max()) <= 5e-5 * float(T0.abs().max())
    if tuple(pbc) == (0, 0, 0):
        d = (H - sim0.heff(md)).double()
        assert float(d[:, 1:-1, 1:-1, 1:-1].abs().max()) <= 2e-5 * float(H.abs().max())   # interior: same field
        assert float(d.abs().max()) > 1e-2 * float(H.abs().max())                           # faces: not
    sim.close(); sim0.close()


@pytest.mark.parametrize("grid,fast", [((24, 10, 6), 0), ((64, 32, 32), 63), ((30, 12, 1), 0)])
def test_staircase_geometry(grid, fast):
    """SURVEY 8(f) row f-2 (reading A15): cells with m = 0 are empty."""
    wl = util.small(grid, (3e-9, 4e-9, 5e-9), geometry=True, j=(1e12, -5e11, 0.0), P=0.5, xi=0.04, alpha=0.1)
    m = wlm.initial_m(wl)
    Nx, Ny, Nz = grid
    z, y, x = np.meshgrid(np.arange(Nz), np.arange(Ny), np.arange(Nx), indexing="ij")
    shape = ((x - Nx / 2.0) / (Nx / 2.0)) ** 2 + ((y - Ny / 2.0) / (Ny / 2.0)) ** 2 <= 1.0     # elliptic cylinder
    shape &= ~((abs(x - Nx // 3) <= 1) & (abs(y - Ny // 2) <= 1))                                  # with a hole
    m = m * shape[None].astype(np.float32)
    m64 = m.astype(np.float64)
    pb = util.oracle_problem(wl)
    sim = util.gpu_sim(wl, fast=fast)
    md = util.to_dev(m)
    _cmp(sim.heff(md), pb.heff(m64), TOL_H)
    _cmp(sim.torque(md), pb.torque(m64), TOL_H)
    mo = m64.copy()
    for _ in range(5):
        mo = orc.rk4_step(pb.torque, mo, 5e-14)
    sim.steps_fixed(md, "rk4", 5e-14, 5)
    out = md.double().cpu().numpy()
    assert np.abs(out - mo).max() <= TOL_M
    assert np.all(out[:, ~shape] == 0.0) and np.isfinite(out).all()
    sim.close()
