"""python -m paper_1102_3069_b200.selfcheck NX NY NZ [--pbc a b c] [--films B] [--ranks R]

Runs every entry point of the hot path once on a seeded state of the given grid and prints checksums: a small,
oracle-free target for compute-sanitizer (racecheck / memcheck) and for a first look at a new machine."""
from __future__ import annotations

import argparse

import numpy as np


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("grid", type=int, nargs=3)
    ap.add_argument("--pbc", type=int, nargs=3, default=[0, 0, 0])
    ap.add_argument("--films", type=int, default=0)
    ap.add_argument("--ranks", type=int, default=0)
    a = ap.parse_args()
    import torch
    import paper_1102_3069_b200 as mm
    from paper_1102_3069_b200 import workloads as wlm
    wl = wlm.scaled(wlm.config(3), tuple(a.grid), pbc=tuple(a.pbc))       # thermal field and current on
    m = wlm.initial_m(wl)
    if a.ranks:
        from paper_1102_3069_b200 import dist as mmd
        ranks = [mmd.SlabRank(wl.grid, wl.cell, wl.pbc, wl.mat, r, a.ranks) for r in range(a.ranks)]
        ms = [torch.from_numpy(np.ascontiguousarray(m[:, r.slab.z0:r.slab.z1])).cuda() for r in ranks]
        out = torch.cat(mmd.evaluate_local(ranks, ms, "torque", step=1, dt_thermal=5e-14), dim=1)
        print("slab torque checksum", float(out.double().abs().sum()))
        return
    if a.films:
        m = np.ascontiguousarray(np.repeat(m, a.films, axis=1))
    sim = mm.Sim(wl.grid, wl.cell, wl.pbc, wl.mat, nfilms=a.films)
    md = torch.from_numpy(m).cuda()
    print("H_ms checksum", float(sim.demag_field(md).double().abs().sum()))
    print("H_eff checksum", float(sim.heff(md, step=1, dt_thermal=5e-14).double().abs().sum()))
    print("torque checksum", float(sim.torque(md, step=1, dt_thermal=5e-14).double().abs().sum()))
    sim.steps_fixed(md, "rk4", 5e-14, 6)
    sim.set_material(dict(wl.mat, T=0.0))
    sim.steps_fixed(md, "rkdp", 5e-14, 2)
    n, err, dt, t = sim.steps_adaptive(md, "rkdp", 3, 5e-14, 1e-5)
    print("state checksum", float(md.double().abs().sum()), "accepted", n, "launches", sim.launch_count())
    sim.close()


if __name__ == "__main__":
    main()
