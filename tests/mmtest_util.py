"""Test helpers: build the oracle problem and the CUDA context from one Workload."""
import numpy as np

from oracle import mm_oracle as orc
from paper_1102_3069_b200 import workloads as wlm


def oracle_material(matd):
    return orc.Material(Ms=matd["Ms"], Aex=matd["Aex"], alpha=matd["alpha"],
                        gamma0=matd.get("gamma0") or orc.GAMMA0_DEFAULT, Ku=matd["Ku"],
                        anis_u=tuple(matd["anis_u"]), Bext=tuple(matd["Bext"]), T=matd["T"],
                        seed=matd["seed"], j=tuple(matd["j"]), P=matd["P"], xi=matd["xi"],
                        stt_literal_eq7=bool(matd["stt_literal_eq7"]), K1=matd.get("K1", 0.0), K2=matd.get("K2", 0.0),
                        anis_c1=tuple(matd.get("anis_c1", (1.0, 0.0, 0.0))),
                        anis_c2=tuple(matd.get("anis_c2", (0.0, 1.0, 0.0))),
                        exchange_in_kernel=bool(matd.get("exchange_in_kernel", False)),
                        geometry=bool(matd.get("geometry", False)))


def oracle_problem(wl, demag="fft"):
    return orc.Problem(wl.grid, wl.cell, wl.pbc, oracle_material(wl.mat), demag=demag)


def gpu_sim(wl, demag=True, fast=True, options=None):
    import paper_1102_3069_b200 as mm
    sim = mm.Sim(wl.grid, wl.cell, wl.pbc, wl.mat, demag=demag, options=options)
    sim.set_fast_path(fast)
    return sim


def to_dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def small(grid, cell=(3e-9, 4e-9, 5e-9), pbc=(0, 0, 0), init="random", seed=7, **mat):
    base = dict(alpha=0.1, Ku=2e4, anis_u=(1.0, 2.0, 0.5), Bext=(0.01, -0.02, 0.005))
    base.update(mat)
    return wlm.Workload(f"small_{'x'.join(map(str, grid))}", tuple(grid), tuple(cell), tuple(pbc),
                        wlm._mat(**base), init, seed)
