"""Multi-GPU reading of DESIGN.md section 9: replicas only.  `python bench.py --gpus 2 --dry` must start two
ranks of bench.py itself (as the driver's torchrun launch does), rendezvous over gloo, and aggregate with the
same function the GPU arm uses: job time = max over ranks, value = all ranks' evaluations / that time.
No data-path collective exists to test."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _last_json(out):
    return json.loads([l for l in out.splitlines() if l.startswith("{")][-1])


def test_gpus_flag_spawns_that_many_ranks_and_aggregates_over_them():
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "10", "--dry"],
                         capture_output=True, text=True, env=env, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    d = _last_json(out.stdout)
    # stub times 0.5 s (rank 0) and 0.75 s (rank 1): the slower replica sets the job time
    assert d["n_gpus"] == 2 and abs(d["sec"] - 0.75) < 1e-12
    assert abs(d["value"] - 2 * 40 / 0.75) < 1e-9


def test_launched_by_torchrun_directly_as_the_driver_does():
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29631", os.path.join(ROOT, "bench.py"),
                          "--gpus", "2", "--steps", "5", "--dry"],
                         capture_output=True, text=True, env=env, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    d = _last_json(out.stdout)
    assert d["n_gpus"] == 2 and abs(d["value"] - 2 * 20 / 0.75) < 1e-9


def test_replica_aggregate_single_rank():
    sys.path.insert(0, ROOT)
    import bench
    sec, value = bench.replica_aggregate(0.25, 40, 1)
    assert sec == 0.25 and value == 160.0
