"""Multi-GPU reading of DESIGN.md section 9: replicas only.  The aggregation bench.py uses for N > 1
(barrier, max over ranks of the timed region, value = all ranks' evaluations / that time) is checked
here with two CPU processes over gloo; no data-path collective exists to test."""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys, json
    import torch, torch.distributed as dist
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    sec = 0.5 + 0.25 * rank              # rank 1 is the slower replica
    evals = 40                           # per rank: weak scaling, every replica does the same work
    dist.barrier()
    t = torch.tensor([sec], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    value = world * evals / float(t.item())
    if rank == 0:
        print(json.dumps({"value": value, "n_gpus": world, "sec": float(t.item())}))
    dist.destroy_process_group()
""")


def test_two_rank_replica_aggregation(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29631", str(w)],
                         capture_output=True, text=True, env=env, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    import json
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["n_gpus"] == 2 and abs(d["sec"] - 0.75) < 1e-12
    assert abs(d["value"] - 2 * 40 / 0.75) < 1e-9
