"""Multi-GPU slab decomposition: the host-side partition and the
all-to-all bookkeeping of the LIBRARY (mm_slab_partition, mm_slab_segment), checked on the CPU -- single process
for the ownership properties, two processes over gloo for the exchange itself.  No oracle is involved: this is
index arithmetic of the product's own host code."""
import json
import os
import subprocess
import sys
import textwrap

import numpy as np
import pytest

import paper_1102_3069_b200 as mm

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CASES = [((512, 512, 64), (0, 0, 0), 8), ((64, 32, 64), (0, 0, 0), 2), ((64, 32, 64), (0, 0, 0), 3),
         ((128, 64, 32), (0, 0, 1), 4), ((768, 384, 64), (0, 0, 0), 8), ((64, 32, 5), (0, 0, 0), 5)]


@pytest.mark.parametrize("grid,pbc,R", CASES)
def test_every_plane_and_every_column_has_exactly_one_owner(grid, pbc, R):
    Cx = (grid[0] if pbc[0] else 2 * grid[0]) // 2 + 1
    slabs = [mm.mm.slab_partition(grid, pbc, R, r) for r in range(R)]
    planes = np.zeros(grid[2], dtype=int)
    cols = np.zeros(Cx, dtype=int)
    for r, s in enumerate(slabs):
        assert (s.rank, s.nranks) == (r, R) and s.z0 < s.z1 and s.kx0 < s.kx1
        assert s.kx0 % 16 == 0 and (s.kx1 % 16 == 0 or s.kx1 == Cx)      # whole 16-column tiles
        planes[s.z0:s.z1] += 1
        cols[s.kx0:s.kx1] += 1
    assert (planes == 1).all() and (cols == 1).all()
    nz = [s.z1 - s.z0 for s in slabs]
    assert max(nz) - min(nz) <= 1                                        # balanced
    assert [s.z0 for s in slabs] == sorted(s.z0 for s in slabs)          # contiguous, in rank order


@pytest.mark.parametrize("grid,pbc,R", CASES)
def test_segments_tile_both_buffers_and_counts_match_between_ranks(grid, pbc, R):
    Py = grid[1] if pbc[1] else 2 * grid[1]
    Cx = (grid[0] if pbc[0] else 2 * grid[0]) // 2 + 1
    seg = {(r, p, c): mm.mm.slab_segment(grid, pbc, R, r, p, c) for r in range(R) for p in range(R) for c in range(3)}
    for r in range(R):
        s = mm.mm.slab_partition(grid, pbc, R, r)
        ws = lambda q: (q.kx1 - q.kx0 + 7) // 8 * 8            # row stride of a rank's columns (64-byte rows)
        nzl, W = s.z1 - s.z0, ws(s)
        slab = np.zeros(3 * nzl * Py * sum(ws(mm.mm.slab_partition(grid, pbc, R, q)) for q in range(R)), dtype=int)
        pen = np.zeros(3 * grid[2] * Py * W, dtype=int)
        for p in range(R):
            for c in range(3):
                so, sc, po, pc = seg[(r, p, c)]
                slab[so:so + sc] += 1
                pen[po:po + pc] += 1
                # what r sends to p is what p expects from r, in both directions
                assert sc == seg[(p, r, c)][3] and pc == seg[(p, r, c)][1]
        assert (slab == 1).all() and (pen == 1).all()                    # no gap, no overlap


def test_bad_partitions_are_refused():
    with pytest.raises(mm.mm.MMError):
        mm.mm.slab_partition((64, 32, 4), (0, 0, 0), 5, 0)               # more ranks than planes
    with pytest.raises(mm.mm.MMError):
        mm.mm.slab_partition((16, 32, 64), (0, 0, 0), 3, 0)              # 17 columns = 2 tiles < 3 ranks
    with pytest.raises(mm.mm.MMError):
        mm.mm.slab_partition((64, 32, 64), (0, 0, 0), 2, 2)              # rank out of range


WORKER = textwrap.dedent("""
    import json, sys
    import numpy as np, torch, torch.distributed as dist
    sys.path.insert(0, %r)
    import paper_1102_3069_b200 as mm
    dist.init_process_group("gloo")
    r, R = dist.get_rank(), dist.get_world_size()
    grid, pbc = (32, 8, 6), (0, 0, 0)
    Py, Nz = 16, grid[2]
    me = mm.mm.slab_partition(grid, pbc, R, r)
    peers = [mm.mm.slab_partition(grid, pbc, R, p) for p in range(R)]
    ws = lambda q: (q.kx1 - q.kx0 + 7) // 8 * 8
    nzl, W = me.z1 - me.z0, ws(me)

    def gid(c, z, ky, kx):                       # one id per element of the y-transformed half spectrum
        return ((c * Nz + z) * Py + ky) * 64 + kx

    # slab side as the forward y pass leaves it: [peer][3][nzl][Py][W(peer)]
    slab = torch.empty(3 * nzl * Py * sum(ws(q) for q in peers), dtype=torch.int64)
    for p, ps in enumerate(peers):
        for c in range(3):
            so, sc, _, _ = mm.mm.slab_segment(grid, pbc, R, r, p, c)
            z, ky, kx = np.meshgrid(np.arange(me.z0, me.z1), np.arange(Py), ps.kx0 + np.arange(ws(ps)), indexing="ij")
            slab[so:so + sc] = torch.from_numpy(gid(c, z, ky, kx).ravel())
    pen = torch.full((3 * Nz * Py * W,), -1, dtype=torch.int64)
    ops, keep = [], []
    for p in range(R):
        for c in range(3):
            so, sc, po, pc = mm.mm.slab_segment(grid, pbc, R, r, p, c)
            if p == r:
                pen[po:po + pc] = slab[so:so + sc]
            else:
                ops.append(dist.P2POp(dist.isend, slab[so:so + sc], p))
                ops.append(dist.P2POp(dist.irecv, pen[po:po + pc], p))
    for w in dist.batch_isend_irecv(ops):
        w.wait()
    # pencil side: [3][Nz][Py][W] holding this rank's columns of EVERY plane
    c, z, ky, kx = np.meshgrid(np.arange(3), np.arange(Nz), np.arange(Py), me.kx0 + np.arange(W), indexing="ij")
    ok1 = bool((pen.numpy() == gid(c, z, ky, kx).ravel()).all())
    # and back
    back = torch.full_like(slab, -1)
    ops = []
    for p in range(R):
        for c_ in range(3):
            so, sc, po, pc = mm.mm.slab_segment(grid, pbc, R, r, p, c_)
            if p == r:
                back[so:so + sc] = pen[po:po + pc]
            else:
                ops.append(dist.P2POp(dist.isend, pen[po:po + pc], p))
                ops.append(dist.P2POp(dist.irecv, back[so:so + sc], p))
    for w in dist.batch_isend_irecv(ops):
        w.wait()
    ok2 = bool((back == slab).all())
    res = torch.tensor([int(ok1), int(ok2)])
    dist.all_reduce(res, op=dist.ReduceOp.MIN)
    if r == 0:
        print(json.dumps({"to_pencil": int(res[0]), "back": int(res[1]), "world": R}))
    dist.destroy_process_group()
""")


def test_two_process_all_to_all_moves_every_element_to_its_owner_and_back(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER % ROOT)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29641", str(w)],
                         capture_output=True, text=True, env=env, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-3000:]
    d = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert d == {"to_pencil": 1, "back": 1, "world": 2}
