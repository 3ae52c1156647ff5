"""Slab decomposition over several GPUs (include/mm.h "multi-GPU slab decomposition").

Marshalling and communication plumbing only: every arithmetic step runs in the library's kernels
(mm_dist_forward / mm_dist_mid / mm_dist_backward).  What happens here is what the library leaves to its
caller: the two all-to-alls between the phases and the one-plane halo exchange of m.

Two transports with the same segment lists:
  * NcclTransport -- one process per GPU, torch.distributed (backend nccl): batched isend / irecv of the
    contiguous (peer, component) segments, i.e. a flat all-to-all over NVLink / NVSwitch;
  * LocalTransport -- all ranks are contexts of ONE process on ONE GPU and a "send" is a device-to-device copy.
    This is the single-GPU stand-in the tests use (ranks run one after the other, phase by phase: no kernel
    ever waits for another rank).
"""
from __future__ import annotations

import ctypes as C

from . import mm as _mm


class SlabRank:
    """One rank's context (mm_create_dist) with torch views of its two exchange buffers."""

    def __init__(self, grid, cell, pbc, mat, rank, nranks, demag=True, stream=None):
        import torch
        self.torch = torch
        self.L = _mm.lib()
        self.grid = tuple(int(v) for v in grid)
        self.pbc = tuple(int(v) for v in pbc)
        self.rank, self.nranks = int(rank), int(nranks)
        self.slab = _mm.slab_partition(grid, pbc, nranks, rank)
        self.peers = [_mm.slab_partition(grid, pbc, nranks, p) for p in range(nranks)]
        self.shape = (3, self.slab.z1 - self.slab.z0, self.grid[1], self.grid[0])
        self.ctx = C.c_void_p()
        s = stream if stream is not None else torch.cuda.current_stream()
        st = self.L.mm_create_dist(C.byref(self.ctx), _mm._i3(grid), _mm._d3(cell), _mm._i3(pbc),
                                   C.c_void_p(s.cuda_stream), self.rank, self.nranks)
        if st != _mm.MM_OK:
            raise _mm.MMError(st, self.L.mm_last_error(None).decode())
        m = mat if isinstance(mat, _mm.Material) else _mm.Material.from_dict(mat, demag)
        self._chk(self.L.mm_set_material(self.ctx, C.byref(m)))
        self._chk(self.L.mm_demag_init(self.ctx))
        sb, pb, ns, npn = C.c_void_p(), C.c_void_p(), C.c_size_t(), C.c_size_t()
        self._chk(self.L.mm_dist_buffers(self.ctx, C.byref(sb), C.byref(ns), C.byref(pb), C.byref(npn)))
        self.slab_buf = self._view(sb.value, ns.value)
        self.pencil_buf = self._view(pb.value, npn.value)

    def _view(self, ptr, nelem):
        """A torch float32 view (2 floats per complex element) of library-owned device memory."""
        torch = self.torch

        class _Holder:                      # __cuda_array_interface__ of a raw pointer; the context owns the memory
            pass
        h = _Holder()
        h.__cuda_array_interface__ = {"shape": (2 * nelem,), "typestr": "<f4", "data": (ptr, False), "version": 2}
        return torch.as_tensor(h, device="cuda")

    def _chk(self, st):
        if st != _mm.MM_OK:
            raise _mm.MMError(st, self.L.mm_last_error(self.ctx).decode())

    def segment(self, peer, comp):
        """(slab view, pencil view) of the contiguous segment exchanged with `peer` for component comp."""
        so, sc, po, pc = C.c_size_t(), C.c_size_t(), C.c_size_t(), C.c_size_t()
        self._chk(self.L.mm_dist_segment(self.ctx, peer, comp, C.byref(so), C.byref(sc), C.byref(po), C.byref(pc)))
        return (self.slab_buf[2 * so.value: 2 * (so.value + sc.value)],
                self.pencil_buf[2 * po.value: 2 * (po.value + pc.value)])

    def _dev(self, t):
        assert t.is_cuda and t.dtype == self.torch.float32 and t.is_contiguous() and tuple(t.shape) == self.shape
        return C.c_void_p(t.data_ptr())

    def forward(self, m):
        self._chk(self.L.mm_dist_forward(self.ctx, self._dev(m)))

    def mid(self):
        self._chk(self.L.mm_dist_mid(self.ctx))

    def backward(self, m, halo_lo, halo_hi, out, what, step=0, dt_thermal=0.0):
        p = lambda t: C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)
        self._chk(self.L.mm_dist_backward(self.ctx, self._dev(m) if m is not None else C.c_void_p(0), p(halo_lo),
                                          p(halo_hi), self._dev(out), int(what), int(step), float(dt_thermal)))

    def stage_input(self, m, method, stage):
        """The field stage `stage` acts on, as a torch view (m itself for stage 0, else a buffer of the context)."""
        out = C.c_void_p()
        self._chk(self.L.mm_dist_stage_input(self.ctx, _mm.METHODS[method], int(stage), self._dev(m), C.byref(out)))
        if out.value == m.data_ptr():
            return m
        n = 1
        for v in self.shape:
            n *= v
        return self._view(out.value, n // 2).view(self.shape)

    def backward_stage(self, m, method, stage, dt, step, halo_lo, halo_hi):
        p = lambda t: C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)
        self._chk(self.L.mm_dist_backward_stage(self.ctx, self._dev(m), _mm.METHODS[method], int(stage), float(dt),
                                                int(step), p(halo_lo), p(halo_hi)))

    def halo_neighbours(self):
        """(rank below, rank above) whose boundary planes this rank needs, None at an open end of the grid."""
        lo = self.rank - 1 if self.rank > 0 else (self.nranks - 1 if self.pbc[2] > 0 else None)
        hi = self.rank + 1 if self.rank + 1 < self.nranks else (0 if self.pbc[2] > 0 else None)
        if self.nranks == 1 and self.pbc[2] > 0:
            lo = hi = 0
        return lo, hi

    def close(self):
        if self.ctx:
            self.L.mm_destroy(self.ctx)
            self.ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class LocalTransport:
    """All ranks in one process on one GPU: a send is a device-to-device copy (test stand-in for NVLink)."""

    def __init__(self, ranks):
        self.ranks = ranks

    def all_to_all(self, to_pencil: bool):
        R = len(self.ranks)
        for src in self.ranks:
            for dst in self.ranks:
                for comp in range(3):
                    s_slab, _ = src.segment(dst.rank, comp)          # what src holds for dst (slab side)
                    _, d_pen = dst.segment(src.rank, comp)           # where dst keeps src's planes (pencil side)
                    if to_pencil:
                        d_pen.copy_(s_slab)
                    else:
                        s_slab.copy_(d_pen)
        return R

    def halos(self, ms):
        """Boundary planes of every rank's m: list of (halo_lo, halo_hi) per rank (None at an open end)."""
        out = []
        for r in self.ranks:
            lo, hi = r.halo_neighbours()
            out.append((ms[lo][:, -1].contiguous() if lo is not None else None,
                        ms[hi][:, 0].contiguous() if hi is not None else None))
        return out


class NcclTransport:
    """One process per GPU (torch.distributed, backend nccl): every (peer, component) segment is one isend and one
    irecv, batched, so each all-to-all is a single NCCL group over NVLink / NVSwitch."""

    def __init__(self, rank_ctx: SlabRank, group=None):
        import torch.distributed as dist
        self.dist, self.r, self.group = dist, rank_ctx, group

    def all_to_all(self, to_pencil: bool):
        dist, r = self.dist, self.r
        ops = []
        for peer in range(r.nranks):
            for comp in range(3):
                slab, pen = r.segment(peer, comp)
                send, recv = (slab, pen) if to_pencil else (pen, slab)
                if peer == r.rank:
                    recv.copy_(send)
                else:
                    ops.append(dist.P2POp(dist.isend, send, peer, self.group))
                    ops.append(dist.P2POp(dist.irecv, recv, peer, self.group))
        for w in (dist.batch_isend_irecv(ops) if ops else []):
            w.wait()

    def halos(self, m):
        dist, r, torch = self.dist, self.r, self.r.torch
        lo, hi = r.halo_neighbours()
        h_lo = torch.empty_like(m[:, 0]) if lo is not None else None
        h_hi = torch.empty_like(m[:, 0]) if hi is not None else None
        ops = []
        first, last = m[:, 0].contiguous(), m[:, -1].contiguous()
        if lo is not None:
            ops += [dist.P2POp(dist.isend, first, lo, self.group), dist.P2POp(dist.irecv, h_lo, lo, self.group)]
        if hi is not None:
            ops += [dist.P2POp(dist.isend, last, hi, self.group), dist.P2POp(dist.irecv, h_hi, hi, self.group)]
        for w in (dist.batch_isend_irecv(ops) if ops else []):
            w.wait()
        return h_lo, h_hi


WHAT = {"demag": 0, "heff": 1, "torque": 2}


def evaluate_local(ranks, ms, what="heff", step=0, dt_thermal=0.0):
    """One evaluation on `ranks` (all in this process), phase by phase; ms[r] is rank r's slab of m.
    Returns the list of output slabs."""
    tr = LocalTransport(ranks)
    for r, m in zip(ranks, ms):
        r.forward(m)
    tr.all_to_all(True)
    for r in ranks:
        r.mid()
    tr.all_to_all(False)
    hal = tr.halos(ms)
    outs = []
    for r, m, (lo, hi) in zip(ranks, ms, hal):
        o = r.torch.empty_like(m)
        r.backward(m, lo, hi, o, WHAT[what], step, dt_thermal)
        outs.append(o)
    return outs


def evaluate_nccl(rank_ctx, m, what="heff", step=0, dt_thermal=0.0, group=None):
    """One evaluation of this process's slab with the exchanges over NCCL."""
    tr = NcclTransport(rank_ctx, group)
    rank_ctx.forward(m)
    tr.all_to_all(True)
    rank_ctx.mid()
    tr.all_to_all(False)
    lo, hi = tr.halos(m)
    o = rank_ctx.torch.empty_like(m)
    rank_ctx.backward(m, lo, hi, o, WHAT[what], step, dt_thermal)
    return o


NSTAGES = {"rk1": 1, "rk2": 2, "rk3": 3, "rk4": 4}


def steps_fixed_local(ranks, ms, method, dt, n, step0=0):
    """n fixed steps of rk1 / rk2 / rk3 / rk4 on `ranks` (all in this process); ms[r] is updated in place."""
    tr = LocalTransport(ranks)
    for i in range(n):
        for s in range(NSTAGES[method]):
            ins = [r.stage_input(m, method, s) for r, m in zip(ranks, ms)]
            for r, x in zip(ranks, ins):
                r.forward(x)
            tr.all_to_all(True)
            for r in ranks:
                r.mid()
            tr.all_to_all(False)
            hal = tr.halos(ins)
            for r, m, (lo, hi) in zip(ranks, ms, hal):
                r.backward_stage(m, method, s, dt, step0 + i, lo, hi)


def steps_fixed_nccl(rank_ctx, m, method, dt, n, step0=0, group=None):
    """The same for this process's slab with the exchanges over NCCL."""
    tr = NcclTransport(rank_ctx, group)
    for i in range(n):
        for s in range(NSTAGES[method]):
            x = rank_ctx.stage_input(m, method, s)
            rank_ctx.forward(x)
            tr.all_to_all(True)
            rank_ctx.mid()
            tr.all_to_all(False)
            lo, hi = tr.halos(x)
            rank_ctx.backward_stage(m, method, s, dt, step0 + i, lo, hi)
