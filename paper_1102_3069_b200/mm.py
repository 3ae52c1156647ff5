"""ctypes binding of include/mm.h.  Same names as the C entry points; marshalling only.

torch is used for device memory and streams, nothing else.  There is no CPU fallback: the library
must be built (python -m paper_1102_3069_b200.build) and a CUDA device must be present for anything
but the two host-side test hooks.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.environ.get("MM_B200_LIB") or os.path.join(_HERE, "libmm_b200.so")      # override: A/B builds

MM_OK = 0
STATUS = {0: "MM_OK", 1: "MM_EINVAL", 2: "MM_ENOMEM", 3: "MM_ECUDA", 4: "MM_ESTATE",
          5: "MM_EUNSUPPORTED", 6: "MM_ENUMERIC"}
METHODS = {"rk1": 0, "rk2": 1, "rk4": 2, "rkdp": 3, "rk12": 4, "rk23": 5, "rk3": 6, "rkck": 7}


class MMError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


class Material(C.Structure):
    """mm_material of include/mm.h (SI units)."""
    _fields_ = [("Ms", C.c_double), ("Aex", C.c_double), ("alpha", C.c_double), ("gamma0", C.c_double),
                ("Ku", C.c_double), ("anis_u", C.c_double * 3), ("Bext", C.c_double * 3),
                ("T", C.c_double), ("seed", C.c_uint64), ("j", C.c_double * 3), ("P", C.c_double),
                ("xi", C.c_double), ("stt_literal_eq7", C.c_int), ("demag", C.c_int),
                ("K1", C.c_double), ("K2", C.c_double), ("exchange_in_kernel", C.c_int), ("geometry", C.c_int),
                ("anis_c1", C.c_double * 3), ("anis_c2", C.c_double * 3)]

    @classmethod
    def from_dict(cls, d, demag=True):
        m = cls()
        m.Ms = d["Ms"]; m.Aex = d.get("Aex", 0.0); m.alpha = d.get("alpha", 0.0)
        m.gamma0 = d.get("gamma0", 0.0); m.Ku = d.get("Ku", 0.0)
        m.anis_u = (C.c_double * 3)(*d.get("anis_u", (0.0, 0.0, 1.0)))
        m.Bext = (C.c_double * 3)(*d.get("Bext", (0.0, 0.0, 0.0)))
        m.T = d.get("T", 0.0); m.seed = int(d.get("seed", 0))
        m.j = (C.c_double * 3)(*d.get("j", (0.0, 0.0, 0.0)))
        m.P = d.get("P", 0.0); m.xi = d.get("xi", 0.0)
        m.stt_literal_eq7 = int(bool(d.get("stt_literal_eq7", False)))
        m.demag = int(bool(demag))
        m.K1 = d.get("K1", 0.0); m.K2 = d.get("K2", 0.0)
        m.exchange_in_kernel = int(bool(d.get("exchange_in_kernel", False)))
        m.geometry = int(bool(d.get("geometry", False)))
        m.anis_c1 = (C.c_double * 3)(*d.get("anis_c1", (1.0, 0.0, 0.0)))
        m.anis_c2 = (C.c_double * 3)(*d.get("anis_c2", (0.0, 1.0, 0.0)))
        return m


class Slab(C.Structure):
    """mm_slab of include/mm.h."""
    _fields_ = [("rank", C.c_int), ("nranks", C.c_int), ("z0", C.c_int), ("z1", C.c_int), ("kx0", C.c_int),
                ("kx1", C.c_int)]


_lib = None


def lib():
    """Load libmm_b200.so (fails loudly if it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIBPATH):
            raise MMError(3, f"{_LIBPATH} is missing: run `python -m paper_1102_3069_b200.build` "
                             "(there is no CPU fallback)")
        L = C.CDLL(_LIBPATH)
        vp, i3, d3 = C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_double)
        L.mm_create.argtypes = [C.POINTER(vp), i3, d3, i3, vp]
        L.mm_set_material.argtypes = [vp, C.POINTER(Material)]
        L.mm_demag_init.argtypes = [vp]
        for f in (L.mm_heff, L.mm_torque):
            f.argtypes = [vp, vp, vp, C.c_double, C.c_uint64, C.c_double]
        L.mm_step.argtypes = [vp, vp, C.c_int, d3, C.c_double, d3, d3, i3]
        L.mm_steps_fixed.argtypes = [vp, vp, C.c_int, C.c_double, C.c_int, d3, d3]
        L.mm_steps_fixed_host.argtypes = [vp, vp, C.c_int, C.c_double, C.c_int, d3, d3]
        L.mm_steps_adaptive.argtypes = [vp, vp, C.c_int, C.c_int, d3, C.c_double, d3, i3, d3]
        L.mm_steps_maxdm.argtypes = [vp, vp, C.c_int, C.c_double, C.c_int, d3, d3]
        L.mm_average.argtypes = [vp, vp, d3]
        L.mm_average_static.argtypes = [vp, C.c_size_t, vp, vp, C.c_char_p, C.c_size_t]
        L.mm_kernel_timing.argtypes = [vp, C.c_int]
        L.mm_kernel_times.argtypes = [vp, d3, C.POINTER(C.c_uint64)]
        L.mm_fused_eval.argtypes = [vp, vp, C.c_int, C.c_int, C.c_double, C.c_uint64]
        L.mm_reset_stepper.argtypes = [vp, C.c_uint64]
        L.mm_demag_field.argtypes = [vp, vp, vp]
        L.mm_get_demag_kernel.argtypes = [vp, C.c_int, vp, C.c_size_t]
        L.mm_demag_tensor_host.argtypes = [d3, i3, i3, C.c_size_t, vp, vp]
        L.mm_demag_khat_host.argtypes = [d3, i3, i3, vp, C.c_size_t]
        L.mm_padded_size.argtypes = [vp, i3, i3]
        L.mm_padded_size_of.argtypes = [i3, i3, i3, i3]
        L.mm_set_option.argtypes = [vp, C.c_char_p, C.c_int]
        L.mm_launch_count.argtypes = [vp]
        L.mm_launch_count.restype = C.c_uint64
        L.mm_set_fast_path.argtypes = [vp, C.c_int]
        L.mm_copy_bandwidth.argtypes = [vp, vp, vp, C.c_size_t, C.c_int, d3]
        sz = C.POINTER(C.c_size_t)
        L.mm_create_batch.argtypes = [C.POINTER(vp), i3, d3, i3, vp, C.c_int]
        L.mm_batch_set_field.argtypes = [vp, vp]
        L.mm_slab_partition.argtypes = [i3, i3, C.c_int, C.c_int, C.POINTER(Slab)]
        L.mm_create_dist.argtypes = [C.POINTER(vp), i3, d3, i3, vp, C.c_int, C.c_int]
        L.mm_dist_buffers.argtypes = [vp, C.POINTER(vp), sz, C.POINTER(vp), sz]
        L.mm_dist_segment.argtypes = [vp, C.c_int, C.c_int, sz, sz, sz, sz]
        L.mm_slab_segment.argtypes = [i3, i3, C.c_int, C.c_int, C.c_int, C.c_int, sz, sz, sz, sz]
        L.mm_dist_forward.argtypes = [vp, vp]
        L.mm_dist_mid.argtypes = [vp]
        L.mm_dist_backward.argtypes = [vp, vp, vp, vp, vp, C.c_int, C.c_uint64, C.c_double]
        L.mm_dist_stage_input.argtypes = [vp, C.c_int, C.c_int, vp, C.POINTER(vp)]
        L.mm_dist_backward_stage.argtypes = [vp, vp, C.c_int, C.c_int, C.c_double, C.c_uint64, vp, vp]
        L.mm_last_error.argtypes = [vp]
        L.mm_last_error.restype = C.c_char_p
        L.mm_destroy.argtypes = [vp]
        L.mm_destroy.restype = None
        _lib = L
    return _lib


def _i3(v):
    return (C.c_int * 3)(*[int(x) for x in v])


def _d3(v):
    return (C.c_double * 3)(*[float(x) for x in v])


def demag_tensor_host(cell, grid, pbc, offsets) -> np.ndarray:
    """mm_demag_tensor_host: the library's real-space tensor (xx,yy,zz,xy,xz,yz) at integer offsets."""
    off = np.ascontiguousarray(np.asarray(offsets, dtype=np.int64).reshape(-1, 3))
    out = np.zeros((off.shape[0], 6), dtype=np.float64)
    st = lib().mm_demag_tensor_host(_d3(cell), _i3(grid), _i3(pbc), off.shape[0],
                                    off.ctypes.data_as(C.c_void_p), out.ctypes.data_as(C.c_void_p))
    if st != MM_OK:
        raise MMError(st, "mm_demag_tensor_host")
    return out


def slab_partition(grid, pbc, nranks, rank) -> Slab:
    """mm_slab_partition: planes and spectrum columns of one rank (host only)."""
    out = Slab()
    st = lib().mm_slab_partition(_i3(grid), _i3(pbc), int(nranks), int(rank), C.byref(out))
    if st != MM_OK:
        raise MMError(st, "mm_slab_partition")
    return out


def slab_segment(grid, pbc, nranks, rank, peer, comp):
    """mm_slab_segment: (slab_off, slab_count, pencil_off, pencil_count) in complex elements (host only)."""
    v = [C.c_size_t() for _ in range(4)]
    st = lib().mm_slab_segment(_i3(grid), _i3(pbc), int(nranks), int(rank), int(peer), int(comp), *[C.byref(x) for x in v])
    if st != MM_OK:
        raise MMError(st, "mm_slab_segment")
    return tuple(int(x.value) for x in v)


AVERAGE_STATIC_MAX_CELLS = 67108864          # MM_AVERAGE_STATIC_MAX_CELLS of include/mm.h


def average_static(field, out, stream=None):
    """mm_average_static: <f> of a CUDA float32 tensor [3, ...] into the CUDA float64 tensor out[3] (caller's memory),
    through the library's fixed scratch array -- nothing is allocated on the way, no host synchronisation."""
    assert field.is_cuda and field.is_contiguous() and field.shape[0] == 3 and str(field.dtype) == "torch.float32"
    assert out.is_cuda and out.is_contiguous() and out.numel() == 3 and str(out.dtype) == "torch.float64"
    err = C.create_string_buffer(512)
    st = lib().mm_average_static(C.c_void_p(field.data_ptr()), field.numel() // 3, C.c_void_p(out.data_ptr()),
                                 C.c_void_p(stream.cuda_stream if stream is not None else 0), err, len(err))
    if st != MM_OK:
        raise MMError(st, err.value.decode())
    return out


def demag_khat_host(cell, grid, pbc) -> np.ndarray:
    """mm_demag_khat_host: K-hat octant, shape (6, Cz, Cy, Cx) float32, as uploaded by mm_demag_init."""
    P, Cs = (C.c_int * 3)(), (C.c_int * 3)()
    st = lib().mm_padded_size_of(_i3(grid), _i3(pbc), P, Cs)
    if st != MM_OK:
        raise MMError(st, "mm_padded_size_of")
    out = np.zeros((6, Cs[2], Cs[1], Cs[0]), dtype=np.float32)
    st = lib().mm_demag_khat_host(_d3(cell), _i3(grid), _i3(pbc), out.ctypes.data_as(C.c_void_p), out.size)
    if st != MM_OK:
        raise MMError(st, "mm_demag_khat_host")
    return out


class Sim:
    """One mm_ctx.  Fields are torch CUDA float32 tensors of shape (3, Nz, Ny, Nx)."""

    def __init__(self, grid, cell, pbc=(0, 0, 0), mat=None, demag=True, stream=None, demag_init=True,
                 options=None, nfilms=0):
        import torch
        self.torch = torch
        self.L = lib()
        self.grid = tuple(int(v) for v in grid)
        self.shape = (3, int(nfilms) if nfilms else self.grid[2], self.grid[1], self.grid[0])
        self.ctx = C.c_void_p()
        if torch.cuda.is_available():
            torch.cuda.init()
            s = stream if stream is not None else torch.cuda.current_stream()
            sp = C.c_void_p(s.cuda_stream)
        else:
            sp = C.c_void_p(0)
        if nfilms:                # mm_create_batch: nfilms independent films, fields (3, nfilms, Ny, Nx)
            st = self.L.mm_create_batch(C.byref(self.ctx), _i3(grid), _d3(cell), _i3(pbc), sp, int(nfilms))
        else:
            st = self.L.mm_create(C.byref(self.ctx), _i3(grid), _d3(cell), _i3(pbc), sp)
        if st != MM_OK:
            raise MMError(st, self.L.mm_last_error(None).decode())
        for k, v in (options or {}).items():
            self.set_option(k, v)
        if mat is not None:
            self.set_material(mat, demag)
        if demag_init:
            self.demag_init()

    def _chk(self, st):
        if st != MM_OK:
            raise MMError(st, self.L.mm_last_error(self.ctx).decode())

    def _dev(self, t):
        assert t.is_cuda and t.dtype == self.torch.float32 and t.is_contiguous() and tuple(t.shape) == self.shape
        return C.c_void_p(t.data_ptr())

    def set_material(self, mat, demag=True):
        m = mat if isinstance(mat, Material) else Material.from_dict(mat, demag)
        self._chk(self.L.mm_set_material(self.ctx, C.byref(m)))

    def set_option(self, key, value):
        self._chk(self.L.mm_set_option(self.ctx, key.encode(), int(value)))

    def batch_set_field(self, B):
        """One applied field (tesla) per film, array (nfilms, 3); None: the material's uniform field again."""
        if B is None:
            self._chk(self.L.mm_batch_set_field(self.ctx, C.c_void_p(0)))
            return
        b = np.ascontiguousarray(np.asarray(B, dtype=np.float64).reshape(self.shape[1], 3))
        self._chk(self.L.mm_batch_set_field(self.ctx, b.ctypes.data_as(C.c_void_p)))

    def demag_init(self):
        self._chk(self.L.mm_demag_init(self.ctx))

    def new_field(self):
        return self.torch.empty(self.shape, dtype=self.torch.float32, device="cuda")

    def heff(self, m, out=None, step=0, dt_thermal=0.0, t=0.0):
        out = self.new_field() if out is None else out
        self._chk(self.L.mm_heff(self.ctx, self._dev(m), self._dev(out), t, step, dt_thermal))
        return out

    def torque(self, m, out=None, step=0, dt_thermal=0.0, t=0.0):
        out = self.new_field() if out is None else out
        self._chk(self.L.mm_torque(self.ctx, self._dev(m), self._dev(out), t, step, dt_thermal))
        return out

    def demag_field(self, m, out=None):
        out = self.new_field() if out is None else out
        self._chk(self.L.mm_demag_field(self.ctx, self._dev(m), self._dev(out)))
        return out

    def step(self, m, method, dt, tol=1e-5, t=0.0):
        """One trial step; returns (accepted, err, dt_next, t)."""
        dtv, tv, err, acc = C.c_double(dt), C.c_double(t), C.c_double(0.0), C.c_int(0)
        self._chk(self.L.mm_step(self.ctx, self._dev(m), METHODS[method], C.byref(dtv), tol, C.byref(tv),
                                 C.byref(err), C.byref(acc)))
        return bool(acc.value), err.value, dtv.value, tv.value

    def steps_fixed(self, m, method, dt, n, t=0.0):
        tv, err = C.c_double(t), C.c_double(0.0)
        self._chk(self.L.mm_steps_fixed(self.ctx, self._dev(m), METHODS[method], dt, n, C.byref(tv),
                                        C.byref(err)))
        return tv.value, err.value

    def steps_adaptive(self, m, method, ntrials, dt, tol=1e-5, t=0.0):
        """ntrials trial steps with the step controller on the device; returns (naccepted, last_err, dt_next, t)."""
        dtv, tv, err, nacc = C.c_double(dt), C.c_double(t), C.c_double(0.0), C.c_int(0)
        self._chk(self.L.mm_steps_adaptive(self.ctx, self._dev(m), METHODS[method], int(ntrials), C.byref(dtv), tol,
                                           C.byref(tv), C.byref(nacc), C.byref(err)))
        return nacc.value, err.value, dtv.value, tv.value

    def steps_maxdm(self, m, method, max_dm, n, t=0.0):
        """n steps with dt = max_dm / max|dm/dt| each; returns (t, last_dt)."""
        tv, dtv = C.c_double(t), C.c_double(0.0)
        self._chk(self.L.mm_steps_maxdm(self.ctx, self._dev(m), METHODS[method], max_dm, int(n), C.byref(tv),
                                        C.byref(dtv)))
        return tv.value, dtv.value

    def average(self, f):
        out = (C.c_double * 3)()
        self._chk(self.L.mm_average(self.ctx, self._dev(f), out))
        return np.array([out[0], out[1], out[2]])

    def steps_fixed_host(self, m_host, method, dt, n, t=0.0):
        """m_host: CPU float32 tensor (pinned for full PCIe rate), updated in place."""
        assert (not m_host.is_cuda) and m_host.dtype == self.torch.float32 and m_host.is_contiguous()
        assert tuple(m_host.shape) == self.shape
        tv, err = C.c_double(t), C.c_double(0.0)
        self._chk(self.L.mm_steps_fixed_host(self.ctx, C.c_void_p(m_host.data_ptr()), METHODS[method], dt, n,
                                             C.byref(tv), C.byref(err)))
        return tv.value, err.value

    def kernel_timing(self, enable=True):
        self._chk(self.L.mm_kernel_timing(self.ctx, int(enable)))

    def kernel_times(self):
        sec, cnt = (C.c_double * 7)(), (C.c_uint64 * 7)()
        self._chk(self.L.mm_kernel_times(self.ctx, sec, cnt))
        names = ("fwd_x", "fwd_y", "mid", "inv_y", "inv_x", "other", "epi")
        return {n: (sec[i], int(cnt[i])) for i, n in enumerate(names)}

    def fused_eval(self, m, method, stage, dt, step=0):
        self._chk(self.L.mm_fused_eval(self.ctx, self._dev(m), METHODS[method], stage, dt, step))

    def reset_stepper(self, step_index=0):
        self._chk(self.L.mm_reset_stepper(self.ctx, step_index))

    def get_demag_kernel(self, comp):
        P, Cs = self.padded_size()
        out = np.zeros((Cs[2], Cs[1], Cs[0]), dtype=np.float32)
        self._chk(self.L.mm_get_demag_kernel(self.ctx, comp, out.ctypes.data_as(C.c_void_p), out.size))
        return out

    def padded_size(self):
        P, Cs = (C.c_int * 3)(), (C.c_int * 3)()
        self._chk(self.L.mm_padded_size(self.ctx, P, Cs))
        return tuple(P), tuple(Cs)

    def launch_count(self):
        return int(self.L.mm_launch_count(self.ctx))

    def set_fast_path(self, enable):
        self._chk(self.L.mm_set_fast_path(self.ctx, -1 if enable is True else int(enable)))

    def copy_bandwidth(self, src, dst, reps=10):
        sec = C.c_double(0.0)
        nbytes = src.numel() * src.element_size()
        self._chk(self.L.mm_copy_bandwidth(self.ctx, C.c_void_p(src.data_ptr()), C.c_void_p(dst.data_ptr()),
                                           nbytes, reps, C.byref(sec)))
        return sec.value

    def close(self):
        if self.ctx:
            self.L.mm_destroy(self.ctx)
            self.ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
