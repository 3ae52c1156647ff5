"""mm_average_static (include/mm.h): the <f> reduction without a context and without any device allocation -- its
scratch is a fixed file-scope device array of the library.  Checked against the existing path (mm_average of a
context) at the tolerance tests/test_gpu_parity.py::test_average_magnetisation uses, on two calls in a row.
Collected last on purpose (the suite runs with pytest -x); it must pass alone and after the other tests."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_1102_3069_b200 import mm as mmb              # noqa: E402
from paper_1102_3069_b200 import workloads as wlm       # noqa: E402
import mmtest_util as util                               # noqa: E402

TOL_AVG = 1e-7          # as in test_average_magnetisation


def test_average_static_matches_mm_average_on_two_calls_in_a_row():
    """Two different fields, one call after the other on one stream (the second call finds the first one's partial
    sums in the shared array), then the first field again: existing path within TOL_AVG, repeat bit for bit."""
    import torch
    # 96 x 40 x 8 = 30 720 cells = 3.75 blocks of 8192 (ragged tail); 64 x 32 x 64 = 131 072 cells = 16 blocks
    for grid in ((96, 40, 8), (64, 32, 64)):
        wl = util.small(grid, (3e-9, 4e-9, 5e-9), seed=11)
        sim = util.gpu_sim(wl)
        ma = util.to_dev(wlm.initial_m(wl))
        mb = (ma * torch.tensor([0.25, -2.0, 3.0], device="cuda").view(3, 1, 1, 1) + 0.5).contiguous()
        ref_a, ref_b = sim.average(ma), sim.average(mb)
        out_a = torch.zeros(3, dtype=torch.float64, device="cuda")
        out_b = torch.full((3,), 7.0, dtype=torch.float64, device="cuda")
        out_a2 = torch.full((3,), -1.0, dtype=torch.float64, device="cuda")
        mmb.average_static(mb, out_a2)           # (the first call on a device loads the module and looks the array up)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        mmb.average_static(ma, out_a)
        mmb.average_static(mb, out_b)
        mmb.average_static(ma, out_a2)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before                 # cudaMemGetInfo: no device memory was taken
        got_a, got_b = out_a.cpu().numpy(), out_b.cpu().numpy()
        assert np.abs(got_a - ref_a).max() <= TOL_AVG, (got_a, ref_a)
        assert np.abs(got_b - ref_b).max() <= TOL_AVG * 3.5, (got_b, ref_b)   # |f| up to 3.5 here
        assert np.array_equal(got_a, out_a2.cpu().numpy())
        # and against a plain fp64 sum of the same numbers
        assert np.abs(got_b - mb.double().reshape(3, -1).mean(dim=1).cpu().numpy()).max() <= 1e-12
        sim.close()


def test_average_static_on_a_side_stream_and_one_cell():
    import torch
    st = torch.cuda.Stream()
    f = torch.tensor([[1.5], [-2.0], [0.25]], dtype=torch.float32, device="cuda")
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        mmb.average_static(f, out, stream=st)
    st.synchronize()
    assert out.cpu().tolist() == [1.5, -2.0, 0.25]


def test_average_static_rejects_sizes_beyond_its_scratch_and_bad_arguments():
    import torch
    L = mmb.lib()
    f = torch.zeros(3, 16, dtype=torch.float32, device="cuda")
    out = torch.full((3,), 9.0, dtype=torch.float64, device="cuda")
    err = C.create_string_buffer(512)
    fp, op = C.c_void_p(f.data_ptr()), C.c_void_p(out.data_ptr())
    # one cell more than the scratch array covers: refused before anything is launched (the field is never read)
    st = L.mm_average_static(fp, mmb.AVERAGE_STATIC_MAX_CELLS + 1, op, None, err, len(err))
    assert mmb.STATUS[st] == "MM_EUNSUPPORTED"
    msg = err.value.decode()
    assert "too large" in msg and str(mmb.AVERAGE_STATIC_MAX_CELLS) in msg
    assert L.mm_average_static(fp, 0, op, None, err, len(err)) == 1 and "ncell" in err.value.decode()
    assert L.mm_average_static(None, 16, op, None, err, len(err)) == 1
    assert L.mm_average_static(fp, 16, None, None, None, 0) == 1          # no message buffer is fine
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [9.0, 9.0, 9.0]                          # nothing ran
    assert L.mm_average_static(fp, 16, op, None, err, len(err)) == 0 and err.value == b""
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [0.0, 0.0, 0.0]
