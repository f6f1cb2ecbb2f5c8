"""nh_cfl_dt_static against the context path (-m gpu).

nh_cfl_dt_static is the one entry point of the library for callers that are not allowed to allocate
device memory -- a host application whose own memory manager has taken the whole GPU, a
latency-bound loop that cannot take the device-wide stall of cudaMalloc / cudaFree, a plug-in that
may not own device memory (include/nh_b200.h).  Its reduction scratch is an array compiled into the
library and shared by all calls on a device, so what has to be shown is that (1) it returns the
time step the existing path (nh_create + nh_set_state + nh_compute_dt) returns, bit for bit as
tests/test_gpu_parity.py::test_cfl_dt_bit_exact demands of a CFL step, and (2) that this still
holds for a second call that finds the first call's leftovers in the array -- here a small, slow
state after a large, fast one, so that a stale partial maximum anywhere would shorten its dt.

The tensors below are the caller's inputs and outputs; the library itself allocates nothing.
This file sorts last on purpose: under `pytest -x` a failure here hides no other test.
"""
import numpy as np
import pytest

from paper_1706_04551_b200 import inputs

pytestmark = pytest.mark.gpu

DX, DY = 0.5, 0.4
PRM = dict(g=9.81, cfl=0.45, delta=1e-5)


def _state(nx, ny, seed, speedup):
    s = inputs.random_smooth_state(nx, ny, DX, DY, seed=seed, depth=1.0, dry_fraction=0.2)
    s["qx"] = s["qx"] * speedup
    s["qy"] = s["qy"] * speedup
    return s


def _dt_context_path(nh, s, nx, ny):
    g = nh.NH(nx, ny, DX, DY, s["H"], **PRM)
    g.set_state(s["h"], s["qx"], s["qy"], s["w"], s["p"])
    dt = g.compute_dt()
    g.close()
    return dt


def test_two_calls_in_a_row_match_the_context_path():
    import torch
    from paper_1706_04551_b200 import nh
    nh.lib()
    dev = torch.device("cuda:0")
    big = (701, 297)     # 51 partial maxima, ragged last CTA
    small = (133, 21)    # 1 partial maximum: slots 1..50 still hold the first call's values
    sa, sb = _state(*big, seed=11, speedup=40.0), _state(*small, seed=5, speedup=1.0)
    want_a, want_b = _dt_context_path(nh, sa, *big), _dt_context_path(nh, sb, *small)
    assert 0.0 < want_a < want_b          # the leftovers are the dangerous kind

    ta = [torch.from_numpy(np.ascontiguousarray(sa[k])).to(dev) for k in ("h", "qx", "qy")]
    tb = [torch.from_numpy(np.ascontiguousarray(sb[k])).to(dev) for k in ("h", "qx", "qy")]
    out_a = torch.full((1,), -1.0, dtype=torch.float64, device=dev)
    out_b = torch.full((1,), -1.0, dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream()
    # the first call on a device is the set-up call (it looks up the address of the built-in array,
    # and the CUDA runtime loads the module's code then); its result counts like any other
    nh.cfl_dt_static(*tb, out_b, DX, DY, stream=stream, **PRM)
    torch.cuda.synchronize()
    assert out_b.item() == want_b
    out_b.fill_(-1.0)
    torch.cuda.synchronize()
    mem_before = torch.cuda.mem_get_info()[0]
    nh.cfl_dt_static(*ta, out_a, DX, DY, stream=stream, **PRM)   # call 1
    nh.cfl_dt_static(*tb, out_b, DX, DY, stream=stream, **PRM)   # call 2, same stream, no sync between
    torch.cuda.synchronize()
    mem_after = torch.cuda.mem_get_info()[0]
    assert out_a.item() == want_a
    assert out_b.item() == want_b
    assert mem_after >= mem_before        # the device's free memory did not shrink across the two calls
    # and once more the other way round (large after small)
    out_a.fill_(-1.0)
    nh.cfl_dt_static(*ta, out_a, DX, DY, stream=stream, **PRM)
    torch.cuda.synchronize()
    assert out_a.item() == want_a


def test_refuses_what_it_cannot_do():
    import torch
    from paper_1706_04551_b200 import nh
    dev = torch.device("cuda:0")
    limit = nh.cfl_dt_static_max_cells()
    assert limit == 8192 * 8192
    z = torch.zeros((4, 4), dtype=torch.float64, device=dev)
    out = torch.full((1,), -1.0, dtype=torch.float64, device=dev)
    L = nh.lib()
    # one row more than the built-in scratch covers: refused before anything is launched
    st = L.nh_cfl_dt_static(8192, 8193, DX, DY, 9.81, 0.5, 1e-5, z.data_ptr(), z.data_ptr(), z.data_ptr(),
                            out.data_ptr(), None)
    assert st == nh.EINVAL
    msg = L.nh_static_last_error().decode()
    assert "exceed" in msg and str(limit) in msg
    # host arrays are refused instead of being handed to a kernel
    hz = np.zeros((4, 4))
    with pytest.raises(nh.NHError) as e:
        nh.cfl_dt_static(hz, hz, hz, out, DX, DY)
    assert e.value.code == nh.EINVAL and "device pointers" in str(e.value)
    torch.cuda.synchronize()
    assert out.item() == -1.0             # neither refusal wrote the output
    # still water: every wet cell moves at sqrt(g h) only; all dry: no rate at all -> dt = 0
    h1 = torch.ones((4, 4), dtype=torch.float64, device=dev)
    nh.cfl_dt_static(h1, z, z, out, DX, DY, g=9.81, cfl=0.5)
    torch.cuda.synchronize()
    c = np.sqrt(9.81 * 1.0)
    assert out.item() == 0.5 / (c / DX + c / DY)
    nh.cfl_dt_static(z, z, z, out, DX, DY)
    torch.cuda.synchronize()
    assert out.item() == 0.0
