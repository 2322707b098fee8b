"""kratos_hydro_totals_static: the conserved totals for a program that cannot let this library allocate.

Who needs it: a host application that has given the whole GPU to its own memory pool (a mesh manager, a tensor
library's caching allocator), so that a later cudaMalloc from a guest library fails or steals pages; and code that
runs between the steps of a live simulation, where the device-wide wait inside cudaMalloc / cudaFree would stall every
stream.  Every other entry point needs a handle, and creating a handle allocates.  This one takes the caller's own
device buffer and keeps its partial sums in an array compiled into the library (include/kratos_hydro.h, "Conserved
totals without any allocation").

What is checked: the call gives what the handle-based kratos_hydro_totals gives for the same state -- on two calls in a
row that share the built-in array, the second on a much smaller state, so that the slots the first call filled and the
second does not use are still there, stale, when the second one sums up.  Then the output-on-device form, the refusal
of a state larger than the stated maximum, and that the device's free memory does not move across a call.

This file is named to be collected last: under `pytest -x` a failure here must not hide another test.
"""
import ctypes
import math

import numpy as np
import pytest

from paper_2501_02317_b200 import binding, inputs

# what tests/test_gpu_parity.py::test_state_roundtrip_and_totals allows between the totals kernels and math.fsum
RTOL_TOTALS = 2e-16


def _handle_totals(pr):
    """The existing path: a handle (which allocates), set_state, kratos_hydro_totals."""
    nx, ny, nz = pr.shape
    h = binding.KratosHydro(nx, ny, nz, pr.gamma, pr.bc, precision=binding.PREC_FP64)
    h.set_state(pr.U)
    tot = h.totals()
    h.destroy()
    return tot


def test_totals_static_refuses_a_state_beyond_its_maximum():
    """ncell is checked before anything touches the GPU, so this runs on any box: no kernel sees the fake address."""
    L = binding.load()
    out = (ctypes.c_double * 5)()
    fake = ctypes.c_void_p(256)
    for ncell in (binding.TOTALS_STATIC_MAX_CELLS + 1, 0, -7):
        rc = L.kratos_hydro_totals_static(fake, ncell, ctypes.cast(out, ctypes.c_void_p), 0, None)
        assert rc == binding.ERR_ARG
        assert "KRATOS_TOTALS_STATIC_MAX_CELLS" in binding.last_error()
    assert L.kratos_hydro_totals_static(None, 16, ctypes.cast(out, ctypes.c_void_p), 0, None) == binding.ERR_ARG
    assert L.kratos_hydro_totals_static(fake, 16, None, 0, None) == binding.ERR_ARG


@pytest.mark.gpu
def test_totals_static_matches_the_handle_path_on_two_calls_in_a_row():
    import torch

    # 1st state: 3 091 487 cells -> the full grid of 592 blocks, some twenty strides per thread, a ragged tail (N is odd);
    # 2nd state: 6 993 cells -> 28 blocks: 564 slots per field keep the first call's partial sums.
    big = inputs.random_smooth(203, 157, 97, seed=11)
    small = inputs.random_smooth(37, 21, 9, seed=1)
    want_big, want_small = _handle_totals(big), _handle_totals(small)

    Ub = torch.from_numpy(big.U).cuda()
    Us = torch.from_numpy(small.U).cuda()
    got_big = binding.totals_static(Ub)          # first call: also the one-time look-up of the array's address
    got_small = binding.totals_static(Us)        # second call, same array, nothing cleared in between
    for got, want, pr in ((got_big, want_big, big), (got_small, want_small, small)):
        np.testing.assert_allclose(got, want, rtol=RTOL_TOTALS, atol=1e-300)
        exact = np.array([math.fsum(pr.U[m].ravel()) for m in range(5)])
        np.testing.assert_allclose(got, exact, rtol=RTOL_TOTALS, atol=1e-300)
    # same kernels, same grid, same order of summation: in fact the very same bits
    np.testing.assert_array_equal(got_big, want_big)
    np.testing.assert_array_equal(got_small, want_small)

    # and back to the big one: whatever the small call left behind does not matter either
    np.testing.assert_array_equal(binding.totals_static(Ub), want_big)


@pytest.mark.gpu
def test_totals_static_result_on_the_device_and_on_a_side_stream():
    import torch

    pr = inputs.random_smooth(64, 48, 20, seed=3)
    want = _handle_totals(pr)
    U = torch.from_numpy(pr.U).cuda()
    out = torch.full((5,), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        ret = binding.totals_static(U, out=out)      # asynchronous on s (torch's current stream)
    s.synchronize()
    assert ret is out
    np.testing.assert_array_equal(out.cpu().numpy(), want)
    # a host pointer where a device pointer was promised (and the reverse) is refused, not dereferenced
    L = binding.load()
    host = (ctypes.c_double * 5)()
    assert L.kratos_hydro_totals_static(ctypes.c_void_p(U.data_ptr()), pr.U.size // 5, ctypes.cast(host, ctypes.c_void_p), 1, None) == binding.ERR_ARG
    assert L.kratos_hydro_totals_static(ctypes.cast(host, ctypes.c_void_p), 1, ctypes.cast(host, ctypes.c_void_p), 0, None) == binding.ERR_ARG


@pytest.mark.gpu
def test_totals_static_leaves_the_free_device_memory_where_it_was():
    import torch

    pr = inputs.random_smooth(96, 64, 32, seed=5)
    U = torch.from_numpy(pr.U).cuda()
    out = torch.empty(5, dtype=torch.float64, device="cuda")
    first = binding.totals_static(U)              # set-up and lazy loading of the two kernels happen here
    binding.totals_static(U, out=out)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        again = binding.totals_static(U)
        binding.totals_static(U, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
    np.testing.assert_array_equal(again, first)
    np.testing.assert_array_equal(out.cpu().numpy(), first)
