"""paper_2501_02317_b200/outofcore.py: one Heun step of a host-resident block, streamed through the GPU in z chunks with
four planes of overlap (the step's domain of dependence).  Every returned plane must equal the undivided step bit for bit
(same reference pressure; the z seams of the TMA kernel are bitwise invisible), whatever the chunk height and the z rule."""
import numpy as np
import pytest
import torch

import oracle
from paper_2501_02317_b200 import binding, inputs
from paper_2501_02317_b200.outofcore import HALO, HostStepper
from parity_utils import MIXED, assert_parity

pytestmark = pytest.mark.gpu
P, F, O, R = binding.BC_PERIODIC, binding.BC_FREE, binding.BC_OUTFLOW, binding.BC_REFLECT


@pytest.mark.parametrize("chunk", [3, 8, 13, 64])
@pytest.mark.parametrize("shape,bc", [((64, 32, 40), (P, P, P, P, P, P)), ((32, 32, 37), (F, O, R, R, R, O))])
def test_streamed_step_equals_the_in_core_step_bit_for_bit(shape, bc, chunk):
    nx, ny, nz = shape
    pr = inputs.random_smooth(nx, ny, nz, seed=chunk + nz, bc=bc, gamma=1.4)
    h = binding.KratosHydro(nx, ny, nz, pr.gamma, pr.bc, precision=MIXED)
    h.set_state(pr.U)
    p_ref = h.get_reference_pressure()
    a = torch.from_numpy(pr.U.copy()).pin_memory()
    b = torch.empty_like(a).pin_memory()
    st = HostStepper(nx, ny, nz, pr.gamma, pr.bc, chunk=chunk, p_ref=p_ref)
    Uo = pr.U.copy()
    for _ in range(3):                       # three steps, ping-pong between the two host buffers
        dt = h.cfl_dt(0.4)
        h.step(dt)
        st.step(a, b, dt)
        oracle.step(Uo, pr.gamma, pr.bc, dt)
        a, b = b, a
    Uin = h.get_state()
    assert st.launch_count() > 0
    h.destroy()
    st.destroy()
    np.testing.assert_array_equal(a.numpy().reshape(Uin.shape), Uin)
    assert_parity(a.numpy().reshape(Uin.shape), Uo, MIXED, what=f"streamed {shape} chunk {chunk}")


def test_plan_covers_the_block_once_and_takes_the_halo_along():
    st = HostStepper(32, 16, 30, 1.4, (P, P, P, P, F, R), chunk=8, p_ref=1.0)
    plan = st.plan()
    assert [p[:2] for p in plan] == [(0, 8), (8, 16), (16, 24), (24, 30)]
    assert plan[0][2:] == (0, 8 + HALO, F, F) and plan[1][2:] == (8 - HALO, 16 + HALO, F, F)
    assert plan[3][2:] == (24 - HALO, 30, F, R)                  # the domain's own rule at its end
    st.destroy()
    sp = HostStepper(32, 16, 30, 1.4, (P,) * 6, chunk=16, p_ref=1.0)
    assert sp.plan()[0][2:4] == (-HALO, 16 + HALO) and sp._runs(-HALO, 3) == [(26, 4), (0, 3)]
    assert sp._runs(28, 34) == [(28, 2), (0, 4)]
    sp.destroy()


def test_streamed_step_takes_the_callers_cell_sizes():
    """A block that is not the unit box (dx != 1/nx): the chunk handles must use the whole block's cell sizes.  With the
    default spacing the streamed step would silently integrate another problem; with the caller's it is the in-core step."""
    nx, ny, nz = 32, 32, 24
    spacing = (0.37 / nx, 2.0 / ny, 1.3 / nz)
    pr = inputs.random_smooth(nx, ny, nz, seed=77, bc=(P, P, R, R, F, O), gamma=1.4)
    h = binding.KratosHydro(nx, ny, nz, pr.gamma, pr.bc, precision=MIXED, spacing=spacing)
    h.set_state(pr.U)
    p_ref = h.get_reference_pressure()
    dt = h.cfl_dt(0.4)
    h.step(dt)
    Uin = h.get_state()
    h.destroy()
    a = torch.from_numpy(pr.U.copy()).pin_memory()
    got = {}
    for name, sp in (("given", spacing), ("default", None)):
        b = torch.empty_like(a).pin_memory()
        st = HostStepper(nx, ny, nz, pr.gamma, pr.bc, chunk=7, p_ref=p_ref, spacing=sp)
        st.step(a, b, dt)
        st.destroy()
        got[name] = b.numpy().reshape(Uin.shape).copy()
    np.testing.assert_array_equal(got["given"], Uin)
    assert not np.array_equal(got["default"], Uin)
    Uo = pr.U.copy()
    oracle.step(Uo, pr.gamma, pr.bc, dt, spacing)
    assert_parity(got["given"], Uo, MIXED, what="streamed step on a non-unit box")
