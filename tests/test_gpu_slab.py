"""Row f-4: one block advanced as z slabs that exchange their ghost planes through communication
boundaries (Sec. 3.1.2, :189-191; Table 2's two-GPU splits, :408-427).  On the single GPU of the test box all
slabs live in one process and advance in lock step on one stream: the same kernels, the same stores into the
neighbours' ghost arrays and the same sequence of C-ABI calls as with one process per GPU (paper_2501_02317_b200/slab.py).
The z-slab seams of the TMA kernel are bitwise invariant and the time step is a maximum over the same cells, so the
decomposed run must reproduce the undivided block BIT FOR BIT."""
import numpy as np
import pytest

import oracle
from paper_2501_02317_b200 import binding, inputs
from paper_2501_02317_b200.slab import SlabDecomposition, SlabSolver
from parity_utils import MIXED, assert_parity

pytestmark = pytest.mark.gpu

P, F, O, R, C = binding.BC_PERIODIC, binding.BC_FREE, binding.BC_OUTFLOW, binding.BC_REFLECT, binding.BC_COMM

CASES = [
    ((64, 32, 24), (P, P, P, P, P, P), 2),     # periodic in z: both faces of both slabs are cuts, the neighbours wrap
    ((64, 32, 24), (P, P, P, P, P, P), 3),
    ((32, 16, 22), (F, O, R, R, F, R), 2),     # physical boundaries at the ends, one cut; 11 + 11 planes
    ((64, 48, 23), (R, R, P, P, O, O), 4),     # uneven slabs: 6 + 6 + 6 + 5 planes
    ((96, 32, 16), (P, P, F, F, P, P), 4),     # slabs of the minimum height: 4 planes, both of each slab's pairs distinct
]


def undivided(pr, nsteps, p_ref):
    nx, ny, nz = pr.shape
    h = binding.KratosHydro(nx, ny, nz, pr.gamma, pr.bc, precision=MIXED)
    h.set_state(pr.U)
    h.set_reference_pressure(p_ref)     # what the decomposed run agreed on (reading S17)
    T0 = h.totals()
    t = h.run(pr.cfl, nsteps)
    U, T1, hits = h.get_state(), h.totals(), h.floor_hits()
    h.destroy()
    return U, t, T0, T1, hits


@pytest.mark.parametrize("shape,bc,world", CASES)
def test_slabs_reproduce_the_undivided_block_bit_for_bit(shape, bc, world):
    nx, ny, nz = shape
    pr = inputs.random_smooth(nx, ny, nz, seed=11 + world, bc=bc, gamma=1.4)
    nsteps = 6
    s = SlabSolver(nx, ny, nz, pr.gamma, pr.bc, world=world)
    s.set_state(pr.U)
    T0 = s.totals()
    t = s.run(pr.cfl, nsteps)
    Us, T1, hits = s.get_state_global(), s.totals(), s.floor_hits()
    launches = s.launch_count()
    p_ref = s.p_ref
    s.destroy()
    Uu, tu, T0u, T1u, hits_u = undivided(pr, nsteps, p_ref)
    assert hits == 0 and hits_u == 0 and launches >= 2 * nsteps * world
    assert t == tu                                   # the same sequence of time steps
    assert np.array_equal(Us, Uu)                    # bit for bit
    assert np.allclose(T0, T0u, rtol=1e-13, atol=1e-9) and np.allclose(T1, T1u, rtol=1e-13, atol=1e-9)   # sums of per-slab sums
    # and the undivided block is the oracle's (so the decomposed one is too)
    Uo = pr.U.copy()
    oracle.run(Uo, pr.gamma, pr.bc, pr.cfl, nsteps)
    assert_parity(Us, Uo, MIXED, what=f"slabs {shape} x{world}")
    if all(b == P for b in bc):
        scale = np.maximum(np.abs(T0), np.abs(pr.U).reshape(5, -1).sum(axis=1))
        assert np.all(np.abs(T1 - T0) <= 1e-13 * scale)


def test_two_runs_in_a_row_and_a_new_state():
    """run() twice equals run() once (the rate left by the last stage 2 is a slab's own: it is reduced again), and
    set_state re-establishes the ghost planes and the common reference pressure."""
    nx, ny, nz = 64, 32, 20
    bc = (P,) * 6
    pr = inputs.random_smooth(nx, ny, nz, seed=5, bc=bc, gamma=5.0 / 3.0)
    s = SlabSolver(nx, ny, nz, pr.gamma, pr.bc, world=2)
    s.set_state(pr.U)
    t = s.run(pr.cfl, 3)
    t = s.run(pr.cfl, 2, t)
    Ua = s.get_state_global()
    s.set_state(pr.U)
    t2 = s.run(pr.cfl, 5)
    Ub = s.get_state_global()
    dt_all = s.cfl_dt(0.4)
    s.destroy()
    assert t == t2 and np.array_equal(Ua, Ub)
    assert dt_all == pytest.approx(oracle.cfl_dt(Ub, pr.gamma, 0.4), rel=1e-13)


def test_communication_boundaries_are_refused_where_they_cannot_be_served():
    with pytest.raises(binding.KratosError):       # x faces: no
        binding.KratosHydro(64, 32, 16, 1.4, (C, C, P, P, P, P))
    with pytest.raises(binding.KratosError):       # not a TMA block
        binding.KratosHydro(40, 32, 16, 1.4, (P, P, P, P, C, C))
    with pytest.raises(binding.KratosError):       # all-fp64
        binding.KratosHydro(64, 32, 16, 1.4, (P, P, P, P, C, C), precision=binding.PREC_FP64)
    with pytest.raises(binding.KratosError):       # van Leer
        binding.KratosHydro(64, 32, 16, 1.4, (P, P, P, P, C, C), integrator=binding.INTEGRATOR_VANLEER)
    h = binding.KratosHydro(64, 32, 16, 1.4, (P, P, P, P, F, C))
    try:
        assert h.get_kernel() == binding.KERNEL_TMA
        with pytest.raises(binding.KratosError):   # a whole step needs the neighbours between its stages
            h.step(1e-3)
        with pytest.raises(binding.KratosError):
            h.run(0.4, 1)
        with pytest.raises(binding.KratosError):   # the low face is physical
            h.ghost_array(0, 0)
        assert h.ghost_array(0, 1) != 0 and len(h.ghost_ipc_handle(1, 1)) == 64
        h.set_state(np.ones((5, 16, 32, 64)) * np.array([1.0, 0, 0, 0, 2.5]).reshape(5, 1, 1, 1))
        h.begin_run(0.4, 0.0)
        h.substep(binding.PHASE_PREPARE)
        with pytest.raises(binding.KratosError):   # no peer yet
            h.substep(binding.PHASE_STAGE1)
        with pytest.raises(binding.KratosError):
            h.set_kernel(binding.KERNEL_SIMPLE)
    finally:
        h.destroy()


def test_substeps_equal_run_on_a_block_without_cuts():
    pr = inputs.random_smooth(64, 32, 12, seed=2, bc=(P, P, F, F, R, O), gamma=1.4)
    nx, ny, nz = pr.shape
    out = []
    for pieces in (False, True):
        h = binding.KratosHydro(nx, ny, nz, pr.gamma, pr.bc, precision=MIXED)
        h.set_state(pr.U)
        if pieces:
            h.begin_run(pr.cfl, 0.0)
            for _ in range(4):
                h.substep(binding.PHASE_PREPARE)
                h.substep(binding.PHASE_STAGE1)
                h.substep(binding.PHASE_STAGE2)
            t, n = h.end_run()
            assert n == 4
        else:
            t = h.run(pr.cfl, 4)
        out.append((t, h.get_state()))
        h.destroy()
    assert out[0][0] == out[1][0] and np.array_equal(out[0][1], out[1][1])


def test_state_through_torch_tensors():
    """set_state from a pinned host tensor (one H2D copy, slabs cut on the device) and get_state_into (slabs joined on the
    device, one D2H copy) move exactly the bytes the numpy path moves."""
    import torch
    nx, ny, nz = 64, 32, 18
    pr = inputs.random_smooth(nx, ny, nz, seed=4, bc=(P,) * 6, gamma=1.4)
    s = SlabSolver(nx, ny, nz, pr.gamma, pr.bc, world=3)
    host = torch.from_numpy(pr.U.copy()).pin_memory()
    s.set_state(host)
    out = torch.empty_like(host).pin_memory()
    s.get_state_into(out)
    assert np.array_equal(out.numpy(), pr.U)
    s.run(pr.cfl, 2)
    a = s.get_state_global()
    s.get_state_into(out)
    assert np.array_equal(out.numpy(), a)
    s.destroy()


# --------------------------------------------------------------------------- one process per slab (the deployment layout)
def _ipc_worker(rank, world, port, shape, bc, nsteps, out, backend="gloo"):
    import os
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    # gloo: all ranks on GPU 0 (NCCL refuses two ranks on one GPU; the test box has one).  nccl: one GPU per rank.
    torch.cuda.set_device(rank if backend == "nccl" else 0)
    dist.init_process_group(backend, rank=rank, world_size=world)
    try:
        nx, ny, nz = shape
        pr = inputs.random_smooth(nx, ny, nz, seed=31, bc=bc, gamma=1.4)
        s = SlabSolver(nx, ny, nz, pr.gamma, pr.bc)                # distributed: this process owns the slab of its rank
        assert s.ranks == [rank] and s.world == world
        s.set_state(pr.U)
        t = s.run(pr.cfl, nsteps)
        U = s.get_state_global()
        out.put((rank, t, U, s.p_ref, s.floor_hits()))
        dist.barrier()
        s.destroy()
    finally:
        dist.destroy_process_group()


def _device_count():
    import torch
    return torch.cuda.device_count()


@pytest.mark.parametrize("shape,bc,world", [((64, 32, 24), (P, P, P, P, P, P), 2), ((32, 32, 21), (F, F, R, R, O, R), 2)])
def test_one_process_per_gpu_over_nccl(shape, bc, world):
    """The deployment itself: one process and one GPU per slab, NCCL for the rate maximum and the ordering token (both
    enqueued on the kernels' stream: no host round trip), the stage kernels' TMA stores landing in the neighbour GPU's
    ghost arrays over NVLink.  Needs `world` GPUs: skipped on the one-GPU test box, where the gloo test below covers the
    same calls."""
    if _device_count() < world:
        pytest.skip("needs %d CUDA devices, this box has %d" % (world, _device_count()))
    test_one_process_per_slab_through_cuda_ipc(shape, bc, world, backend="nccl")


@pytest.mark.parametrize("shape,bc,world", [((64, 32, 24), (P, P, P, P, P, P), 2), ((32, 32, 21), (F, F, R, R, O, R), 3)])
def test_one_process_per_slab_through_cuda_ipc(shape, bc, world, backend="gloo"):
    """The layout of a multi-GPU run -- one process per slab, the neighbours' ghost arrays mapped through CUDA IPC handles
    (kratos_hydro_ghost_ipc_handle / open_peer), reductions and ordering through the process group -- on the one GPU of the
    test box: the processes share it, no kernel waits for another (the host drains the stream before every collective).
    Bit for bit the undivided block."""
    import socket
    import torch.multiprocessing as mp
    nsteps = 4
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_ipc_worker, args=(r, world, port, shape, bc, nsteps, out, backend)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((out.get(timeout=300) for _ in range(world)), key=lambda x: x[0])
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    nx, ny, nz = shape
    pr = inputs.random_smooth(nx, ny, nz, seed=31, bc=bc, gamma=1.4)
    Uu, tu, _, _, hits_u = undivided(pr, nsteps, res[0][3])
    for rank, t, U, p_ref, hits in res:
        assert p_ref == res[0][3] and hits == 0 and hits_u == 0
        assert t == tu
        assert np.array_equal(U, Uu)
