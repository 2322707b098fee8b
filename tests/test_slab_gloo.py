"""Row f-4, host side: the z-slab decomposition and its driver (paper_2501_02317_b200/slab.py)
with world_size-2 and -3 gloo process groups on CPU.

The CUDA blocks deliver their ghost planes from inside the stage kernels through peer memory; that cannot run here.
What runs here is everything else: which planes a rank owns, who its neighbours are, which of the neighbour's planes are
its ghosts (periodic wrap included), what its boundary codes become, and the driver's sequence (common reference
pressure, initial halo push, rate all-reduce(max), PREPARE / STAGE1 / sync / STAGE2) -- with a stand-in block that
evaluates the stages with the ORACLE on its slab padded by its ghost planes and ships its boundary planes with gloo
send / recv.  The decomposed oracle run must equal the undivided oracle run (to the last bits: the only difference is
1 / (1 / rate) in the stand-in's rate), so a wrong plane index, neighbour, side or ordering fails."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_2501_02317_b200 import binding, inputs
from paper_2501_02317_b200.slab import SlabDecomposition, SlabSolver

P, F, O, R, C = binding.BC_PERIODIC, binding.BC_FREE, binding.BC_OUTFLOW, binding.BC_REFLECT, binding.BC_COMM


# --------------------------------------------------------------------------- the bookkeeping alone
def test_planes_partition_the_block_and_neighbours_wrap():
    for nz, world in ((24, 2), (23, 4), (16, 4), (100, 7)):
        d = SlabDecomposition(nz, world, P, P)
        spans = [d.planes(r) for r in range(world)]
        assert spans[0][0] == 0 and spans[-1][1] == nz
        assert all(spans[r][1] == spans[r + 1][0] for r in range(world - 1))
        sizes = [b - a for a, b in spans]
        assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
        for r in range(world):
            assert d.neighbours(r) == ((r - 1) % world, (r + 1) % world)
            assert d.local_bc(r, (F, O, R, R, P, P)) == (F, O, R, R, C, C)
            for side in (0, 1):
                nb, glob, loc = d.ghost_source(r, side)
                z0, z1 = spans[r]
                assert glob == ([(z0 - 2) % nz, (z0 - 1) % nz] if side == 0 else [z1 % nz, (z1 + 1) % nz])
                n0, n1 = spans[nb]
                assert all(n0 <= g < n1 for g in glob) and loc == [g - n0 for g in glob]
                # the neighbour's planes next to ITS other face: what its stage kernels store into my ghost array
                assert loc == ([n1 - n0 - 2, n1 - n0 - 1] if side == 0 else [0, 1])


def test_physical_ends_keep_their_boundary_codes():
    d = SlabDecomposition(22, 3, F, R)
    assert d.neighbours(0) == (None, 1) and d.neighbours(1) == (0, 2) and d.neighbours(2) == (1, None)
    bc = (P, P, O, O, F, R)
    assert d.local_bc(0, bc) == (P, P, O, O, F, C)
    assert d.local_bc(1, bc) == (P, P, O, O, C, C)
    assert d.local_bc(2, bc) == (P, P, O, O, C, R)
    assert d.ghost_source(0, 0) is None and d.ghost_source(2, 1) is None
    one = SlabDecomposition(22, 1, P, P)
    assert one.neighbours(0) == (None, None) and one.local_bc(0, (P,) * 6) == (P,) * 6
    with pytest.raises(ValueError):
        SlabDecomposition(10, 3, P, P)       # 3 planes per slab
    with pytest.raises(ValueError):
        SlabDecomposition(16, 2, P, F)


def test_scatter_and_gather_are_inverse():
    U = np.arange(5 * 11 * 2 * 3, dtype=np.float64).reshape(5, 11, 2, 3)
    d = SlabDecomposition(11, 2, F, F)
    parts = {r: d.scatter(U, r) for r in range(2)}
    assert parts[0].shape[1] == 6 and parts[1].shape[1] == 5 and parts[1].flags.c_contiguous
    assert np.array_equal(d.gather(parts), U)


# --------------------------------------------------------------------------- the driver, with an oracle-backed stand-in block
class OracleBlock:
    """Stand-in for binding.KratosHydro with the interface slab.SlabSolver uses.  Test infrastructure (it calls the oracle)."""
    wires_itself = True
    tensor_device = "cpu"

    def __init__(self, rank, shape, gamma, bc, dec, spacing):
        self.rank, self.gamma, self.bc, self.dec, self.spacing = rank, gamma, tuple(bc), dec, spacing
        nx, ny, nz = shape
        self.U = np.zeros((5, nz, ny, nx))
        self.U1 = np.zeros_like(self.U)
        self.ghost = {(a, s): np.zeros((5, 2, ny, nx)) for a in (0, 1) for s in (0, 1)}
        self.rate = self.dt = self.t = 0.0
        self.cfl = 0.0
        self.steps = self.launches = 0
        self.p_ref = None

    # ghost planes of state array `a` <- the neighbours' planes next to the common face (what the CUDA kernels store themselves)
    def deliver(self, a):
        src = self.U if a == 0 else self.U1
        nz = src.shape[1]
        reqs, bufs = [], {}
        for side, nb in enumerate(self.dec.neighbours(self.rank)):
            if nb is None:
                continue
            mine = torch.from_numpy(np.ascontiguousarray(src[:, :2] if side == 0 else src[:, nz - 2:]))
            reqs.append(dist.isend(mine, nb, tag=10 * a + (1 - side)))      # into the neighbour's ghosts beyond its OTHER face
            bufs[side] = torch.empty(self.ghost[(a, side)].shape, dtype=torch.float64)
            reqs.append(dist.irecv(bufs[side], nb, tag=10 * a + side))
        for q in reqs:
            q.wait()
        for side, b in bufs.items():
            self.ghost[(a, side)][...] = b.numpy()

    def flux_divergence(self, a):
        src = self.U if a == 0 else self.U1
        lo, hi = self.bc[4] == C, self.bc[5] == C
        parts = ([self.ghost[(a, 0)]] if lo else []) + [src] + ([self.ghost[(a, 1)]] if hi else [])
        pad = np.ascontiguousarray(np.concatenate(parts, axis=1))
        bc = list(self.bc)
        bc[4] = F if lo else bc[4]        # beyond the ghost planes nothing is read by the interior cells' stencil
        bc[5] = F if hi else bc[5]
        L, hits = oracle.flux_divergence(pad, self.gamma, bc, self.spacing)
        z0 = 2 if lo else 0
        return L[:, z0:z0 + src.shape[1]]

    def local_rate(self):
        return 1.0 / oracle.cfl_dt(self.U, self.gamma, 1.0, self.spacing)

    # -- the interface
    def set_state(self, U):
        self.U[...] = U
        self.rate = None

    def get_state(self):
        return self.U.copy()

    def get_reference_pressure(self):
        return 1.0 + self.rank       # (unused by the oracle; the driver must agree on the smallest)

    def set_reference_pressure(self, p):
        self.p_ref = p

    def push_halo(self):
        self.deliver(0)

    def begin_run(self, cfl, t0):
        self.cfl, self.t, self.steps = cfl, t0, 0
        if self.rate is None:
            self.rate = self.local_rate()

    def get_rate(self, out):
        out[0] = self.rate
        return out

    def set_rate(self, t):
        self.rate = float(t[0])

    def substep(self, phase):
        self.launches += 1
        if phase == binding.PHASE_PREPARE:
            self.dt = self.cfl / self.rate
            self.t += self.dt
            self.steps += 1
        elif phase == binding.PHASE_STAGE1:
            self.U1[...] = self.U + self.dt * self.flux_divergence(0)
            self.deliver(1)
        else:
            self.U[...] = 0.5 * self.U + 0.5 * (self.U1 + self.dt * self.flux_divergence(1))
            self.deliver(0)
            self.rate = self.local_rate()

    def end_run(self):
        return self.t, self.steps

    def cfl_dt(self, cfl):
        return cfl / self.local_rate()

    def totals(self):
        return oracle.totals(self.U)

    def floor_hits(self):
        return 0

    def launch_count(self):
        return self.launches

    def destroy(self):
        pass


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, shape, bc, nsteps, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        nx, ny, nz = shape
        pr = inputs.random_smooth(nx, ny, nz, seed=21, bc=bc, gamma=1.4)
        spacing = (1.0 / nx, 1.0 / ny, 1.0 / nz)
        holder = {}

        def make_block(r, shp, gamma, bc_r):
            return OracleBlock(r, shp, gamma, bc_r, holder["dec"], spacing)

        holder["dec"] = SlabDecomposition(nz, world, bc[4], bc[5])
        s = SlabSolver(nx, ny, nz, pr.gamma, pr.bc, make_block=make_block)
        assert s.world == world and s.ranks == [rank]
        # world 3: the whole block as a (host) torch tensor -- a rank must move the planes it owns and no others
        s.set_state(torch.from_numpy(pr.U) if world == 3 else pr.U)
        z0, z1 = s.dec.planes(rank)
        assert s.last_upload_bytes == 5 * 8 * nx * ny * (z1 - z0)
        t = s.run(pr.cfl, nsteps)
        U = s.get_state_global()
        out.put((rank, t, U, s.p_ref, s.totals(), s.cfl_dt(0.4)))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("shape,bc,world", [((12, 10, 16), (P,) * 6, 2), ((8, 6, 14), (F, O, R, R, O, R), 3)])
def test_decomposed_oracle_run_equals_the_undivided_one(shape, bc, world):
    nsteps = 3
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, shape, bc, nsteps, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((out.get(timeout=300) for _ in range(world)), key=lambda x: x[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    nx, ny, nz = shape
    pr = inputs.random_smooth(nx, ny, nz, seed=21, bc=bc, gamma=1.4)
    Uo = pr.U.copy()
    to, _, _ = oracle.run(Uo, pr.gamma, pr.bc, pr.cfl, nsteps)
    for rank, t, U, p_ref, tot, dt_all in res:
        assert t == pytest.approx(to, rel=1e-14)
        assert np.abs(U - Uo).max() <= 1e-13 * np.abs(Uo).max()
        assert p_ref == 1.0                                  # the smallest of the blocks' choices, on every rank
        assert np.allclose(tot, oracle.totals(Uo), rtol=1e-13, atol=1e-12)
        assert dt_all == pytest.approx(oracle.cfl_dt(Uo, pr.gamma, 0.4), rel=1e-14)
