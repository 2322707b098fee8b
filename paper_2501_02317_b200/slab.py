"""One block cut into z slabs, one slab per GPU.

PAPER.md Sec. 3.1.2: blocks talk to each other through communication boundaries ("c-boundaries")
whose ghost zones are filled from the neighbouring block; Table 2 times two-GPU splits of one
domain.  Here the domain is cut along z (the slowest index: every cut face is two contiguous planes per field), each
rank owns ``nz / world`` planes (+1 on the first ``nz % world`` ranks) and creates its block with ``BC_COMM`` on the
cut faces.  Nothing in this file touches the state: the halo exchange is part of the stage kernels (a block stores
its planes next to a cut face a second time, straight into the neighbour's ghost array over peer memory, see
``include/kratos_hydro.h``), and what is left for the host is

* the bookkeeping of the decomposition (``SlabDecomposition``: planes, neighbours, boundary codes, peer wiring),
* ordering: stage 2 of a block may start only after stage 1 of its neighbours, the next stage 1 only after their
  stage 2 (``comm.sync()``: stream order when all blocks live in one process on one stream, a one-element
  all-reduce on the NCCL stream across processes), and
* the time step: the CFL rate maximum over all blocks (one 8-byte all-reduce(max) per step), and one
  reference pressure for all blocks (reading S17).

``SlabSolver`` is the driver.  With ``torch.distributed`` initialised (one process per GPU, NCCL) every process
holds its own slab and the neighbours' ghost arrays are mapped through CUDA IPC handles; without it all slabs live
in this process on the current device and advance in lock step on one stream -- the same kernels, the same peer
stores, the same sequence of calls, which is how the path is tested on a single GPU (bit for bit equal to the
undivided block).
"""
from __future__ import annotations

import numpy as np

from . import binding

BC_COMM = binding.BC_COMM


class SlabDecomposition:
    """Host-side bookkeeping of ``world`` z slabs of a block with ``nz`` planes.  No device work, no state."""

    MIN_PLANES = 4   # a block's stencil reaches two planes: the two planes it sends on either side must be distinct

    def __init__(self, nz: int, world: int, bc_z_lo: int, bc_z_hi: int):
        if world < 1:
            raise ValueError("world must be >= 1")
        if (bc_z_lo == binding.BC_PERIODIC) != (bc_z_hi == binding.BC_PERIODIC):
            raise ValueError("periodic on one side only")
        if world > 1 and nz // world < self.MIN_PLANES:
            raise ValueError(f"{nz} planes over {world} ranks: every slab needs >= {self.MIN_PLANES} planes")
        self.nz, self.world = int(nz), int(world)
        self.bc_z = (int(bc_z_lo), int(bc_z_hi))
        self.periodic = bc_z_lo == binding.BC_PERIODIC

    def planes(self, rank: int):
        """[z0, z1): the global planes rank owns (balanced: the first nz % world ranks own one more)."""
        q, r = divmod(self.nz, self.world)
        z0 = rank * q + min(rank, r)
        return z0, z0 + q + (1 if rank < r else 0)

    def neighbours(self, rank: int):
        """(rank below, rank above) across the cut faces; None where the face is a physical boundary of the domain.
        A periodic domain wraps (with world == 1 the block keeps its own periodic boundary: no cut at all)."""
        if self.world == 1:
            return None, None
        lo = rank - 1 if rank > 0 else (self.world - 1 if self.periodic else None)
        hi = rank + 1 if rank < self.world - 1 else (0 if self.periodic else None)
        return lo, hi

    def local_bc(self, rank: int, bc):
        """The six boundary codes of rank's block: BC_COMM on cut faces, the domain's own codes elsewhere."""
        lo, hi = self.neighbours(rank)
        out = list(int(b) for b in bc)
        out[4] = BC_COMM if lo is not None else self.bc_z[0]
        out[5] = BC_COMM if hi is not None else self.bc_z[1]
        return tuple(out)

    def ghost_source(self, rank: int, side: int):
        """Where the two ghost planes beyond z face ``side`` of rank's block come from:
        (neighbour rank, [global planes], [the neighbour's local planes]), ascending z; None at a physical boundary."""
        nb = self.neighbours(rank)[side]
        if nb is None:
            return None
        z0, z1 = self.planes(rank)
        glob = [(z0 - 2 + i) % self.nz for i in range(2)] if side == 0 else [(z1 + i) % self.nz for i in range(2)]
        n0, _ = self.planes(nb)
        return nb, glob, [z - n0 for z in glob]

    def scatter(self, U: np.ndarray, rank: int) -> np.ndarray:
        z0, z1 = self.planes(rank)
        return np.ascontiguousarray(U[:, z0:z1])

    def gather(self, parts, out=None) -> np.ndarray:
        """parts: {rank: local state [5, nz_r, ny, nx]} for every rank."""
        first = parts[0]
        if out is None:
            out = np.empty((5, self.nz) + first.shape[2:], dtype=first.dtype)
        for r in range(self.world):
            z0, z1 = self.planes(r)
            out[:, z0:z1] = parts[r]
        return out


class _LocalComm:
    """All blocks in this process, on one device and one stream: stream order is the synchronisation."""
    rank, world = 0, 1

    def sync(self, device):
        pass

    def all_max(self, t):
        return t

    def all_min_float(self, x):
        return x

    def all_sum(self, a):
        return a

    def all_gather_object(self, obj):
        return [obj]


class _DistComm:
    """One process per GPU (torch.distributed).  NCCL: the collectives are enqueued on the current CUDA stream, so they
    order the ranks' streams without a host round trip.  Any other backend (gloo: the CPU test of the host logic, and two
    processes sharing the one GPU of a test box): the stream is drained first and the collective runs on host tensors."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.nccl = dist.get_backend(group) == "nccl"
        self._token = None

    def _drain(self, device):
        import torch
        if not self.nccl and torch.device(device).type == "cuda":
            torch.cuda.current_stream().synchronize()

    def sync(self, device):
        # no rank passes this point before every rank's stream has reached it
        import torch
        self._drain(device)
        if self._token is None:
            # created once: NCCL reduces it on this rank's GPU (the device is spelled out -- torch.device("cuda") carries
            # no index and never compares equal to the "cuda:0" a tensor reports), any other backend on the host
            dev = torch.device("cuda", torch.cuda.current_device()) if self.nccl else torch.device("cpu")
            self._token = torch.zeros(1, dtype=torch.float32, device=dev)
        self.dist.all_reduce(self._token, group=self.group)

    def all_max(self, t):
        if self.nccl or t.device.type == "cpu":
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX, group=self.group)
            return t
        self._drain(t.device)
        h = t.cpu()
        self.dist.all_reduce(h, op=self.dist.ReduceOp.MAX, group=self.group)
        t.copy_(h)
        return t

    def all_min_float(self, x):
        import torch
        t = torch.tensor([float(x)], dtype=torch.float64, device="cuda" if self.nccl else "cpu")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MIN, group=self.group)
        return float(t.item())

    def all_sum(self, a):
        import torch
        t = torch.as_tensor(np.asarray(a, dtype=np.float64), device="cuda" if self.nccl else "cpu")
        self.dist.all_reduce(t, group=self.group)
        return t.cpu().numpy()

    def all_gather_object(self, obj):
        out = [None] * self.world
        self.dist.all_gather_object(out, obj, group=self.group)
        return out


class SlabSolver:
    """A block of nx x ny x nz cells advanced as ``world`` z slabs (Heun, mixed precision, TMA kernel).

    Distributed (``torch.distributed`` initialised, or ``group`` given): ``world`` = the group's size, this process owns
    the slab of its rank on the current CUDA device.  Otherwise ``world`` slabs are created in this process.
    ``make_block(rank, (nx, ny, nz_r), gamma, bc_r)``: factory of the per-rank block (default: ``binding.KratosHydro``);
    a stand-in that sets ``wires_itself`` delivers its halos by its own means (CPU test of the host logic).
    """

    def __init__(self, nx, ny, nz, gamma, bc, world=None, group=None, stream=None, precision=binding.PREC_MIXED,
                 spacing=None, make_block=None):
        import torch
        import torch.distributed as dist
        distributed = group is not None or (dist.is_available() and dist.is_initialized())
        self.comm = _DistComm(group) if distributed else _LocalComm()
        self.world = self.comm.world if distributed else int(world or 1)
        self.shape = (int(nx), int(ny), int(nz))
        self.gamma = float(gamma)
        self.dec = SlabDecomposition(nz, self.world, bc[4], bc[5])
        self.ranks = [self.comm.rank] if distributed else list(range(self.world))
        self.stream = stream
        if spacing is None:
            spacing = (1.0 / nx, 1.0 / ny, 1.0 / nz)   # of the WHOLE block: a slab has fewer planes, not thinner ones
        self.blocks = {}
        for r in self.ranks:
            z0, z1 = self.dec.planes(r)
            bc_r = self.dec.local_bc(r, bc)
            if make_block is not None:
                self.blocks[r] = make_block(r, (nx, ny, z1 - z0), gamma, bc_r)
            else:
                self.blocks[r] = binding.KratosHydro(nx, ny, z1 - z0, gamma, bc_r, precision=precision, spacing=spacing,
                                                     stream=stream)
        first = self.blocks[self.ranks[0]]
        self.device = getattr(first, "tensor_device", "cuda")
        self._rate = {r: torch.zeros(1, dtype=torch.float64, device=self.device) for r in self.ranks}
        if not getattr(first, "wires_itself", False):
            self._wire()

    # -- peers: every block learns where its neighbours keep the ghost planes it has to fill
    def _wire(self):
        if isinstance(self.comm, _LocalComm):
            for r, b in self.blocks.items():
                for side, nb in enumerate(self.dec.neighbours(r)):
                    if nb is not None:   # my planes next to face `side` are the neighbour's ghosts beyond its OTHER face
                        b.set_peer(side, self.blocks[nb].ghost_array(0, 1 - side), self.blocks[nb].ghost_array(1, 1 - side))
            return
        r = self.ranks[0]
        mine = {}
        for side, nb in enumerate(self.dec.neighbours(r)):
            if nb is not None:
                mine[side] = (self.blocks[r].ghost_ipc_handle(0, side), self.blocks[r].ghost_ipc_handle(1, side))
        table = self.comm.all_gather_object(mine)
        for side, nb in enumerate(self.dec.neighbours(r)):
            if nb is not None:
                hs, hp = table[nb][1 - side]
                self.blocks[r].open_peer(side, hs, hp)

    def _ctx(self):
        import contextlib
        import torch
        if self.stream is not None and hasattr(self.stream, "cuda_stream"):
            return torch.cuda.stream(self.stream)   # the collectives go onto the stream the kernels run on
        return contextlib.nullcontext()

    # -- state
    def set_state(self, U):
        """U: the state of the WHOLE block, [5, nz, ny, nx] float64 on the host (every rank takes its planes), or
        {rank: local state} for the ranks this process owns."""
        import torch
        self.last_upload_bytes = 0     # host -> device bytes of this call (this process)
        if isinstance(U, torch.Tensor):
            nx, ny, nz = self.shape
            Uv = U.reshape(5, nz, ny, nx)
            with self._ctx():
                if U.is_cuda or len(self.blocks) == self.world:
                    # every plane is wanted on this device: one copy onto it, the slabs are cut there
                    Ud = Uv.to(self.device, non_blocking=True)
                    self.last_upload_bytes = 0 if U.is_cuda else U.numel() * 8
                    for r, b in self.blocks.items():
                        z0, z1 = self.dec.planes(r)
                        b.set_state(Ud[:, z0:z1].contiguous())
                    del Ud
                else:
                    # one process per GPU: only the planes this rank owns cross the bus, one contiguous run per field
                    # (a block that fits only when decomposed is never whole on any one device)
                    for r, b in self.blocks.items():
                        z0, z1 = self.dec.planes(r)
                        part = torch.empty((5, z1 - z0, ny, nx), dtype=torch.float64, device=self.device)
                        for m in range(5):
                            part[m].copy_(Uv[m, z0:z1], non_blocking=True)
                        self.last_upload_bytes += part.numel() * 8
                        b.set_state(part)
                        del part
        else:
            for r, b in self.blocks.items():
                loc = U[r] if isinstance(U, dict) else self.dec.scatter(U, r)
                self.last_upload_bytes += loc.size * 8 if isinstance(loc, np.ndarray) else 0
                b.set_state(loc)
        # one reference pressure for the whole domain (reading S17): the smallest of the blocks' own choices
        p = min(b.get_reference_pressure() for b in self.blocks.values())
        p = self.comm.all_min_float(p)
        for b in self.blocks.values():
            b.set_reference_pressure(p)
        self.p_ref = p
        with self._ctx():
            for b in self.blocks.values():
                b.push_halo()
            self.comm.sync(self.device)

    def get_state(self):
        """{rank: local state} of the ranks this process owns."""
        return {r: b.get_state() for r, b in self.blocks.items()}

    def get_state_into(self, out):
        """Local mode: the whole block into ``out``, a float64 torch tensor of 5*nx*ny*nz elements (pinned host memory or
        device); the slabs are joined on the device and leave in one copy."""
        import torch
        nx, ny, nz = self.shape
        with self._ctx():
            full = torch.empty((5, nz, ny, nx), dtype=torch.float64, device=self.device)
            for r, b in self.blocks.items():
                z0, z1 = self.dec.planes(r)
                part = torch.empty((5, z1 - z0, ny, nx), dtype=torch.float64, device=self.device)
                b.get_state(part)
                full[:, z0:z1] = part
            out.view(5, nz, ny, nx).copy_(full, non_blocking=True)
            torch.cuda.current_stream().synchronize()
        return out

    def get_state_global(self):
        """The whole block on every rank (host).  Local mode: a gather; distributed: an all-gather of the slabs."""
        parts = self.get_state()
        if isinstance(self.comm, _DistComm):
            merged = {}
            for d in self.comm.all_gather_object(parts):
                merged.update(d)
            parts = merged
        return self.dec.gather(parts)

    # -- the path
    def run(self, cfl, nsteps, t0=0.0):
        """nsteps Heun steps of the whole block; every dt from the CFL rate maximum over all slabs.  Returns t."""
        import torch
        with self._ctx():
            for b in self.blocks.values():
                b.begin_run(cfl, t0)
            for _ in range(int(nsteps)):
                for r, b in self.blocks.items():
                    b.get_rate(self._rate[r])
                rate = self._rate[self.ranks[0]]
                for r in self.ranks[1:]:
                    torch.maximum(rate, self._rate[r], out=rate)
                rate = self.comm.all_max(rate)          # also orders this step after every neighbour's last stage 2
                for b in self.blocks.values():
                    b.set_rate(rate)
                    b.substep(binding.PHASE_PREPARE)
                for b in self.blocks.values():
                    b.substep(binding.PHASE_STAGE1)
                self.comm.sync(self.device)             # stage 2 reads what the neighbours' stage 1 delivered
                for b in self.blocks.values():
                    b.substep(binding.PHASE_STAGE2)
            self.comm.sync(self.device)
        t = [b.end_run()[0] for b in self.blocks.values()]
        return t[0]

    def cfl_dt(self, cfl):
        """CFL time step of the whole block: cfl over the rate maximum of all slabs (each slab's fp64 reduction)."""
        rate = max(float(cfl) / b.cfl_dt(cfl) for b in self.blocks.values())
        rate = -self.comm.all_min_float(-rate)
        return float(cfl) / rate

    def totals(self):
        s = np.zeros(5)
        for b in self.blocks.values():
            s += b.totals()
        return np.asarray(self.comm.all_sum(s))

    def floor_hits(self):
        return int(self.comm.all_sum([sum(b.floor_hits() for b in self.blocks.values())])[0])

    def launch_count(self):
        return sum(b.launch_count() for b in self.blocks.values())

    def destroy(self):
        for b in self.blocks.values():
            b.destroy()
        self.blocks = {}
