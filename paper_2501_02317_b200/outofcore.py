"""One Heun step of a block whose state lives in (pinned) host memory, streamed through the GPU in z chunks.

The end-to-end cost of a step on host-resident data is the PCIe round trip of the state (2 x 40 B per cell), not the 7 ms of
arithmetic; copying the whole block in, stepping, and copying it out leaves each of the three engines (host-to-device copy,
SMs, device-to-host copy) idle two thirds of the time.  A Heun step has a domain of dependence of four planes (two stages
x the two-cell stencil of PLM + HLLC), so the block is cut into chunks of ``chunk`` planes; each chunk
travels with four extra planes on either cut side, is advanced as a block of its own (the extra planes absorb what the
artificial Free boundary at their outer end gets wrong; the domain's real boundary rule is kept where a chunk touches the
end of the block), and only its own planes travel back.  Two buffers on two streams keep the upload of
chunk i+1, the kernels of chunk i and the download of chunk i-1 in flight together; the overlap planes a chunk shares with
its predecessor are copied on the device, so every plane crosses the bus once per direction and step (a periodic block
uploads its wrapped overlap a second time).  The same scheme steps a block that does
not fit the device at all.

Every stage of every chunk runs in the library's kernels through the C-ABI (set_state / step / get_state on device
buffers); this file only schedules copies.  The planes a chunk returns are bit for bit those of the undivided step when the
same reference pressure is used (the slab seams of the TMA kernel are bitwise invisible): tests/test_gpu_outofcore.py.
"""
from __future__ import annotations

from . import binding

HALO = 4   # planes of dependence of one Heun step: 2 stages x 2 cells


class HostStepper:
    def __init__(self, nx, ny, nz, gamma, bc, chunk=64, precision=binding.PREC_MIXED, p_ref=None, spacing=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("HostStepper needs a CUDA device: the product path has no CPU fallback")
        self.shape = (int(nx), int(ny), int(nz))
        self.gamma, self.bc, self.precision = float(gamma), tuple(int(b) for b in bc), precision
        self.periodic = self.bc[4] == binding.BC_PERIODIC
        if nz < 2 * HALO + 1:
            raise ValueError("the block needs more planes than the step's domain of dependence")
        self.chunk = max(1, min(int(chunk), nz))
        # cell sizes (dx, dy, dz) of the WHOLE block, handed to every chunk's handle: a chunk has fewer planes, not thinner
        # ones.  Default: the unit box, as for KratosHydro and SlabSolver.
        self.spacing = (1.0 / nx, 1.0 / ny, 1.0 / nz) if spacing is None else tuple(float(d) for d in spacing)
        if len(self.spacing) != 3:
            raise ValueError("spacing = (dx, dy, dz)")
        self.p_ref = p_ref
        self.streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        self._slots = {}       # (planes, bc_lo, bc_hi, slot) -> (handle, device buffer)
        self.h2d_bytes = self.d2h_bytes = self.d2d_bytes = 0
        self._rates, self.rate = None, float("nan")

    # where the planes [a, b) of a chunk's block come from: runs of host planes, wrapped around a periodic block
    def _runs(self, a, b):
        nz = self.shape[2]
        runs, z = [], a
        while z < b:
            zz = z % nz
            n = min(b - z, nz - zz)
            runs.append((zz, n))
            z += n
        return runs

    def plan(self):
        """[(z0, z1, a, b, bc_lo, bc_hi)]: chunk [z0, z1) travels as planes [a, b) with those z boundary codes.  A periodic
        block wraps (a < 0, b > nz allowed); otherwise the travelling block stops at the end of the domain and keeps the
        domain's boundary rule there."""
        nz, out = self.shape[2], []
        for z0 in range(0, nz, self.chunk):
            z1 = min(z0 + self.chunk, nz)
            if self.periodic:
                out.append((z0, z1, z0 - HALO, z1 + HALO, binding.BC_FREE, binding.BC_FREE))
            else:
                a, b = max(z0 - HALO, 0), min(z1 + HALO, nz)
                out.append((z0, z1, a, b, self.bc[4] if a == 0 else binding.BC_FREE, self.bc[5] if b == nz else binding.BC_FREE))
        return out

    def _slot(self, planes, bc_lo, bc_hi, slot):
        import torch
        key = (planes, bc_lo, bc_hi, slot)
        if key not in self._slots:
            nx, ny, _ = self.shape
            bc = self.bc[:4] + (bc_lo, bc_hi)
            h = binding.KratosHydro(nx, ny, planes, self.gamma, bc, precision=self.precision, spacing=self.spacing,
                                    stream=self.streams[slot])
            bin_ = torch.empty((5, planes, ny, nx), dtype=torch.float64, device="cuda")    # what was uploaded (kept for the next chunk)
            bout = torch.empty((5, planes, ny, nx), dtype=torch.float64, device="cuda")   # the chunk block after the step
            self._slots[key] = (h, bin_, bout)
        return self._slots[key]

    def step(self, src, dst, dt):
        """dst <- one Heun step of length dt of src.  src, dst: float64 torch tensors of 5*nx*ny*nz elements in pinned host
        memory (layout of the C-ABI), distinct.  Returns when dst is complete."""
        import torch
        nx, ny, nz = self.shape
        src, dst = src.view(5, nz, ny, nx), dst.view(5, nz, ny, nx)
        if self.p_ref is None:
            raise ValueError("set p_ref (one reference pressure for all chunks, e.g. KratosHydro.get_reference_pressure)")
        plan = self.plan()
        if self._rates is None or self._rates.numel() != len(plan):
            self._rates = torch.zeros(len(plan), dtype=torch.float64, device="cuda")
        prev = None          # (input buffer, first plane, end plane, event: uploaded) of the previous chunk
        freed = [None, None]  # per slot: event after which its input buffer may be overwritten (the next chunk has copied from it)
        for i, (z0, z1, a, b, bc_lo, bc_hi) in enumerate(plan):
            slot = i & 1
            stream = self.streams[slot]
            h, bin_, bout = self._slot(b - a, bc_lo, bc_hi, slot)
            with torch.cuda.stream(stream):
                if freed[slot] is not None:
                    stream.wait_event(freed[slot])
                # planes the previous chunk has on the device already (its upper overlap = this chunk's lower one) are copied
                # there; everything else comes up from the host, every plane of the block exactly once per step
                lo = a
                if prev is not None and prev[1] <= a < prev[2] and not (a < 0):
                    pbuf, pa, pb, pev = prev
                    n = min(pb, b) - a
                    stream.wait_event(pev)
                    bin_[:, 0:n].copy_(pbuf[:, a - pa:a - pa + n], non_blocking=True)
                    lo = a + n
                    ev = torch.cuda.Event()
                    ev.record(stream)
                    freed[slot ^ 1] = ev
                    self.d2d_bytes += 40 * nx * ny * n
                off = lo - a
                for zz, n in self._runs(lo, b):
                    for f in range(5):      # contiguous runs: plain asynchronous copies
                        bin_[f, off:off + n].copy_(src[f, zz:zz + n], non_blocking=True)
                    off += n
                    self.h2d_bytes += 40 * nx * ny * n
                up = torch.cuda.Event()
                up.record(stream)
                prev = (bin_, a, b, up)
                h.set_state(bin_)
                h.set_reference_pressure(self.p_ref)
                h.step(dt)
                h.get_rate(self._rates[i:i + 1])     # CFL rate of the chunk's new state, reduced inside its stage 2
                h.get_state(bout)
                for f in range(5):
                    dst[f, z0:z1].copy_(bout[f, z0 - a:z1 - a], non_blocking=True)
            self.d2h_bytes += 40 * nx * ny * (z1 - z0)
        for s in self.streams:
            s.synchronize()
        self.rate = float(self._rates.max().item())
        return dst

    def next_dt(self, cfl):
        """CFL time step for the state the last step produced: cfl over the largest of the chunks' rate maxima.
        The chunks' overlap planes take part, so this is the block's own dt or marginally less."""
        return float(cfl) / self.rate

    def launch_count(self):
        return sum(v[0].launch_count() for v in self._slots.values())

    def destroy(self):
        for v in self._slots.values():
            v[0].destroy()
        self._slots = {}
