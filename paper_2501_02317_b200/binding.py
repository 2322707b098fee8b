"""Thin ctypes front end of the C-ABI in ``include/kratos_hydro.h`` -- argument marshalling only.

Every step of the path runs in the CUDA kernels of ``libkratos_hydro.so``; there is no Python or
CPU fallback: if the library is missing it is built with nvcc, and if that fails, or no CUDA
device is present when a solver is created, an exception is raised.

PyTorch is used for device memory and streams only (``torch.Tensor.data_ptr()``,
``torch.cuda.current_stream().cuda_stream``); numpy arrays are accepted as host buffers.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

PREC_MIXED, PREC_FP64, PREC_SINGLE = 0, 1, 2
BC_PERIODIC, BC_FREE, BC_OUTFLOW, BC_REFLECT, BC_COMM = 0, 1, 2, 3, 4
PHASE_PREPARE, PHASE_STAGE1, PHASE_STAGE2 = 0, 1, 2
INTEGRATOR_HEUN, INTEGRATOR_VANLEER = 0 << 4, 1 << 4   # scheme word bits 4-5
KERNEL_AUTO, KERNEL_SIMPLE, KERNEL_TILED, KERNEL_PAIRED, KERNEL_TMA, KERNEL_STRIP = 0, 1, 2, 3, 5, 6
OK, ERR_ARG, ERR_ALLOC, ERR_CUDA, ERR_NONFINITE = 0, -1, -2, -3, -4

# every symbol include/kratos_hydro.h declares
SYMBOLS = [
    "kratos_hydro_create", "kratos_hydro_destroy", "kratos_hydro_set_spacing", "kratos_hydro_set_stream",
    "kratos_hydro_set_kernel", "kratos_hydro_get_kernel", "kratos_hydro_set_zchunk", "kratos_hydro_set_state", "kratos_hydro_get_state",
    "kratos_hydro_cfl_dt", "kratos_hydro_step", "kratos_hydro_run", "kratos_hydro_run_until",
    "kratos_hydro_totals", "kratos_hydro_floor_hits", "kratos_hydro_status", "kratos_hydro_launch_count",
    "kratos_hydro_set_profiling", "kratos_hydro_get_timing", "kratos_hydro_last_error", "kratos_hydro_version",
    # communication boundaries and the pieces of a run (multi-block driver: slab.py)
    "kratos_hydro_ghost_array", "kratos_hydro_ghost_ipc_handle", "kratos_hydro_set_peer", "kratos_hydro_open_peer",
    "kratos_hydro_push_halo", "kratos_hydro_begin_run", "kratos_hydro_substep", "kratos_hydro_end_run",
    "kratos_hydro_get_rate", "kratos_hydro_set_rate", "kratos_hydro_get_reference_pressure",
    "kratos_hydro_set_reference_pressure",
    # the totals for callers that may not allocate device memory (no handle)
    "kratos_hydro_totals_static",
]

_lib = None


class KratosError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"kratos_hydro error {code}: {msg}")
        self.code = code


def library_path() -> str:
    return _build.LIB


def load() -> ctypes.CDLL:
    """Load (building first if needed) the C-ABI library and declare its signatures."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    if not os.path.exists(path):
        raise ImportError("libkratos_hydro.so is missing and could not be built: no fallback exists")
    L = ctypes.CDLL(path)
    vp, d, i = ctypes.c_void_p, ctypes.c_double, ctypes.c_int
    dp, ip, llp = ctypes.POINTER(d), ctypes.POINTER(i), ctypes.POINTER(ctypes.c_longlong)
    L.kratos_hydro_create.restype = vp
    L.kratos_hydro_create.argtypes = [i, i, i, d, i, ip]
    L.kratos_hydro_destroy.restype = None
    L.kratos_hydro_destroy.argtypes = [vp]
    L.kratos_hydro_set_spacing.restype = i
    L.kratos_hydro_set_spacing.argtypes = [vp, d, d, d]
    L.kratos_hydro_set_stream.restype = i
    L.kratos_hydro_set_stream.argtypes = [vp, vp]
    L.kratos_hydro_set_kernel.restype = i
    L.kratos_hydro_set_kernel.argtypes = [vp, i]
    L.kratos_hydro_get_kernel.restype = i
    L.kratos_hydro_get_kernel.argtypes = [vp, ip]
    L.kratos_hydro_set_zchunk.restype = i
    L.kratos_hydro_set_zchunk.argtypes = [vp, i]
    L.kratos_hydro_set_state.restype = i
    L.kratos_hydro_set_state.argtypes = [vp, vp, i]
    L.kratos_hydro_get_state.restype = i
    L.kratos_hydro_get_state.argtypes = [vp, vp, i]
    L.kratos_hydro_cfl_dt.restype = i
    L.kratos_hydro_cfl_dt.argtypes = [vp, d, dp]
    L.kratos_hydro_step.restype = i
    L.kratos_hydro_step.argtypes = [vp, d]
    L.kratos_hydro_run.restype = i
    L.kratos_hydro_run.argtypes = [vp, d, i, dp]
    L.kratos_hydro_run_until.restype = i
    L.kratos_hydro_run_until.argtypes = [vp, d, d, i, dp, ip]
    L.kratos_hydro_totals.restype = i
    L.kratos_hydro_totals.argtypes = [vp, dp]
    L.kratos_hydro_floor_hits.restype = i
    L.kratos_hydro_floor_hits.argtypes = [vp, llp]
    L.kratos_hydro_status.restype = i
    L.kratos_hydro_status.argtypes = [vp]
    L.kratos_hydro_launch_count.restype = i
    L.kratos_hydro_launch_count.argtypes = [vp, llp]
    L.kratos_hydro_set_profiling.restype = i
    L.kratos_hydro_set_profiling.argtypes = [vp, i]
    L.kratos_hydro_get_timing.restype = i
    L.kratos_hydro_get_timing.argtypes = [vp, dp, llp]
    ucp = ctypes.POINTER(ctypes.c_ubyte)
    L.kratos_hydro_ghost_array.restype = i
    L.kratos_hydro_ghost_array.argtypes = [vp, i, i, ctypes.POINTER(vp)]
    L.kratos_hydro_ghost_ipc_handle.restype = i
    L.kratos_hydro_ghost_ipc_handle.argtypes = [vp, i, i, ucp]
    L.kratos_hydro_set_peer.restype = i
    L.kratos_hydro_set_peer.argtypes = [vp, i, vp, vp]
    L.kratos_hydro_open_peer.restype = i
    L.kratos_hydro_open_peer.argtypes = [vp, i, ucp, ucp]
    L.kratos_hydro_push_halo.restype = i
    L.kratos_hydro_push_halo.argtypes = [vp]
    L.kratos_hydro_begin_run.restype = i
    L.kratos_hydro_begin_run.argtypes = [vp, d, d]
    L.kratos_hydro_substep.restype = i
    L.kratos_hydro_substep.argtypes = [vp, i]
    L.kratos_hydro_end_run.restype = i
    L.kratos_hydro_end_run.argtypes = [vp, dp, ip]
    L.kratos_hydro_get_rate.restype = i
    L.kratos_hydro_get_rate.argtypes = [vp, vp, i]
    L.kratos_hydro_set_rate.restype = i
    L.kratos_hydro_set_rate.argtypes = [vp, vp, i]
    L.kratos_hydro_get_reference_pressure.restype = i
    L.kratos_hydro_get_reference_pressure.argtypes = [vp, dp]
    L.kratos_hydro_set_reference_pressure.restype = i
    L.kratos_hydro_set_reference_pressure.argtypes = [vp, d]
    L.kratos_hydro_last_error.restype = ctypes.c_char_p
    L.kratos_hydro_last_error.argtypes = []
    L.kratos_hydro_version.restype = ctypes.c_char_p
    L.kratos_hydro_version.argtypes = []
    L.kratos_hydro_totals_static.restype = i
    L.kratos_hydro_totals_static.argtypes = [vp, ctypes.c_longlong, vp, i, vp]
    _lib = L
    return L


def last_error() -> str:
    return load().kratos_hydro_last_error().decode()


def version() -> str:
    return load().kratos_hydro_version().decode()


def _check(rc: int):
    if rc != OK:
        raise KratosError(rc, last_error())


def _buffer(x):
    """(address, on_device, keepalive) of a numpy array or torch tensor holding 5*N float64."""
    if isinstance(x, np.ndarray):
        if x.dtype != np.float64 or not x.flags.c_contiguous:
            raise ValueError("host buffer must be C-contiguous float64")
        return x.ctypes.data, 0, x
    import torch
    if isinstance(x, torch.Tensor):
        if x.dtype != torch.float64 or not x.is_contiguous():
            raise ValueError("tensor must be contiguous float64")
        return x.data_ptr(), 1 if x.is_cuda else 0, x
    raise TypeError(type(x))


TOTALS_STATIC_MAX_CELLS = 1 << 31


def totals_static(U, out=None, stream=None, ncell=None):
    """``kratos_hydro_totals_static``: the five conserved totals of a state that already sits in device memory, for
    programs that cannot let this library allocate -- the device is wholly owned by their own memory pool, or they
    are in the middle of a run and cannot take the device-wide wait a ``cudaMalloc`` / ``cudaFree`` brings.  No handle
    is created; the partial sums go to an array built into the library (shared by all calls on a device: do not let two
    calls overlap on the GPU).  The first call on a device should be made outside any stream capture.

    ``U``: CUDA tensor, contiguous float64, 5*ncell values (``ncell`` defaults to ``U.numel() // 5``; at most
    ``TOTALS_STATIC_MAX_CELLS``).  ``out``: None -> a new numpy array of 5 (the call synchronises ``stream``), or a
    CUDA float64 tensor of 5 on the same device (asynchronous).  ``stream``: a torch.cuda.Stream, a raw cudaStream_t
    integer, or None for torch's current stream.  Equals ``KratosHydro.totals()`` of the same state bit for bit."""
    import torch
    L = load()
    if not (isinstance(U, torch.Tensor) and U.is_cuda):
        raise TypeError("U must be a CUDA tensor (the caller owns the state on the device)")
    ptr, _dev, _keep = _buffer(U)
    n = U.numel() // 5 if ncell is None else int(ncell)
    if ncell is None and U.numel() != 5 * n:
        raise ValueError("state must hold 5*ncell values")
    if stream is None:
        stream = torch.cuda.current_stream(U.device)
    sptr = ctypes.c_void_p(int(getattr(stream, "cuda_stream", stream) or 0))
    with torch.cuda.device(U.device):
        if out is None:
            host = (ctypes.c_double * 5)()
            _check(L.kratos_hydro_totals_static(ctypes.c_void_p(ptr), n, ctypes.cast(host, ctypes.c_void_p), 0, sptr))
            return np.array(host[:])
        optr, odev, _keep2 = _buffer(out)
        if out.numel() != 5:
            raise ValueError("out must hold 5 values")
        _check(L.kratos_hydro_totals_static(ctypes.c_void_p(ptr), n, ctypes.c_void_p(optr), odev, sptr))
        return out


class KratosHydro:
    """One uniform block on the current CUDA device.  Method names mirror the C entry points."""

    def __init__(self, nx, ny, nz, gamma, bc, precision=PREC_MIXED, spacing=None, kernel=KERNEL_AUTO,
                 stream=None, integrator=INTEGRATOR_HEUN):
        L = load()
        self._L = L
        self.shape = (int(nx), int(ny), int(nz))
        self.ncell = int(nx) * int(ny) * int(nz)
        bc_arr = (ctypes.c_int * 6)(*[int(b) for b in bc])
        self._h = L.kratos_hydro_create(int(nx), int(ny), int(nz), float(gamma), int(precision) | int(integrator), bc_arr)
        if not self._h:
            raise KratosError(ERR_ARG, last_error())
        if spacing is not None:
            self.set_spacing(*spacing)
        if kernel != KERNEL_AUTO:
            self.set_kernel(kernel)
        if stream is not None:
            self.set_stream(stream)

    # -- lifetime
    def destroy(self):
        if getattr(self, "_h", None):
            self._L.kratos_hydro_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    # -- configuration
    def set_spacing(self, dx, dy, dz):
        _check(self._L.kratos_hydro_set_spacing(self._h, float(dx), float(dy), float(dz)))

    def set_stream(self, stream):
        """``stream``: a torch.cuda.Stream, a raw cudaStream_t integer, or None/0 for the default stream."""
        ptr = getattr(stream, "cuda_stream", stream) or 0
        _check(self._L.kratos_hydro_set_stream(self._h, ctypes.c_void_p(int(ptr))))

    def set_kernel(self, variant):
        _check(self._L.kratos_hydro_set_kernel(self._h, int(variant)))

    def get_kernel(self):
        v = ctypes.c_int(0)
        _check(self._L.kratos_hydro_get_kernel(self._h, ctypes.byref(v)))
        return v.value

    def set_zchunk(self, planes):
        _check(self._L.kratos_hydro_set_zchunk(self._h, int(planes)))

    # -- state
    def set_state(self, U):
        ptr, dev, _keep = _buffer(U)
        n = U.size if isinstance(U, np.ndarray) else U.numel()
        if n != 5 * self.ncell:
            raise ValueError("state must hold 5*nx*ny*nz values")
        _check(self._L.kratos_hydro_set_state(self._h, ctypes.c_void_p(ptr), dev))

    def get_state(self, out=None):
        nx, ny, nz = self.shape
        if out is None:
            out = np.empty((5, nz, ny, nx), dtype=np.float64)
        ptr, dev, _keep = _buffer(out)
        _check(self._L.kratos_hydro_get_state(self._h, ctypes.c_void_p(ptr), dev))
        return out

    # -- the path
    def cfl_dt(self, cfl):
        dt = ctypes.c_double(0.0)
        _check(self._L.kratos_hydro_cfl_dt(self._h, float(cfl), ctypes.byref(dt)))
        return dt.value

    def step(self, dt):
        _check(self._L.kratos_hydro_step(self._h, float(dt)))

    def run(self, cfl, nsteps, t0=0.0):
        t = ctypes.c_double(float(t0))
        _check(self._L.kratos_hydro_run(self._h, float(cfl), int(nsteps), ctypes.byref(t)))
        return t.value

    def run_until(self, cfl, t_end, max_steps=10 ** 7, t0=0.0):
        t = ctypes.c_double(float(t0))
        n = ctypes.c_int(0)
        _check(self._L.kratos_hydro_run_until(self._h, float(cfl), float(t_end), int(max_steps),
                                              ctypes.byref(t), ctypes.byref(n)))
        return t.value, n.value

    # -- diagnostics
    def totals(self):
        out = (ctypes.c_double * 5)()
        _check(self._L.kratos_hydro_totals(self._h, out))
        return np.array(out[:])

    def floor_hits(self):
        n = ctypes.c_longlong(0)
        _check(self._L.kratos_hydro_floor_hits(self._h, ctypes.byref(n)))
        return n.value

    def status(self):
        """Raises KratosError (ERR_NONFINITE / ERR_CUDA) if the run so far went wrong; synchronises."""
        _check(self._L.kratos_hydro_status(self._h))

    def launch_count(self):
        n = ctypes.c_longlong(0)
        _check(self._L.kratos_hydro_launch_count(self._h, ctypes.byref(n)))
        return n.value

    def set_profiling(self, enable=True):
        """True / 1: events around every launch; n > 1: around the launches of every n-th step; False / 0: off."""
        _check(self._L.kratos_hydro_set_profiling(self._h, int(enable)))

    def get_timing(self):
        """{'stage1': (ms, launches), 'stage2': ..., 'other': ...} since set_profiling."""
        ms = (ctypes.c_double * 3)()
        n = (ctypes.c_longlong * 3)()
        _check(self._L.kratos_hydro_get_timing(self._h, ms, n))
        return {k: (ms[i], n[i]) for i, k in enumerate(("stage1", "stage2", "other"))}

    # -- communication boundaries and the pieces of a run (include/kratos_hydro.h, "Communication boundaries")
    def ghost_array(self, array, side):
        """Device address of this block's ghost array (int)."""
        p = ctypes.c_void_p(0)
        _check(self._L.kratos_hydro_ghost_array(self._h, int(array), int(side), ctypes.byref(p)))
        return int(p.value)

    def ghost_ipc_handle(self, array, side):
        """The 64 bytes of the CUDA IPC handle of that ghost array."""
        buf = (ctypes.c_ubyte * 64)()
        _check(self._L.kratos_hydro_ghost_ipc_handle(self._h, int(array), int(side), buf))
        return bytes(buf)

    def set_peer(self, side, peer_ghost_state, peer_ghost_pred):
        _check(self._L.kratos_hydro_set_peer(self._h, int(side), ctypes.c_void_p(int(peer_ghost_state)),
                                             ctypes.c_void_p(int(peer_ghost_pred))))

    def open_peer(self, side, handle_state, handle_pred):
        a = (ctypes.c_ubyte * 64).from_buffer_copy(bytes(handle_state))
        b = (ctypes.c_ubyte * 64).from_buffer_copy(bytes(handle_pred))
        _check(self._L.kratos_hydro_open_peer(self._h, int(side), a, b))

    def push_halo(self):
        _check(self._L.kratos_hydro_push_halo(self._h))

    def begin_run(self, cfl, t0=0.0):
        _check(self._L.kratos_hydro_begin_run(self._h, float(cfl), float(t0)))

    def substep(self, phase):
        _check(self._L.kratos_hydro_substep(self._h, int(phase)))

    def end_run(self):
        t = ctypes.c_double(0.0)
        n = ctypes.c_int(0)
        _check(self._L.kratos_hydro_end_run(self._h, ctypes.byref(t), ctypes.byref(n)))
        return t.value, n.value

    def get_rate(self, out=None):
        """The CFL rate maximum: a float, or written into a 1-element float64 tensor / array (device: asynchronous)."""
        if out is None:
            v = ctypes.c_double(0.0)
            _check(self._L.kratos_hydro_get_rate(self._h, ctypes.cast(ctypes.byref(v), ctypes.c_void_p), 0))
            return v.value
        ptr, dev, _keep = _buffer(out)
        _check(self._L.kratos_hydro_get_rate(self._h, ctypes.c_void_p(ptr), dev))
        return out

    def set_rate(self, rate):
        if isinstance(rate, (int, float)):
            v = ctypes.c_double(float(rate))
            _check(self._L.kratos_hydro_set_rate(self._h, ctypes.cast(ctypes.byref(v), ctypes.c_void_p), 0))
            return
        ptr, dev, _keep = _buffer(rate)
        _check(self._L.kratos_hydro_set_rate(self._h, ctypes.c_void_p(ptr), dev))

    def get_reference_pressure(self):
        v = ctypes.c_double(0.0)
        _check(self._L.kratos_hydro_get_reference_pressure(self._h, ctypes.byref(v)))
        return v.value

    def set_reference_pressure(self, p_ref):
        _check(self._L.kratos_hydro_set_reference_pressure(self._h, float(p_ref)))
