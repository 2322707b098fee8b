"""ORACLE -- test infrastructure, not product.

ctypes front end of ``oracle/kratos_oracle.c`` (the plain fp64 CPU restatement of the
Kratos hydro hot path, arXiv 2501.02317) plus ``oracle/exact_riemann.py`` (the exact
Riemann solution used to pin it).  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package.
It imports nothing from ``paper_2501_02317_b200`` and the CUDA path never imports it.

All functions take / return numpy float64 arrays in the layout of the C-ABI boundary:
conserved state ``U[5, nz, ny, nx]`` = (rho, m_x, m_y, m_z, eps), x fastest.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "kratos_oracle.c")
_LIB = os.path.join(_HERE, "libkratos_oracle.so")

PERIODIC, FREE, OUTFLOW, REFLECT = 0, 1, 2, 3

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP on outer loops, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
               "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        llp = ctypes.POINTER(ctypes.c_longlong)
        d, i = ctypes.c_double, ctypes.c_int
        L.orc_minmod.restype = d
        L.orc_minmod.argtypes = [d, d]
        L.orc_cons_to_prim.restype = None
        L.orc_cons_to_prim.argtypes = [dp, d, dp, llp]
        L.orc_hllc.restype = None
        L.orc_hllc.argtypes = [dp, dp, d, dp]
        L.orc_fill_ghosts_axis.restype = None
        L.orc_fill_ghosts_axis.argtypes = [dp, i, i, i, i, i, i]
        L.orc_flux_divergence.restype = i
        L.orc_flux_divergence.argtypes = [dp, i, i, i, d, ip, d, d, d, dp, llp]
        L.orc_step.restype = i
        L.orc_step.argtypes = [dp, i, i, i, d, ip, d, d, d, d, llp]
        L.orc_step_vl.restype = i
        L.orc_step_vl.argtypes = [dp, i, i, i, d, ip, d, d, d, d, llp]
        L.orc_run_vl.restype = i
        L.orc_run_vl.argtypes = [dp, i, i, i, d, ip, d, d, d, d, i, d, dp, llp]
        L.orc_cfl_dt.restype = d
        L.orc_cfl_dt.argtypes = [dp, i, i, i, d, d, d, d, d, llp]
        L.orc_run.restype = i
        L.orc_run.argtypes = [dp, i, i, i, d, ip, d, d, d, d, i, d, dp, llp]
        L.orc_totals.restype = None
        L.orc_totals.argtypes = [dp, ctypes.c_longlong, dp]
        L.orc_num_threads.restype = i
        L.orc_num_threads.argtypes = []
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _bc(bc):
    arr = (ctypes.c_int * 6)(*[int(b) for b in bc])
    return arr


def _chk(U: np.ndarray):
    if U.dtype != np.float64 or U.ndim != 4 or U.shape[0] != 5 or not U.flags.c_contiguous:
        raise ValueError("U must be C-contiguous float64 [5, nz, ny, nx]")
    _, nz, ny, nx = U.shape
    return nx, ny, nz


def default_spacing(nx, ny, nz):
    """Unit box: dx_d = 1/n_d on active axes (1.0 on inactive ones, unused)."""
    return tuple(1.0 / n if n > 1 else 1.0 for n in (nx, ny, nz))


def minmod(a: float, b: float) -> float:
    return lib().orc_minmod(a, b)


def cons_to_prim(u, gamma: float):
    u = np.ascontiguousarray(u, dtype=np.float64)
    w = np.zeros(5)
    hits = ctypes.c_longlong(0)
    lib().orc_cons_to_prim(_dp(u), gamma, _dp(w), ctypes.byref(hits))
    return w, hits.value


def hllc(WL, WR, gamma: float) -> np.ndarray:
    """WL, WR = (rho, p, u, v, w) in the face-normal frame -> F = (mass, mom_n, mom_t1, mom_t2, energy)."""
    WL = np.ascontiguousarray(WL, dtype=np.float64)
    WR = np.ascontiguousarray(WR, dtype=np.float64)
    F = np.zeros(5)
    lib().orc_hllc(_dp(WL), _dp(WR), gamma, _dp(F))
    return F


def fill_ghosts_axis(Wpad: np.ndarray, nx, ny, nz, axis, bc_lo, bc_hi) -> None:
    """In-place ghost fill of the padded primitive array [5, pz, py, px] along one axis."""
    assert Wpad.dtype == np.float64 and Wpad.flags.c_contiguous
    lib().orc_fill_ghosts_axis(_dp(Wpad), nx, ny, nz, axis, bc_lo, bc_hi)


def flux_divergence(U: np.ndarray, gamma, bc, spacing=None):
    nx, ny, nz = _chk(U)
    dx, dy, dz = spacing or default_spacing(nx, ny, nz)
    L = np.zeros_like(U)
    hits = ctypes.c_longlong(0)
    rc = lib().orc_flux_divergence(_dp(U), nx, ny, nz, gamma, _bc(bc), dx, dy, dz, _dp(L), ctypes.byref(hits))
    if rc:
        raise MemoryError("oracle allocation failed")
    return L, hits.value


HEUN, VANLEER = "heun", "vanleer"   # Sec. 3.3


def step(U: np.ndarray, gamma, bc, dt, spacing=None, integrator=HEUN) -> int:
    """One step in place (Heun by default, van Leer predictor-corrector on request); returns the number of floor
    activations."""
    nx, ny, nz = _chk(U)
    dx, dy, dz = spacing or default_spacing(nx, ny, nz)
    hits = ctypes.c_longlong(0)
    fn = lib().orc_step_vl if integrator == VANLEER else lib().orc_step
    rc = fn(_dp(U), nx, ny, nz, gamma, _bc(bc), dx, dy, dz, dt, ctypes.byref(hits))
    if rc:
        raise MemoryError("oracle allocation failed")
    return hits.value


def cfl_dt(U: np.ndarray, gamma, cfl, spacing=None) -> float:
    nx, ny, nz = _chk(U)
    dx, dy, dz = spacing or default_spacing(nx, ny, nz)
    hits = ctypes.c_longlong(0)
    return lib().orc_cfl_dt(_dp(U), nx, ny, nz, gamma, dx, dy, dz, cfl, ctypes.byref(hits))


def run(U: np.ndarray, gamma, bc, cfl, nsteps, t0=0.0, t_end=0.0, spacing=None, integrator=HEUN):
    """Advance in place; returns (t, steps_taken, floor_hits)."""
    nx, ny, nz = _chk(U)
    dx, dy, dz = spacing or default_spacing(nx, ny, nz)
    t = ctypes.c_double(t0)
    hits = ctypes.c_longlong(0)
    fn = lib().orc_run_vl if integrator == VANLEER else lib().orc_run
    n = fn(_dp(U), nx, ny, nz, gamma, _bc(bc), dx, dy, dz, cfl, nsteps, t_end,
                      ctypes.byref(t), ctypes.byref(hits))
    if n < 0:
        raise MemoryError("oracle allocation failed")
    return t.value, n, hits.value


def totals(U: np.ndarray) -> np.ndarray:
    _chk(U)
    out = np.zeros(5)
    lib().orc_totals(_dp(U), U[0].size, _dp(out))
    return out


def num_threads() -> int:
    return lib().orc_num_threads()
