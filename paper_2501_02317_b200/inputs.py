"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs C1..C5).

This module serves BOTH the oracle-side tests and the CUDA path, and therefore holds
none of the method's arithmetic: no primitive recovery, reconstruction, Riemann solver,
update or time-step formula.  It only lays out an initial state on the unit box
(cell centres x_i = (i + 1/2) dx, dx = 1/n per active axis) and stores it as the
conserved array the C-ABI boundary takes,

    U[5, nz, ny, nx] = (rho, rho v_x, rho v_y, rho v_z, eps),  eps = p/(gamma-1) + rho v^2/2

(the definition of the total energy density).  Random numbers come from
``torch.Generator().manual_seed(seed)`` on the CPU in fp64, so the same seed gives the
same bits on every machine.  Everything is imported lazily so that neither the CUDA
extension nor the oracle is pulled in.

Shapes follow the paper's tests: 1D shock tubes, 2D 2048^2
Kelvin-Helmholtz-like shear layers, 3D 256^3-class uniform boxes
(PAPER.md:384-439).  The paper's own problem data (Toro's tables, Woodward-Colella) are
not reproduced; these seeded states stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

PERIODIC, FREE, OUTFLOW, REFLECT = 0, 1, 2, 3


@dataclass
class Problem:
    name: str
    U: np.ndarray            # [5, nz, ny, nx] float64, C-contiguous
    gamma: float
    bc: tuple                # (x-lo, x-hi, y-lo, y-hi, z-lo, z-hi)
    cfl: float = 0.4
    nsteps: int = 0          # fixed step count (0: run to t_end)
    t_end: float = 0.0       # end time (0: run nsteps)
    meta: dict = field(default_factory=dict)

    @property
    def shape(self):
        _, nz, ny, nx = self.U.shape
        return nx, ny, nz

    @property
    def spacing(self):
        return tuple(1.0 / n if n > 1 else 1.0 for n in self.shape)

    @property
    def ncell(self):
        return int(self.U[0].size)


def prim_to_cons(rho, p, vx, vy, vz, gamma) -> np.ndarray:
    """Pack primitive fields (any common shape [nz,ny,nx]) into U[5,nz,ny,nx]."""
    rho = np.asarray(rho, dtype=np.float64)
    shp = rho.shape
    U = np.empty((5,) + shp, dtype=np.float64)
    vx = np.broadcast_to(np.asarray(vx, dtype=np.float64), shp)
    vy = np.broadcast_to(np.asarray(vy, dtype=np.float64), shp)
    vz = np.broadcast_to(np.asarray(vz, dtype=np.float64), shp)
    p = np.broadcast_to(np.asarray(p, dtype=np.float64), shp)
    U[0] = rho
    U[1] = rho * vx
    U[2] = rho * vy
    U[3] = rho * vz
    U[4] = p / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)
    return U


def centres(n: int) -> np.ndarray:
    return (np.arange(n, dtype=np.float64) + 0.5) / n


def _randn(seed: int, *shape) -> np.ndarray:
    import torch
    g = torch.Generator().manual_seed(int(seed))
    return torch.randn(*shape, generator=g, dtype=torch.float64).numpy()


def _rand(seed: int, *shape) -> np.ndarray:
    import torch
    g = torch.Generator().manual_seed(int(seed))
    return torch.rand(*shape, generator=g, dtype=torch.float64).numpy()


# ----------------------------------------------------------------------------- C1
def riemann_states(seed: int):
    """Left/right (rho, u, p): rho ~ U[0.1,1], u ~ U[-1,1], p ~ U[0.1,1] (BASELINE.json config 1)."""
    r = _rand(seed, 6)
    rho_l, rho_r = 0.1 + 0.9 * r[0], 0.1 + 0.9 * r[1]
    u_l, u_r = -1.0 + 2.0 * r[2], -1.0 + 2.0 * r[3]
    p_l, p_r = 0.1 + 0.9 * r[4], 0.1 + 0.9 * r[5]
    return (float(rho_l), float(u_l), float(p_l)), (float(rho_r), float(u_r), float(p_r))


def riemann_1d(seed: int = 1, n: int = 256, axis: int = 0, states=None, gamma: float = 1.4,
               t_end: float = 0.2, bc_code: int = FREE) -> Problem:
    """C1: 1D two-state discontinuity at 0.5 along ``axis`` (0=x, 1=y, 2=z), gamma = 1.4."""
    (rl, ul, pl), (rr, ur, pr) = states if states is not None else riemann_states(seed)
    x = centres(n)
    left = x < 0.5
    rho = np.where(left, rl, rr)
    u = np.where(left, ul, ur)
    p = np.where(left, pl, pr)
    shp = [1, 1, 1]
    shp[2 - axis] = n  # array order is [z, y, x]
    rho, u, p = rho.reshape(shp), u.reshape(shp), p.reshape(shp)
    v = [0.0, 0.0, 0.0]
    v[axis] = u
    U = prim_to_cons(rho, p, v[0], v[1], v[2], gamma)
    bc = [PERIODIC] * 6
    bc[2 * axis] = bc[2 * axis + 1] = bc_code
    return Problem("C1_riemann_1d", np.ascontiguousarray(U), gamma, tuple(bc), t_end=t_end,
                   meta=dict(left=(rl, ul, pl), right=(rr, ur, pr), axis=axis, n=n, seed=seed))


# ----------------------------------------------------------------------------- waves
def wave_1d(n: int, kind: str = "contact", amplitude: float = 0.1, shape: str = "sin",
            v0: float = 1.0, axis: int = 0) -> Problem:
    """Sec. 4.1 eigen-waves: rho0 = 1, p0 = 5/3, gamma = 5/3, L = 1, periodic.
    contact: only rho varies, advected at v0.  shear: only a tangential velocity varies.
    sound: right-going linear sound wave on a gas at rest (period 1 since c0 = 5/3... see note)."""
    gamma = 5.0 / 3.0
    rho0, p0 = 1.0, 5.0 / 3.0
    x = centres(n)
    dq = amplitude * np.sin(2 * np.pi * x) if shape == "sin" else np.where(x < 0.5, amplitude, 0.0)
    rho = np.full(n, rho0)
    p = np.full(n, p0)
    un = np.full(n, v0)
    ut = np.zeros(n)
    if kind == "contact":
        rho = rho0 + dq
    elif kind == "shear":
        ut = dq.copy()
    elif kind == "sound":
        c0 = np.sqrt(gamma * p0 / rho0)
        rho = rho0 + dq
        p = p0 + c0 * c0 * dq
        un = v0 + c0 * dq / rho0
    else:
        raise ValueError(kind)
    shp = [1, 1, 1]
    shp[2 - axis] = n
    v = [np.zeros(n).reshape(shp)] * 3
    v = list(v)
    v[axis] = un.reshape(shp)
    v[(axis + 1) % 3] = ut.reshape(shp)
    U = prim_to_cons(rho.reshape(shp), p.reshape(shp), v[0], v[1], v[2], gamma)
    return Problem("wave_1d_" + kind, np.ascontiguousarray(U), gamma, (PERIODIC,) * 6, t_end=1.0,
                   meta=dict(kind=kind, amplitude=amplitude, shape=shape, v0=v0, axis=axis, n=n))


# ----------------------------------------------------------------------------- C2
def advected_wave_2d(n: int = 512, t_end: float = 1.0) -> Problem:
    """C2: rho = 1 + 0.2 sin(2 pi (x+y)), p = 1, v = (1,1,0), gamma = 5/3, periodic unit box."""
    gamma = 5.0 / 3.0
    x = centres(n)
    X, Y = np.meshgrid(x, x, indexing="xy")  # [y, x]
    rho = (1.0 + 0.2 * np.sin(2 * np.pi * (X + Y)))[None]
    U = prim_to_cons(rho, 1.0, 1.0, 1.0, 0.0, gamma)
    return Problem("C2_advected_wave_2d", np.ascontiguousarray(U), gamma, (PERIODIC,) * 6,
                   t_end=t_end, meta=dict(n=n))


# ----------------------------------------------------------------------------- C3
def shear_layer_2d(n: int = 2048, seed: int = 3, nsteps: int = 100) -> Problem:
    """C3: rho = 2 for |y-0.5| < 0.25 else 1; v_x = +0.5 inside / -0.5 outside; p = 2.5;
    v_y = 0.01 * N(0,1) per cell; gamma = 5/3; periodic."""
    gamma = 5.0 / 3.0
    y = centres(n)
    inside = (np.abs(y - 0.5) < 0.25)[:, None]
    rho = np.where(inside, 2.0, 1.0) * np.ones((n, n))
    vx = np.where(inside, 0.5, -0.5) * np.ones((n, n))
    vy = 0.01 * _randn(seed, n, n)
    U = prim_to_cons(rho[None], 2.5, vx[None], vy[None], 0.0, gamma)
    return Problem("C3_shear_layer_2d", np.ascontiguousarray(U), gamma, (PERIODIC,) * 6,
                   nsteps=nsteps, meta=dict(n=n, seed=seed))


# ----------------------------------------------------------------------------- C4
def point_blast_3d(n: int = 256, nsteps: int = 50, bc_code: int = OUTFLOW) -> Problem:
    """C4: rho = 1, v = 0, p = 1e-5; thermal energy 1.0 spread uniformly over the cells whose
    centre is within 3 cells of the box centre; gamma = 5/3; outflow on all sides."""
    gamma = 5.0 / 3.0
    x = centres(n)
    dx = 1.0 / n
    r2 = ((x[:, None, None] - 0.5) ** 2 + (x[None, :, None] - 0.5) ** 2 + (x[None, None, :] - 0.5) ** 2)
    hot = r2 < (3.0 * dx) ** 2
    count = int(hot.sum())
    eg = np.full((n, n, n), 1e-5 / (gamma - 1.0))
    eg[hot] = 1.0 / (count * dx ** 3)
    p = (gamma - 1.0) * eg
    U = prim_to_cons(np.ones((n, n, n)), p, 0.0, 0.0, 0.0, gamma)
    return Problem("C4_point_blast_3d", np.ascontiguousarray(U), gamma, (bc_code,) * 6,
                   nsteps=nsteps, meta=dict(n=n, hot_cells=count))


# ----------------------------------------------------------------------------- C5
def _gaussian_field(seed: int, n: int, kmax: int = 8) -> np.ndarray:
    """Real field [z,y,x] = Re sum_k A_k exp(2 pi i k.x) over integer modes 1 <= |k| <= kmax with
    independent complex Gaussian A_k of variance |k|^-2 (taking the real part is the Hermitian
    symmetrisation).  Evaluated as three small separable contractions."""
    ks = np.arange(-kmax, kmax + 1)
    KZ, KY, KX = np.meshgrid(ks, ks, ks, indexing="ij")
    kk = np.sqrt((KX ** 2 + KY ** 2 + KZ ** 2).astype(np.float64))
    mask = (kk >= 1.0) & (kk <= kmax)
    amp = np.where(mask, 1.0 / np.where(kk > 0, kk, 1.0), 0.0)
    g = _randn(seed, 2, ks.size, ks.size, ks.size)
    A = amp * (g[0] + 1j * g[1])                       # [kz, ky, kx]
    x = centres(n)
    E = np.exp(2j * np.pi * np.outer(x, ks))            # [n, k]
    T1 = np.einsum("abc,xc->abx", A, E)                 # [kz, ky, x]
    T2 = np.einsum("abx,yb->ayx", T1, E)                # [kz, y, x]
    T2 = T2.reshape(ks.size, n * n)
    out = E.real @ T2.real - E.imag @ T2.imag           # [z, y*x]
    return out.reshape(n, n, n)


def turbulence_3d(n: int = 512, seed: int = 5, nsteps: int = 20, gamma: float = 1.001) -> Problem:
    """C5: rho = 1, p = 1, random-phase Gaussian velocity with per-mode power ~ k^-2 on
    1 <= |k| <= 8, scaled to rms Mach 1; gamma = 1.001; periodic."""
    v = [_gaussian_field(seed * 1000 + c, n) for c in range(3)]
    cs = np.sqrt(gamma * 1.0 / 1.0)
    rms = np.sqrt(np.mean(v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    for c in range(3):
        v[c] *= cs / rms
    U = prim_to_cons(np.ones((n, n, n)), 1.0, v[0], v[1], v[2], gamma)
    return Problem("C5_turbulence_3d", np.ascontiguousarray(U), gamma, (PERIODIC,) * 6,
                   nsteps=nsteps, meta=dict(n=n, seed=seed))


# ----------------------------------------------------------------------------- Liska-Wendroff implosion
def implosion_2d(n: int = 400, nsteps: int = 0, t_end: float = 0.045 / 0.3) -> Problem:
    """Sec. 4.4, Eq. 7: gamma = 1.4, (rho, p) = (0.125, 0.14) where x + y < 0.15 and (1, 1)
    elsewhere, gas at rest, reflecting walls on all four sides.  The test lives on the box [0, 0.3]^2; the Euler
    equations carry no length scale, so it is set up here on the unit box used everywhere in this package
    (corner region x + y < 1/2) and times scale by 1/0.3 (t = 0.045 there is t = 0.15 here).  Cell centres
    exactly on the diagonal x + y = 1/2 do not occur for even n."""
    gamma = 1.4
    x = centres(n)
    corner = (x[None, :] + x[:, None]) < 0.5          # [y, x]
    rho = np.where(corner, 0.125, 1.0)[None]
    p = np.where(corner, 0.14, 1.0)[None]
    U = prim_to_cons(rho, p, 0.0, 0.0, 0.0, gamma)
    return Problem("implosion_2d", np.ascontiguousarray(U), gamma, (REFLECT, REFLECT, REFLECT, REFLECT, PERIODIC, PERIODIC),
                   nsteps=nsteps, t_end=(0.0 if nsteps else t_end), meta=dict(n=n))


# ----------------------------------------------------------------------------- misc small cases
def random_smooth(nx: int, ny: int, nz: int, seed: int, gamma: float = 1.4, bc=(PERIODIC,) * 6,
                  amp: float = 0.3) -> Problem:
    """Generic ragged-size test state: O(1) background plus a few random low-k modes and a weak
    per-cell noise in every primitive; positive rho, p by construction."""
    r = _randn(seed, 5, nz, ny, nx)
    zc, yc, xc = centres(nz)[:, None, None], centres(ny)[None, :, None], centres(nx)[None, None, :]
    ph = _rand(seed + 7, 5, 3) * 2 * np.pi
    f = []
    for m in range(5):
        s = np.sin(2 * np.pi * xc + ph[m, 0]) * (nx > 1) + np.sin(2 * np.pi * yc + ph[m, 1]) * (ny > 1) \
            + np.sin(2 * np.pi * zc + ph[m, 2]) * (nz > 1)
        f.append(amp * s / 3.0 + 0.02 * r[m])
    rho = 1.0 + f[0]
    p = 1.0 + f[1]
    vx = f[2] * 2.0 * (nx > 1)
    vy = f[3] * 2.0 * (ny > 1)
    vz = f[4] * 2.0 * (nz > 1)
    U = prim_to_cons(rho, p, vx, vy, vz, gamma)
    return Problem("random_smooth", np.ascontiguousarray(U), gamma, tuple(bc), nsteps=4,
                   meta=dict(seed=seed))
