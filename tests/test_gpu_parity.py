"""GPU parity: the CUDA path (through the C-ABI) against the fp64 CPU oracle, element by element on
the same seeded inputs.  Tolerances are BASELINE.json's: relative L1 per conserved field
<= 1e-12 in all-fp64 mode, <= 1e-5 in mixed precision; conserved totals drift <= 1e-13.

Run with  python -m pytest tests -m gpu  on a B200 box.
"""
import math

import numpy as np
import pytest

import oracle
from paper_2501_02317_b200 import binding, inputs

pytestmark = pytest.mark.gpu

P, F, O, R = 0, 1, 2, 3
MIXED, FP64 = binding.PREC_MIXED, binding.PREC_FP64
SIMPLE, TILED, PAIRED, ROLES = (binding.KERNEL_SIMPLE, binding.KERNEL_TILED, binding.KERNEL_PAIRED,
                                binding.KERNEL_ROLES)
TMA = binding.KERNEL_TMA
KERNELS = [SIMPLE, TILED, PAIRED, ROLES]
TOL = {MIXED: 1e-5, FP64: 1e-12}


def rel_l1_fields(got, ref):
    """Per-field relative L1; fields identically zero in the oracle must be identically zero."""
    out = []
    for m in range(5):
        den = np.abs(ref[m]).sum()
        if den == 0.0:
            assert np.all(got[m] == 0.0), f"field {m} must stay exactly zero"
            out.append(0.0)
        else:
            out.append(float(np.abs(got[m] - ref[m]).sum() / den))
    return out


def make(pr, prec, kernel=binding.KERNEL_AUTO):
    if kernel in (PAIRED, ROLES) and prec != MIXED:
        pytest.skip("the paired and role-split kernels are the mixed-precision path")
    nx, ny, nz = pr.shape
    if kernel == ROLES and min(nx, ny, nz) == 1:
        pytest.skip("the role-split kernel is the 3D path")
    h = binding.KratosHydro(nx, ny, nz, pr.gamma, pr.bc, precision=prec, kernel=kernel)
    h.set_state(pr.U)
    return h


def lockstep(pr, prec, kernel, nsteps, cfl=0.4):
    """Both sides take the oracle's dt sequence (an input like any other); returns (gpu, oracle)."""
    Uo = pr.U.copy()
    h = make(pr, prec, kernel)
    for _ in range(nsteps):
        dt = oracle.cfl_dt(Uo, pr.gamma, cfl)
        oracle.step(Uo, pr.gamma, pr.bc, dt)
        h.step(dt)
    Ug = h.get_state()
    hits = h.floor_hits()
    h.destroy()
    return Ug, Uo, hits


# --------------------------------------------------------------------------- basics
def test_state_roundtrip_and_totals():
    pr = inputs.random_smooth(37, 21, 9, seed=1)
    h = make(pr, MIXED)
    np.testing.assert_array_equal(h.get_state(), pr.U)
    tot = h.totals()
    exact = np.array([math.fsum(pr.U[m].ravel()) for m in range(5)])
    np.testing.assert_allclose(tot, exact, rtol=2e-16, atol=1e-300)
    # device-resident buffers through torch
    import torch
    Ud = torch.from_numpy(pr.U).cuda()
    h.set_state(Ud * 2.0)
    out = torch.empty_like(Ud)
    h.get_state(out)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(out.cpu().numpy(), pr.U * 2.0)
    h.destroy()


@pytest.mark.parametrize("shape", [(1, 1, 50), (1, 40, 1), (33, 1, 1), (1, 24, 36), (20, 1, 17), (9, 21, 37)])
def test_cfl_dt_matches_oracle(shape):
    nz, ny, nx = shape
    pr = inputs.random_smooth(nx, ny, nz, seed=2)
    for prec in (MIXED, FP64):
        h = make(pr, prec)
        assert h.cfl_dt(0.4) == pytest.approx(oracle.cfl_dt(pr.U, pr.gamma, 0.4), rel=1e-13)
        h.destroy()


@pytest.mark.parametrize("prec", [MIXED, FP64])
@pytest.mark.parametrize("kernel", KERNELS)
def test_uniform_state_is_bitwise_fixed_point(prec, kernel):
    U0 = inputs.prim_to_cons(np.full((12, 20, 40), 1.3), 0.7, 0.4, -1.1, 2.2, 1.4)
    for bc in ((P,) * 6, (F,) * 6):
        pr = inputs.Problem("uniform", np.ascontiguousarray(U0), 1.4, bc)
        h = make(pr, prec, kernel)
        for _ in range(3):
            h.step(1e-3)
        np.testing.assert_array_equal(h.get_state(), U0)
        h.destroy()


# --------------------------------------------------------------------------- element-wise parity, small ragged cases
CASES_3D = [
    ((45, 19, 23), (P, P, P, P, P, P)),
    ((37, 33, 10), (F, F, O, O, R, R)),
    ((32, 16, 8), (R, O, P, P, F, R)),
    ((70, 35, 5), (O, R, F, O, P, P)),
]
CASES_2D = [((37, 21, 1), (P, P, P, P, P, P)), ((64, 48, 1), (R, R, O, F, P, P)), ((33, 5, 1), (F, O, R, R, P, P))]
CASES_ANY = [((50, 1, 1), (F, F, P, P, P, P)), ((1, 40, 1), (P, P, R, O, P, P)), ((1, 1, 33), (P, P, P, P, O, R)),
             ((24, 1, 18), (P, P, P, P, F, F)), ((1, 20, 22), (P, P, R, R, P, P))]


@pytest.mark.parametrize("prec", [MIXED, FP64])
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("shape,bc", CASES_3D + CASES_2D)
def test_parity_small_ragged(shape, bc, kernel, prec):
    nx, ny, nz = shape
    pr = inputs.random_smooth(nx, ny, nz, seed=nx + ny + nz, gamma=1.4, bc=bc)
    Ug, Uo, hits = lockstep(pr, prec, kernel, 5)
    assert hits == 0
    err = rel_l1_fields(Ug, Uo)
    assert max(err) <= TOL[prec], err


@pytest.mark.parametrize("prec", [MIXED, FP64])
@pytest.mark.parametrize("shape,bc", CASES_ANY)
def test_parity_other_axis_combinations(shape, bc, prec):
    """1D along y or z, x-z and y-z planes: served by the general (simple) kernel."""
    nx, ny, nz = shape
    pr = inputs.random_smooth(nx, ny, nz, seed=5, gamma=5.0 / 3.0, bc=bc)
    Ug, Uo, hits = lockstep(pr, prec, binding.KERNEL_AUTO, 6)
    assert hits == 0
    assert max(rel_l1_fields(Ug, Uo)) <= TOL[prec]


@pytest.mark.parametrize("kernel", [TILED, PAIRED, ROLES])
@pytest.mark.parametrize("zchunk", [1, 2, 4, 7, 16, 1000])
def test_slab_seams_do_not_change_the_result(zchunk, kernel):
    """Marching slabs of different height must give bit-identical states (one flux per face)."""
    pr = inputs.random_smooth(40, 20, 29, seed=8, gamma=1.4)
    ref = None
    for zc in (zchunk, 29):
        h = make(pr, MIXED, kernel)
        h.set_zchunk(zc)
        for _ in range(3):
            h.step(2e-3)
        U = h.get_state()
        h.destroy()
        if ref is None:
            ref = U
        else:
            np.testing.assert_array_equal(U, ref)


# --------------------------------------------------------------------------- the TMA kernel (nx % 32 == 0, ny % 16 == 0, 3D)
CASES_TMA = [
    ((32, 16, 8), (P, P, P, P, P, P)),       # a single tile: every halo box wraps onto the tile itself
    ((64, 48, 21), (P, P, P, P, P, P)),
    ((64, 32, 10), (F, F, O, O, R, R)),
    ((96, 32, 9), (R, O, P, P, F, R)),
    ((32, 64, 5), (O, R, F, O, P, P)),
    ((64, 32, 4), (R, R, R, R, R, R)),
]


@pytest.mark.parametrize("shape,bc", CASES_TMA)
def test_tma_kernel_parity(shape, bc):
    nx, ny, nz = shape
    pr = inputs.random_smooth(nx, ny, nz, seed=nx + ny + nz, gamma=1.4, bc=bc)
    Ug, Uo, hits = lockstep(pr, MIXED, TMA, 5)
    assert hits == 0
    err = rel_l1_fields(Ug, Uo)
    assert max(err) <= TOL[MIXED], err


@pytest.mark.parametrize("shape,bc", CASES_TMA[1:4])
def test_tma_kernel_equals_paired_kernel_to_rounding(shape, bc):
    """Same float_t arithmetic, different data movement: the two kernels may differ only by how the compiler
    contracts the fp64 flux accumulation (a few ulp of the state)."""
    nx, ny, nz = shape
    pr = inputs.random_smooth(nx, ny, nz, seed=11, gamma=5.0 / 3.0, bc=bc)
    out = []
    for kernel in (PAIRED, TMA):
        h = make(pr, MIXED, kernel)
        for n in range(7):
            h.step(1e-3 * (1.0 + 0.1 * n))
        out.append(h.get_state())
        h.destroy()
    for m in range(5):
        scale = np.abs(out[0][m]).max()
        assert np.abs(out[0][m] - out[1][m]).max() <= 1e-14 * max(scale, 1e-300)


@pytest.mark.parametrize("zchunk", [1, 2, 3, 5, 8, 1000])
def test_tma_kernel_slab_seams(zchunk):
    pr = inputs.random_smooth(64, 32, 29, seed=8, gamma=1.4)
    ref = None
    for zc in (zchunk, 29):
        h = make(pr, MIXED, TMA)
        h.set_zchunk(zc)
        for _ in range(3):
            h.step(2e-3)
        U = h.get_state()
        h.destroy()
        if ref is None:
            ref = U
        else:
            np.testing.assert_array_equal(U, ref)


def test_tma_kernel_conservation_and_auto_choice():
    pr = inputs.turbulence_3d(64, seed=7, nsteps=30)
    h = make(pr, MIXED)   # auto: the TMA kernel serves this block
    T0 = h.totals()
    A0 = np.array([math.fsum(np.abs(pr.U[m]).ravel()) for m in range(5)])
    h.run(0.4, 30)
    T1 = h.totals()
    h.destroy()
    drift = np.abs(T1 - T0) / np.maximum(np.abs(T0), A0)
    assert drift.max() <= 1e-13, drift
    # ragged blocks are refused by the TMA kernel, not silently served by another one
    pr2 = inputs.random_smooth(40, 20, 9, seed=1)
    with pytest.raises(Exception):
        binding.KratosHydro(40, 20, 9, pr2.gamma, pr2.bc, precision=MIXED, kernel=TMA)


def test_strong_jumps_take_every_hllc_branch():
    rng = np.random.default_rng(9)
    nz, ny, nx = 12, 18, 40
    rho = rng.uniform(0.1, 2.0, (nz, ny, nx))
    p = rng.uniform(0.05, 2.0, (nz, ny, nx))
    v = rng.uniform(-2.5, 2.5, (3, nz, ny, nx))
    U = np.ascontiguousarray(inputs.prim_to_cons(rho, p, v[0], v[1], v[2], 1.4))
    pr = inputs.Problem("jumps", U, 1.4, (P,) * 6)
    L, hits = oracle.flux_divergence(U, 1.4, pr.bc)
    assert hits == 0
    dt = 1e-4
    for kernel in KERNELS:
        for prec in (MIXED, FP64):
            if kernel in (PAIRED, ROLES) and prec != MIXED:
                continue
            h = make(pr, prec, kernel)
            h.step(dt)
            Ug = h.get_state()
            h.destroy()
            Uo = U.copy()
            oracle.step(Uo, 1.4, pr.bc, dt)
            # compare the increments: dU/dt against the oracle's
            num = np.abs((Ug - U) - (Uo - U)).sum(axis=(1, 2, 3))
            den = np.abs(Uo - U).sum(axis=(1, 2, 3))
            assert (num / den).max() <= (3e-6 if prec == MIXED else 1e-11)


# --------------------------------------------------------------------------- configs (reduced twins)
@pytest.mark.parametrize("prec", [MIXED, FP64])
@pytest.mark.parametrize("seed", [1, 2, 3, 4])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_c1_riemann_1d(seed, axis, prec):
    """C1: 256 cells, gamma 1.4, Free BC, cfl 0.4, t = 0.2 -- self-driven run on both sides."""
    if axis != 0 and seed > 2:
        pytest.skip("axis interchange covered with two seeds")
    pr = inputs.riemann_1d(seed, 256, axis=axis)
    Uo = pr.U.copy()
    to, no, _ = oracle.run(Uo, pr.gamma, pr.bc, 0.4, 10 ** 6, 0.0, 0.2)
    h = make(pr, prec)
    tg, ng = h.run_until(0.4, 0.2)
    Ug = h.get_state()
    assert h.floor_hits() == 0
    h.destroy()
    assert tg == pytest.approx(0.2, abs=1e-15)
    assert abs(ng - no) <= (0 if prec == FP64 else 1)
    assert max(rel_l1_fields(Ug, Uo)) <= TOL[prec]


@pytest.mark.parametrize("prec", [MIXED, FP64])
def test_c2_advected_wave_reduced(prec):
    pr = inputs.advected_wave_2d(64, t_end=0.5)
    Uo = pr.U.copy()
    oracle.run(Uo, pr.gamma, pr.bc, 0.4, 10 ** 6, 0.0, 0.5)
    h = make(pr, prec)
    tg, _ = h.run_until(0.4, 0.5)
    Ug = h.get_state()
    h.destroy()
    assert tg == 0.5
    assert max(rel_l1_fields(Ug, Uo)) <= TOL[prec]


@pytest.mark.parametrize("prec", [MIXED, FP64])
def test_c3_shear_layer_reduced(prec):
    pr = inputs.shear_layer_2d(256, seed=3, nsteps=100)
    Uo = pr.U.copy()
    oracle.run(Uo, pr.gamma, pr.bc, 0.4, 100)
    h = make(pr, prec)
    h.run(0.4, 100)
    Ug = h.get_state()
    h.destroy()
    assert max(rel_l1_fields(Ug, Uo)) <= TOL[prec]


@pytest.mark.parametrize("prec", [MIXED, FP64])
def test_c4_point_blast_reduced(prec):
    pr = inputs.point_blast_3d(64, nsteps=50)
    Uo = pr.U.copy()
    _, _, hits_o = oracle.run(Uo, pr.gamma, pr.bc, 0.4, 50)
    h = make(pr, prec)
    h.run(0.4, 50)
    Ug = h.get_state()
    hits = h.floor_hits()
    h.destroy()
    assert hits == 0 and hits_o == 0
    assert max(rel_l1_fields(Ug, Uo)) <= TOL[prec]


@pytest.mark.parametrize("prec", [MIXED, FP64])
def test_c5_turbulence_reduced(prec):
    pr = inputs.turbulence_3d(64, seed=5, nsteps=20)
    Uo = pr.U.copy()
    oracle.run(Uo, pr.gamma, pr.bc, 0.4, 20)
    h = make(pr, prec)
    h.run(0.4, 20)
    Ug = h.get_state()
    h.destroy()
    assert max(rel_l1_fields(Ug, Uo)) <= TOL[prec]


# --------------------------------------------------------------------------- conservation (P3) on the GPU
@pytest.mark.parametrize("prec", [MIXED, FP64])
@pytest.mark.parametrize("kernel", KERNELS)
def test_periodic_conservation(prec, kernel):
    pr = inputs.turbulence_3d(48, seed=7, nsteps=30)
    h = make(pr, prec, kernel)
    T0 = h.totals()
    A0 = np.array([math.fsum(np.abs(pr.U[m]).ravel()) for m in range(5)])
    h.run(0.4, 30)
    T1 = h.totals()
    U = h.get_state()
    h.destroy()
    np.testing.assert_allclose(T1, [math.fsum(U[m].ravel()) for m in range(5)], rtol=2e-16, atol=1e-18 * A0.max())
    drift = np.abs(T1 - T0) / np.maximum(np.abs(T0), A0)
    assert drift.max() <= 1e-13, drift


def test_run_equals_manual_stepping_in_fp64():
    """run() (device-resident dt) and cfl_dt()+step() give the same bits in all-fp64 mode."""
    pr = inputs.random_smooth(40, 24, 12, seed=4)
    h1 = make(pr, FP64)
    t1 = h1.run(0.4, 6)
    h2 = make(pr, FP64)
    t2 = 0.0
    for _ in range(6):
        dt = h2.cfl_dt(0.4)
        h2.step(dt)
        t2 += dt
    np.testing.assert_array_equal(h1.get_state(), h2.get_state())
    assert t1 == pytest.approx(t2, rel=1e-15)
    h1.destroy()
    h2.destroy()


def test_step_rejects_bad_dt_and_nonfinite_state_is_reported():
    pr = inputs.random_smooth(32, 16, 1, seed=4)
    h = make(pr, MIXED)
    for bad in (0.0, -1.0, float("nan"), float("inf")):
        with pytest.raises(binding.KratosError) as ei:
            h.step(bad)
        assert ei.value.code == binding.ERR_ARG
    U = pr.U.copy()
    U[0, 0, 3, 3] = float("nan")
    h.set_state(U)
    with pytest.raises(binding.KratosError) as ei:
        h.cfl_dt(0.4)
    assert ei.value.code == binding.ERR_NONFINITE
    h.destroy()


# --------------------------------------------------------------------------- full size, the launch configuration bench.py times
def test_c5_full_size_sampled_against_oracle():
    """C5 at BASELINE.json's size (512^3 periodic, mixed precision, auto kernel and slab height = what bench.py
    times): two Heun steps on the GPU; sampled 12^3 sub-blocks are recomputed by the oracle from the initial
    state of their domain of dependence (2 steps x 2 stages x 2 cells = 8 cells each side), with the same dt
    sequence.  Conserved totals of the whole block must not drift."""
    n, nstep, halo, core = 512, 2, 8, 12
    try:
        pr = inputs.turbulence_3d(n, seed=5, nsteps=nstep)
    except MemoryError:
        pytest.skip("not enough host memory for the 512^3 state")
    h = make(pr, MIXED)
    T0 = h.totals()
    dts = []
    for _ in range(nstep):
        dts.append(h.cfl_dt(0.4))   # fp64 rate maximum over the whole block (matches the oracle's to 1e-13)
        h.step(dts[-1])
    T1 = h.totals()
    Ug = h.get_state()
    assert h.floor_hits() == 0
    h.destroy()
    A0 = np.array([float(np.abs(pr.U[m]).sum()) for m in range(5)])
    assert (np.abs(T1 - T0) / np.maximum(np.abs(T0), A0)).max() <= 1e-13
    # the first dt against the oracle's own reduction over the full state
    assert dts[0] == pytest.approx(oracle.cfl_dt(pr.U, pr.gamma, 0.4), rel=1e-13)
    rng = np.random.default_rng(123)
    w = core + 2 * halo
    corners = [(0, 0, 0), (n - core, n - core, n - core), (250, 9, 121)]   # tile / slab seams and the periodic wrap
    corners += [tuple(int(c) for c in rng.integers(0, n, 3)) for _ in range(5)]
    for (k0, j0, i0) in corners:
        kk = (np.arange(k0 - halo, k0 - halo + w)) % n
        jj = (np.arange(j0 - halo, j0 - halo + w)) % n
        ii = (np.arange(i0 - halo, i0 - halo + w)) % n
        sub = np.ascontiguousarray(pr.U[:, kk][:, :, jj][:, :, :, ii])
        for dt in dts:
            # free boundaries on the sub-block: wrong only within 4 cells of its faces per step
            oracle.step(sub, pr.gamma, (F,) * 6, dt, spacing=(1.0 / n,) * 3)
        ref = sub[:, halo:halo + core, halo:halo + core, halo:halo + core]
        kc = (np.arange(k0, k0 + core)) % n
        jc = (np.arange(j0, j0 + core)) % n
        ic = (np.arange(i0, i0 + core)) % n
        got = Ug[:, kc][:, :, jc][:, :, :, ic]
        err = rel_l1_fields(got, ref)
        assert max(err) <= TOL[MIXED], ((k0, j0, i0), err)


# --------------------------------------------------------------------------- Sec. 4.4 Liska-Wendroff implosion (reflecting walls)
@pytest.mark.parametrize("prec", [MIXED, FP64])
def test_implosion_2d_reduced(prec):
    """Eq. 7 at 128^2 in a box of reflecting walls (BC code 3 on all four sides): parity with the
    oracle while the flow is still deterministic, closed-box conservation of mass and energy, and in all-fp64 mode
    the diagonal symmetry rho(x,y) = rho(y,x), m_x(x,y) = m_y(y,x) to rounding."""
    n, nsteps = 128, 80
    pr = inputs.implosion_2d(n, nsteps=nsteps)
    Uo = pr.U.copy()
    _, _, hits_o = oracle.run(Uo, pr.gamma, pr.bc, 0.4, nsteps)
    h = make(pr, prec)
    T0 = h.totals()
    h.run(0.4, nsteps)
    T1 = h.totals()
    Ug = h.get_state()
    hits = h.floor_hits()
    h.destroy()
    assert hits == 0 and hits_o == 0
    assert max(rel_l1_fields(Ug, Uo)) <= TOL[prec]
    assert abs(T1[0] - T0[0]) <= 1e-13 * T0[0] and abs(T1[4] - T0[4]) <= 1e-13 * T0[4]
    if prec == FP64:
        rho, mx, my, e = Ug[0][0], Ug[1][0], Ug[2][0], Ug[4][0]
        assert np.abs(rho - rho.T).max() <= 1e-12
        assert np.abs(mx - my.T).max() <= 1e-12
        assert np.abs(e - e.T).max() <= 1e-12


def test_implosion_extruded_through_the_tma_kernel():
    """The same problem extruded along z (periodic): the 3D TMA kernel with reflecting boxes in x and y must reproduce
    the 2D oracle run in every z plane, with the z momentum exactly zero."""
    n, nzz, nsteps = 64, 8, 40
    pr2 = inputs.implosion_2d(n, nsteps=nsteps)
    Uo = pr2.U.copy()
    U3 = np.ascontiguousarray(np.repeat(pr2.U, nzz, axis=1))
    pr3 = inputs.Problem("implosion_extruded", U3, pr2.gamma, pr2.bc)
    h = make(pr3, MIXED, TMA)
    h.set_spacing(1.0 / n, 1.0 / n, 1.0 / n)
    for _ in range(nsteps):
        dt = oracle.cfl_dt(Uo, pr2.gamma, 0.4)
        oracle.step(Uo, pr2.gamma, pr2.bc, dt)
        h.step(dt)
    Ug = h.get_state()
    h.destroy()
    assert np.all(Ug[3] == 0.0)
    for k in range(nzz):
        assert np.array_equal(Ug[:, k], Ug[:, 0])          # every plane the same bits
    assert max(rel_l1_fields(Ug[:, :1], Uo)) <= TOL[MIXED]


# --------------------------------------------------------------------------- Sec. 3.3 van Leer integrator (reading S15)
VL = binding.INTEGRATOR_VANLEER
CASES_VL = [((45, 19, 23), (P, P, P, P, P, P)), ((37, 33, 10), (F, F, O, O, R, R)), ((64, 32, 8), (R, O, P, P, F, R)),
            ((64, 48, 21), (P, P, P, P, P, P)), ((96, 32, 9), (F, F, O, O, R, R)),
            ((37, 21, 1), (P, P, P, P, P, P)), ((64, 48, 1), (R, R, O, F, P, P)), ((50, 1, 1), (F, F, P, P, P, P)),
            ((1, 20, 22), (P, P, R, R, P, P))]


@pytest.mark.parametrize("prec", [MIXED, FP64])
@pytest.mark.parametrize("shape,bc", CASES_VL)
def test_vanleer_parity(shape, bc, prec):
    """Predictor kept as float_t primitives, corrector in place: element-wise against the
    oracle's van Leer step with the oracle's dt sequence."""
    nx, ny, nz = shape
    pr = inputs.random_smooth(nx, ny, nz, seed=nx + ny + nz, gamma=1.4, bc=bc)
    Uo = pr.U.copy()
    hs = [binding.KratosHydro(nx, ny, nz, pr.gamma, pr.bc, precision=prec, integrator=VL)]
    if prec == MIXED and nx % 32 == 0 and ny % 16 == 0 and nz > 1:   # auto = TMA predictor: also the general kernels
        hs.append(binding.KratosHydro(nx, ny, nz, pr.gamma, pr.bc, precision=prec, integrator=VL, kernel=SIMPLE))
    for h in hs:
        h.set_state(pr.U)
    for _ in range(5):
        dt = oracle.cfl_dt(Uo, pr.gamma, 0.4)
        oracle.step(Uo, pr.gamma, pr.bc, dt, integrator=oracle.VANLEER)
        for h in hs:
            h.step(dt)
    for h in hs:
        Ug = h.get_state()
        assert h.floor_hits() == 0
        h.destroy()
        err = rel_l1_fields(Ug, Uo)
        assert max(err) <= TOL[prec], err


@pytest.mark.parametrize("prec", [MIXED, FP64])
def test_vanleer_run_conservation_and_fixed_point(prec):
    # device-resident dt (run) against the oracle's run, and conservation "up to the full machine accuracy"
    pr = inputs.turbulence_3d(32, seed=7, nsteps=20)
    Uo = pr.U.copy()
    oracle.run(Uo, pr.gamma, pr.bc, 0.4, 20, integrator=oracle.VANLEER)
    h = binding.KratosHydro(32, 32, 32, pr.gamma, pr.bc, precision=prec, integrator=VL)
    h.set_state(pr.U)
    T0 = h.totals()
    A0 = np.array([math.fsum(np.abs(pr.U[m]).ravel()) for m in range(5)])
    h.run(0.4, 20)
    T1 = h.totals()
    Ug = h.get_state()
    h.destroy()
    assert max(rel_l1_fields(Ug, Uo)) <= TOL[prec]
    assert (np.abs(T1 - T0) / np.maximum(np.abs(T0), A0)).max() <= 1e-13
    # uniform state: bitwise fixed point
    U0 = np.ascontiguousarray(inputs.prim_to_cons(np.full((12, 20, 40), 1.3), 0.7, 0.4, -1.1, 2.2, 1.4))
    h = binding.KratosHydro(40, 20, 12, 1.4, (P,) * 6, precision=prec, integrator=VL)
    h.set_state(U0)
    for _ in range(3):
        h.step(1e-3)
    np.testing.assert_array_equal(h.get_state(), U0)
    h.destroy()


def test_vanleer_refuses_the_heun_stage_kernels_and_bad_scheme_words():
    pr = inputs.random_smooth(64, 32, 8, seed=1)
    h = binding.KratosHydro(64, 32, 8, pr.gamma, pr.bc, precision=MIXED, integrator=VL)
    for k in (TILED, PAIRED, ROLES):
        with pytest.raises(Exception):
            h.set_kernel(k)
    h.set_kernel(TMA)      # the predictor on the TMA machinery (this block qualifies) ...
    h.set_kernel(SIMPLE)   # ... or both sub-steps through the general kernels
    h.destroy()
    with pytest.raises(Exception):
        binding.KratosHydro(64, 32, 8, pr.gamma, pr.bc, precision=MIXED, integrator=2 << 4)


@pytest.mark.parametrize("zchunk", [1, 3, 8, 1000])
def test_vanleer_tma_slab_seams_and_general_kernels_agree(zchunk):
    """van Leer on the TMA kernel: slabs of any height give the same bits, and the result agrees with the general
    one-thread-per-cell kernels to float_t rounding of the stored predictor."""
    pr = inputs.random_smooth(64, 32, 21, seed=8, gamma=1.4, bc=(R, O, P, P, F, R))
    outs = []
    for kern, zc in ((TMA, zchunk), (TMA, 21), (SIMPLE, 0)):
        h = binding.KratosHydro(64, 32, 21, pr.gamma, pr.bc, precision=MIXED, integrator=VL, kernel=kern)
        if zc:
            h.set_zchunk(zc)
        h.set_state(pr.U)
        for _ in range(3):
            h.step(2e-3)
        outs.append(h.get_state())
        h.destroy()
    np.testing.assert_array_equal(outs[0], outs[1])
    assert max(rel_l1_fields(outs[0], outs[2])) <= 1e-6


# --------------------------------------------------------------------------- seeded random blocks through the TMA kernels
@pytest.mark.parametrize("integrator", ["heun", "vanleer"])
def test_random_blocks_boundaries_spacings_and_slabs(integrator):
    """Twelve seeded random combinations of extent (multiples of the 32 x 16 tile), boundary rules per face, cell
    aspect ratio, gamma and slab height: the TMA kernels with the device-resident dt against the oracle's run."""
    rng = np.random.default_rng(77 if integrator == "heun" else 78)
    vl = integrator == "vanleer"
    for it in range(12):
        nx, ny, nz = 32 * int(rng.integers(1, 4)), 16 * int(rng.integers(1, 4)), int(rng.integers(4, 30))
        bc = []
        for _ in range(3):
            bc += [0, 0] if rng.random() < 0.4 else [int(rng.integers(1, 4)), int(rng.integers(1, 4))]
        zc = int(rng.choice([0, 1, 2, 3, 5, 7, 11, 16]))
        pr = inputs.random_smooth(nx, ny, nz, seed=100 + it, gamma=float(rng.choice([1.4, 5 / 3, 1.1])), bc=tuple(bc))
        sp = (1.0 / nx, float(rng.uniform(0.5, 2)) / ny, float(rng.uniform(0.5, 2)) / nz)
        h = binding.KratosHydro(nx, ny, nz, pr.gamma, pr.bc, precision=MIXED, spacing=sp, kernel=TMA,
                                integrator=VL if vl else binding.INTEGRATOR_HEUN)
        if zc:
            h.set_zchunk(zc)
        h.set_state(pr.U)
        T0 = h.totals()
        h.run(0.4, 6)
        Ug, T1, hits = h.get_state(), h.totals(), h.floor_hits()
        h.destroy()
        Uo = pr.U.copy()
        oracle.run(Uo, pr.gamma, pr.bc, 0.4, 6, spacing=sp, integrator=oracle.VANLEER if vl else oracle.HEUN)
        assert hits == 0 and np.isfinite(Ug).all()
        assert max(rel_l1_fields(Ug, Uo)) <= TOL[MIXED], (it, (nx, ny, nz), bc, zc)
        if all(b == 0 for b in bc):
            assert abs(T1[0] - T0[0]) <= 1e-13 * abs(T0[0]) and abs(T1[4] - T0[4]) <= 1e-13 * abs(T0[4])
