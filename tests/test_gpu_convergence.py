"""The paper's convergence experiment (Sec. 4.1, Eq. 6, Fig. 7) on the CUDA path.

Sinusoidal sound, contact and shear waves on the periodic unit interval (rho0 = 1, p0 = 5/3, gamma = 5/3) are evolved for
one crossing time and compared with their initial state in the normalised L1 norm of Eq. 6, at N = 64 ... 1024 cells, in
all three precision modes of the library (all-fp64, mixed, all-fp32 "Single").  What the paper states and this file checks:

  * contact and shear waves, A = 0.1: L1 ~ N^-2, and "the L1 errors of mixed-precision methods are almost identical to the
    full double-precision methods";
  * sound wave, all-fp64, A = 1e-6: L1 ~ N^-2 up to N > 10^3;
  * sound wave, mixed and Single, A = 1e-4: the errors stop falling "with resolutions higher than N ~ 10^2".  This last
    statement is about Kratos' plain fp32 solver; where this library's mixed mode (pressure carried as a deviation from a
    reference pressure, reading S14) and its Single mode leave the N^-2 line is RECORDED here, not asserted --
    next to the all-fp64 run at the same amplitude, which separates rounding from the wave's own nonlinear steepening.

The oracle is pinned by the same experiment (tests/test_oracle_pins.py, P2); here the all-fp64 CUDA run must reproduce the
oracle's error at the sizes the oracle does in a blink, and the other modes are measured against it.  Every run goes through
kratos_hydro_run_until (device-resident dt, landing exactly on the crossing time).  The table is written to
convergence.jsonl in the folder KRATOS_PARITY_RECORD_DIR names (profiles/r3_convergence.md is made from it).
"""
import json
import math
import os

import numpy as np
import pytest

import oracle
from paper_2501_02317_b200 import binding, inputs

pytestmark = pytest.mark.gpu

NS = (64, 128, 256, 512, 1024)
MODES = {"fp64": binding.PREC_FP64, "mixed": binding.PREC_MIXED, "single": binding.PREC_SINGLE}


def paper_l1(q, q0):
    """Eq. 6."""
    return float(np.abs(q - q0).sum() / (q.size * (q0.max() - q0.min())))


def problem(kind, n, amplitude):
    """(Problem, crossing time, field index to measure, divide by rho?).  The sound wave runs on a gas at rest, so that the
    eigenmode's speed is c0 = 5/3 and one crossing takes 0.6; contact and shear waves are advected at v0 = 1."""
    if kind == "sound":
        pr = inputs.wave_1d(n, "sound", amplitude=amplitude, v0=0.0)
        return pr, 1.0 / math.sqrt(pr.gamma * (5.0 / 3.0) / 1.0), 0, False
    pr = inputs.wave_1d(n, kind, amplitude=amplitude)
    return pr, 1.0, (0 if kind == "contact" else 2), kind == "shear"


def measured(U, U0, field, per_rho):
    q, q0 = (U[field] / U[0], U0[field] / U0[0]) if per_rho else (U[field], U0[field])
    return paper_l1(q, q0)


def gpu_error(kind, n, amplitude, prec):
    pr, t_end, field, per_rho = problem(kind, n, amplitude)
    U0 = pr.U.astype(np.float32).astype(np.float64) if prec == binding.PREC_SINGLE else pr.U
    h = binding.KratosHydro(n, 1, 1, pr.gamma, pr.bc, precision=prec)
    h.set_state(U0)
    t, steps = h.run_until(0.4, t_end)
    h.status()
    U, hits = h.get_state(), h.floor_hits()
    h.destroy()
    assert t == t_end and hits == 0
    return measured(U, U0, field, per_rho), steps


def oracle_error(kind, n, amplitude):
    pr, t_end, field, per_rho = problem(kind, n, amplitude)
    U = pr.U.copy()
    t, _, hits = oracle.run(U, pr.gamma, pr.bc, 0.4, 10 ** 7, 0.0, t_end)
    assert t == pytest.approx(t_end, abs=1e-14) and hits == 0
    return measured(U, pr.U, field, per_rho)


def orders(errs):
    return [math.log2(errs[i] / errs[i + 1]) for i in range(len(errs) - 1)]


def record(row):
    out = os.environ.get("KRATOS_PARITY_RECORD_DIR")
    if not out:
        return
    os.makedirs(out, exist_ok=True)
    with open(os.path.join(out, "convergence.jsonl"), "a") as f:
        f.write(json.dumps(row) + "\n")


@pytest.mark.parametrize("kind", ["contact", "shear"])
def test_contact_and_shear_waves_converge_as_n_to_the_minus_two(kind):
    errs = {m: [gpu_error(kind, n, 0.1, p)[0] for n in NS] for m, p in MODES.items()}
    for m in errs:
        record({"wave": kind, "amplitude": 0.1, "mode": m, "n": list(NS), "l1": errs[m], "order": orders(errs[m])})
    # the all-fp64 CUDA path is the oracle's scheme: same error where the oracle is quick
    for i, n in enumerate(NS[:3]):
        assert errs["fp64"][i] == pytest.approx(oracle_error(kind, n, 0.1), rel=1e-7)
    assert all(1.6 < o < 2.2 for o in orders(errs["fp64"])), orders(errs["fp64"])
    # mixed precision "almost identical" to all-fp64 for these waves
    for e_m, e_d in zip(errs["mixed"], errs["fp64"]):
        assert e_m == pytest.approx(e_d, rel=0.05)
    assert all(1.6 < o < 2.2 for o in orders(errs["mixed"])), orders(errs["mixed"])
    # Single: recorded only (the state itself is stored in fp32; where it leaves the line is the measurement)
    assert np.isfinite(errs["single"]).all()


def test_sound_wave_fp64_converges_and_reduced_precision_is_recorded():
    d6 = [gpu_error("sound", n, 1e-6, binding.PREC_FP64)[0] for n in NS]
    record({"wave": "sound", "amplitude": 1e-6, "mode": "fp64", "n": list(NS), "l1": d6, "order": orders(d6)})
    for i, n in enumerate(NS[:3]):   # (the error is 1e-2 ... 1e-3 of an amplitude of 1e-6: rounding differences of 1e-15 show at 1e-6)
        assert d6[i] == pytest.approx(oracle_error("sound", n, 1e-6), rel=1e-4)
    # "achieves convergence up to N > 10^3, following a scaling rule of L1 <~ N^-2"
    assert all(1.6 < o < 2.2 for o in orders(d6)), orders(d6)
    # A = 1e-4, the amplitude the paper uses for its mixed and Single runs: all three modes side by side
    errs = {m: [gpu_error("sound", n, 1e-4, p)[0] for n in NS] for m, p in MODES.items()}
    for m in errs:
        record({"wave": "sound", "amplitude": 1e-4, "mode": m, "n": list(NS), "l1": errs[m], "order": orders(errs[m])})
    # all-fp64 at this amplitude: on the line up to N ~ 256, then the wave's own steepening takes over (not a rounding effect)
    assert errs["fp64"][0] == pytest.approx(d6[0], rel=0.02) and 1.6 < orders(errs["fp64"])[0] < 2.2
    # mixed and Single: recorded, not asserted (see the head of this file)
    assert np.isfinite(errs["mixed"]).all() and np.isfinite(errs["single"]).all()
