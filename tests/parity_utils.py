"""Comparison metrics of the GPU parity tests (CUDA path against the fp64 CPU oracle).

Two bounds per conserved field f (BASELINE.json north_star + DESIGN.md section 7):

* relative L1:  sum |f_gpu - f_orc| / sum |f_orc|  <=  1e-5 (mixed precision), 1e-12 (all-fp64);
* pointwise:    max |f_gpu - f_orc| / scale(f)     <=  1e-4 (mixed),           1e-11 (all-fp64),
  scale(f) = max(max f_orc - min f_orc, 0.1 max |f_orc|): the field's range, or a tenth of its
  magnitude where the field is nearly uniform (fp32 rounding errors scale with the magnitude).
  One wrong cell in a block of 10^4 moves the L1 sum by 10^-4 of its own error and would pass the
  first bound; it cannot pass this one.  Measured on the five BASELINE configs at full size
  (profiles/r3_parity_full_size.md; first measured in round 2): <= 9.2e-6 mixed, <= 8.4e-14 all-fp64.

Fields that are identically zero in the oracle (unused momenta) must be identically zero on the GPU.
"""
import numpy as np

MIXED, FP64, SINGLE = 0, 1, 2
TOL_L1 = {MIXED: 1e-5, FP64: 1e-12}
TOL_MAX = {MIXED: 1e-4, FP64: 1e-11}


def tol_single(nsteps):
    """(rel-L1, pointwise) bounds of the all-fp32 "Single" mode (float2_t = float) against the fp64
    oracle after nsteps Heun steps: the mixed-precision bound for the float_t flux arithmetic
    plus the storage of the state in fp32.  Every stage rounds each conserved value once when it is stored and at
    most once more inside its fp32 update (flux sum, Heun average), relative error <= 2^-24 each: four roundings
    per step, summed without cancellation.  tests/test_oracle_pins.py pins this storage term on the oracle alone."""
    l1 = 1e-5 + 4.0 * nsteps * 2.0 ** -24
    return l1, 10.0 * l1


def single_errors(got, ref, gamma):
    """(rel-L1, pointwise) per field for the Single mode.  As rel_l1_fields / max_norm_fields, except that a momentum
    component is measured against the acoustic momentum rho c, c = sqrt(gamma p / rho), where that is larger than
    the component itself: a rounding of rho, p or E by 2^-24 changes the pressure force on a cell, hence its
    momentum, by ~ dt/dx p 2^-24 ~ rho c 2^-24 per step whether or not the cell moves, so a momentum component that
    is small against rho c (the 1 % seed noise of C3, the transverse components of a 1D tube) has no relative
    accuracy of its own in fp32.  Identically-zero fields must still be identically zero."""
    rho = ref[0]
    v2 = (ref[1] ** 2 + ref[2] ** 2 + ref[3] ** 2) / rho ** 2
    p = (gamma - 1.0) * (ref[4] - 0.5 * rho * v2)
    rc = rho * np.sqrt(gamma * np.maximum(p, 0.0) / rho)
    l1, mx = [], []
    for m in range(5):
        d = np.abs(got[m] - ref[m])
        den = np.abs(ref[m]).sum()
        if den == 0.0:
            assert np.all(got[m] == 0.0), f"field {m} must stay exactly zero"
            l1.append(0.0); mx.append(0.0)
            continue
        scale = field_scale(ref[m])
        if 1 <= m <= 3:
            den = max(den, float(rc.sum()))
            scale = max(scale, 0.1 * float(rc.max()))
        l1.append(float(d.sum() / den))
        mx.append(float(d.max() / scale))
    return l1, mx


def assert_parity_single(got, ref, gamma, nsteps, what=""):
    assert np.isfinite(got).all(), f"{what}: non-finite values in the GPU state"
    l1, mx = single_errors(got, ref, gamma)
    t1, tm = tol_single(nsteps)
    assert max(l1) <= t1, (what, "rel-L1", l1, t1)
    assert max(mx) <= tm, (what, "max-norm", mx, tm)
    return l1, mx


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


def field_scale(ref_m):
    return max(float(ref_m.max() - ref_m.min()), 0.1 * float(np.abs(ref_m).max()))


def max_norm_fields(got, ref):
    """Per-field max |got - ref| / scale(ref); 0 for fields that are identically zero in the oracle."""
    out = []
    for m in range(5):
        s = field_scale(ref[m])
        out.append(0.0 if s == 0.0 else float(np.abs(got[m] - ref[m]).max() / s))
    return out


def assert_parity(got, ref, prec, what="", tol_l1=None, tol_max=None):
    """Both bounds, every field; NaN anywhere fails.  Returns (l1, maxnorm) per field for reporting."""
    assert np.isfinite(got).all(), f"{what}: non-finite values in the GPU state"
    l1 = rel_l1_fields(got, ref)
    mx = max_norm_fields(got, ref)
    assert max(l1) <= (TOL_L1[prec] if tol_l1 is None else tol_l1), (what, "rel-L1", l1)
    assert max(mx) <= (TOL_MAX[prec] if tol_max is None else tol_max), (what, "max-norm", mx)
    return l1, mx
