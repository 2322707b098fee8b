"""Exact solution of the 1D Riemann problem for the ideal-gas Euler equations.

TEST INFRASTRUCTURE (a pin for the oracle) -- not product.

This is the textbook closed-form construction the paper points to for its shock-tube
checks ("semi-analytic solutions", after Toro 2009): find the star
pressure p* as the root of

    f_L(p) + f_R(p) + (u_R - u_L) = 0,
    f_K(p) = (p - p_K) sqrt(A_K / (p + B_K))                      p >  p_K  (shock)
           = 2 c_K / (gamma-1) [ (p/p_K)^((gamma-1)/(2 gamma)) - 1 ]  p <= p_K  (rarefaction)
    A_K = 2 / ((gamma+1) rho_K),  B_K = (gamma-1)/(gamma+1) p_K,

then u* = (u_L + u_R)/2 + (f_R - f_L)/2 and sample the self-similar wave fan at
xi = (x - x0)/t.  It shares nothing with the numerical scheme (no HLLC, no PLM).
"""
from __future__ import annotations

import numpy as np


def _f_and_df(p, rho_k, p_k, c_k, gamma):
    if p > p_k:
        A = 2.0 / ((gamma + 1.0) * rho_k)
        B = (gamma - 1.0) / (gamma + 1.0) * p_k
        s = np.sqrt(A / (p + B))
        return (p - p_k) * s, s * (1.0 - 0.5 * (p - p_k) / (p + B))
    pr = p / p_k
    return (2.0 * c_k / (gamma - 1.0) * (pr ** ((gamma - 1.0) / (2.0 * gamma)) - 1.0),
            pr ** (-(gamma + 1.0) / (2.0 * gamma)) / (rho_k * c_k))


def star_state(rho_l, u_l, p_l, rho_r, u_r, p_r, gamma):
    """Return (p*, u*).  Raises if the data generate vacuum."""
    c_l = np.sqrt(gamma * p_l / rho_l)
    c_r = np.sqrt(gamma * p_r / rho_r)
    if 2.0 * (c_l + c_r) / (gamma - 1.0) <= u_r - u_l:
        raise ValueError("vacuum is generated")

    def g(p):
        fl, dfl = _f_and_df(p, rho_l, p_l, c_l, gamma)
        fr, dfr = _f_and_df(p, rho_r, p_r, c_r, gamma)
        return fl + fr + (u_r - u_l), dfl + dfr

    # g is monotone increasing and concave: bracket, then safeguarded Newton
    lo, hi = 1e-300, max(p_l, p_r)
    while g(hi)[0] < 0.0:
        hi *= 2.0
    p = 0.5 * (p_l + p_r)
    for _ in range(200):
        val, der = g(p)
        if val > 0.0:
            hi = min(hi, p)
        else:
            lo = max(lo, p)
        pn = p - val / der
        if not (lo < pn < hi):
            pn = 0.5 * (lo + hi)
        if abs(pn - p) <= 1e-15 * max(abs(pn), abs(p)):
            p = pn
            break
        p = pn
    fl, _ = _f_and_df(p, rho_l, p_l, c_l, gamma)
    fr, _ = _f_and_df(p, rho_r, p_r, c_r, gamma)
    return p, 0.5 * (u_l + u_r) + 0.5 * (fr - fl)


def sample(xi, rho_l, u_l, p_l, rho_r, u_r, p_r, gamma):
    """Exact (rho, u, p) at similarity coordinates xi = (x - x0)/t (array)."""
    xi = np.asarray(xi, dtype=np.float64)
    ps, us = star_state(rho_l, u_l, p_l, rho_r, u_r, p_r, gamma)
    c_l = np.sqrt(gamma * p_l / rho_l)
    c_r = np.sqrt(gamma * p_r / rho_r)
    gm1, gp1 = gamma - 1.0, gamma + 1.0
    rho = np.empty_like(xi)
    u = np.empty_like(xi)
    p = np.empty_like(xi)

    left = xi <= us
    # ---- left of the contact
    if ps > p_l:  # left shock
        s_l = u_l - c_l * np.sqrt(gp1 / (2 * gamma) * ps / p_l + gm1 / (2 * gamma))
        rho_sl = rho_l * ((ps / p_l + gm1 / gp1) / (gm1 / gp1 * ps / p_l + 1.0))
        pre = left & (xi <= s_l)
        post = left & (xi > s_l)
        rho[pre], u[pre], p[pre] = rho_l, u_l, p_l
        rho[post], u[post], p[post] = rho_sl, us, ps
    else:  # left rarefaction
        c_sl = c_l * (ps / p_l) ** (gm1 / (2 * gamma))
        head, tail = u_l - c_l, us - c_sl
        pre = left & (xi <= head)
        fan = left & (xi > head) & (xi < tail)
        post = left & (xi >= tail)
        rho[pre], u[pre], p[pre] = rho_l, u_l, p_l
        fac = 2.0 / gp1 + gm1 / (gp1 * c_l) * (u_l - xi[fan])
        rho[fan] = rho_l * fac ** (2.0 / gm1)
        u[fan] = 2.0 / gp1 * (c_l + gm1 / 2.0 * u_l + xi[fan])
        p[fan] = p_l * fac ** (2.0 * gamma / gm1)
        rho[post], u[post], p[post] = rho_l * (ps / p_l) ** (1.0 / gamma), us, ps
    # ---- right of the contact
    right = ~left
    if ps > p_r:  # right shock
        s_r = u_r + c_r * np.sqrt(gp1 / (2 * gamma) * ps / p_r + gm1 / (2 * gamma))
        rho_sr = rho_r * ((ps / p_r + gm1 / gp1) / (gm1 / gp1 * ps / p_r + 1.0))
        pre = right & (xi >= s_r)
        post = right & (xi < s_r)
        rho[pre], u[pre], p[pre] = rho_r, u_r, p_r
        rho[post], u[post], p[post] = rho_sr, us, ps
    else:  # right rarefaction
        c_sr = c_r * (ps / p_r) ** (gm1 / (2 * gamma))
        head, tail = u_r + c_r, us + c_sr
        pre = right & (xi >= head)
        fan = right & (xi < head) & (xi > tail)
        post = right & (xi <= tail)
        rho[pre], u[pre], p[pre] = rho_r, u_r, p_r
        fac = 2.0 / gp1 - gm1 / (gp1 * c_r) * (u_r - xi[fan])
        rho[fan] = rho_r * fac ** (2.0 / gm1)
        u[fan] = 2.0 / gp1 * (-c_r + gm1 / 2.0 * u_r + xi[fan])
        p[fan] = p_r * fac ** (2.0 * gamma / gm1)
        rho[post], u[post], p[post] = rho_r * (ps / p_r) ** (1.0 / gamma), us, ps
    return rho, u, p


def wave_speeds(rho_l, u_l, p_l, rho_r, u_r, p_r, gamma):
    """(leftmost, rightmost) speed of the exact wave fan -- used to find plateau cells."""
    ps, us = star_state(rho_l, u_l, p_l, rho_r, u_r, p_r, gamma)
    c_l = np.sqrt(gamma * p_l / rho_l)
    c_r = np.sqrt(gamma * p_r / rho_r)
    gm1, gp1 = gamma - 1.0, gamma + 1.0
    if ps > p_l:
        a = u_l - c_l * np.sqrt(gp1 / (2 * gamma) * ps / p_l + gm1 / (2 * gamma))
        a_in = a
    else:
        a = u_l - c_l
        a_in = us - c_l * (ps / p_l) ** (gm1 / (2 * gamma))
    if ps > p_r:
        b = u_r + c_r * np.sqrt(gp1 / (2 * gamma) * ps / p_r + gm1 / (2 * gamma))
        b_in = b
    else:
        b = u_r + c_r
        b_in = us + c_r * (ps / p_r) ** (gm1 / (2 * gamma))
    return dict(p_star=ps, u_star=us, left_outer=a, left_inner=a_in, right_inner=b_in, right_outer=b)
