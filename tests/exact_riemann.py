"""Exact solution of the 1D special-relativistic Riemann problem for an ideal gas (no tangential
velocity, no magnetic field) — test infrastructure for the Minkowski shock-tube pin (north_star).

Written from the jump conditions and the Riemann invariants themselves (Taub adiabat across a shock;
J+- constant across a simple wave; p and v continuous at the contact), and self-checked against
them in tests/test_oracle_scheme_pins.py.  Units c = 1.  State = (rho, p, v).
"""
import math

import numpy as np
from scipy.optimize import brentq


class Gas:
    def __init__(self, gam):
        self.g = gam

    def h(self, rho, p):          # specific enthalpy
        return 1.0 + self.g / (self.g - 1.0) * p / rho

    def cs(self, rho, p):
        return math.sqrt(self.g * p / (rho * self.h(rho, p)))


def _shock(gas, a, p, sign):
    """State behind a shock running into state a=(rho,p,v) with post-shock pressure p > p_a.
    sign=+1: shock moves to the right relative to a (a is the right state); -1: to the left.
    Returns (rho_b, v_b, V_shock)."""
    g = gas.g
    rho_a, p_a, v_a = a
    h_a = gas.h(rho_a, p_a)
    # Taub adiabat  h_b^2 - h_a^2 = (h_b/rho_b + h_a/rho_a)(p - p_a)  with rho_b = g p / ((g-1)(h_b-1))
    k = (g - 1.0) * (p - p_a) / (g * p)
    A = 1.0 - k
    B = k
    Cc = -h_a * h_a - h_a * (p - p_a) / rho_a
    h_b = (-B + math.sqrt(B * B - 4.0 * A * Cc)) / (2.0 * A)
    rho_b = g * p / ((g - 1.0) * (h_b - 1.0))
    j2 = (p - p_a) / (h_a / rho_a - h_b / rho_b)      # (proper mass flux)^2
    j = math.sqrt(j2)
    ua, ub = j / rho_a, j / rho_b                     # |Gamma v| of a and b in the shock frame
    va_s, vb_s = ua / math.sqrt(1 + ua * ua), ub / math.sqrt(1 + ub * ub)
    vrel = (va_s - vb_s) / (1.0 - va_s * vb_s)        # speed of b relative to a (towards the shock motion)
    v_b = (v_a + sign * vrel) / (1.0 + sign * v_a * vrel)
    Vs = (v_a + sign * va_s) / (1.0 + sign * v_a * va_s)
    return rho_b, v_b, Vs


def _rarefaction(gas, a, p, sign):
    """State reached from a through a simple wave down to pressure p <= p_a.
    sign=-1: wave of the lambda_- family (left state), +1: lambda_+ family (right state)."""
    g = gas.g
    rho_a, p_a, v_a = a
    rho = rho_a * (p / p_a) ** (1.0 / g)
    cs_a, cs = gas.cs(rho_a, p_a), gas.cs(rho, p)
    sq = math.sqrt(g - 1.0)
    # J_-+ = 1/2 ln((1+v)/(1-v)) -+ sign ... : for the left wave J_+ is constant, for the right wave J_-
    fac = (((sq + cs_a) / (sq - cs_a)) * ((sq - cs) / (sq + cs))) ** (2.0 / sq)
    if sign > 0:
        fac = 1.0 / fac
    R = (1.0 + v_a) / (1.0 - v_a) * fac
    v = (R - 1.0) / (R + 1.0)
    return rho, v


def _behind(gas, a, p, sign):
    if p > a[1]:
        rho, v, _ = _shock(gas, a, p, sign)
    else:
        rho, v = _rarefaction(gas, a, p, sign)
    return rho, v


def solve(gam, left, right):
    gas = Gas(gam)
    f = lambda p: _behind(gas, left, p, -1)[1] - _behind(gas, right, p, +1)[1]
    lo, hi = 1e-12 * min(left[1], right[1]), 1e3 * max(left[1], right[1])
    pstar = brentq(f, lo, hi, xtol=1e-15, rtol=1e-14, maxiter=500)
    rhoL, vstar = _behind(gas, left, pstar, -1)
    rhoR, vstar2 = _behind(gas, right, pstar, +1)
    return dict(gas=gas, left=left, right=right, pstar=pstar, vstar=0.5 * (vstar + vstar2), rhoLstar=rhoL,
                rhoRstar=rhoR, dv=vstar - vstar2)


def sample(sol, xi):
    """(rho, p, v) at xi = (x - x0)/t for an array xi."""
    gas = sol["gas"]
    L, R = sol["left"], sol["right"]
    ps, vs = sol["pstar"], sol["vstar"]
    xi = np.atleast_1d(np.asarray(xi, dtype=float))
    out = np.zeros((3, xi.size))

    def wave(a, sign, rho_star):
        """returns (speed_outer, speed_inner, fan) for the wave adjacent to state a"""
        if ps > a[1]:
            _, _, Vs = _shock(gas, a, ps, sign)
            return Vs, Vs, False
        cs_a = gas.cs(a[0], a[1]); cs_s = gas.cs(rho_star, ps)
        head = (a[2] + sign * cs_a) / (1 + sign * a[2] * cs_a)
        tail = (vs + sign * cs_s) / (1 + sign * vs * cs_s)
        return head, tail, True

    lh, lt, lfan = wave(L, -1, sol["rhoLstar"])
    rh, rt, rfan = wave(R, +1, sol["rhoRstar"])

    def in_fan(a, sign, x):
        def g(p):
            rho, v = _rarefaction(gas, a, p, sign)
            cs = gas.cs(rho, p)
            return (v + sign * cs) / (1 + sign * v * cs) - x
        p = brentq(g, ps, a[1], xtol=1e-15, rtol=1e-14)
        rho, v = _rarefaction(gas, a, p, sign)
        return rho, p, v

    for n, x in enumerate(xi):
        if x <= lh:
            out[:, n] = L
        elif x < lt:
            out[:, n] = in_fan(L, -1, x)
        elif x < vs:
            out[:, n] = (sol["rhoLstar"], ps, vs)
        elif x < rt:
            out[:, n] = (sol["rhoRstar"], ps, vs)
        elif x < rh and rfan:
            out[:, n] = in_fan(R, +1, x)
        else:
            out[:, n] = R
    return out
