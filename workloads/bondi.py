"""Magnetised Bondi (Michel) flow with a split-monopole-free radial field in Kerr-Schild coordinates:
the steady-state / convergence workload of BASELINE.json config C2 (not in the paper; A38).

Exact for a = 0: the radial field is parallel to the flow and exerts no force, so the hydrodynamic
Michel solution stays an exact steady solution of ideal GR-MHD.  For a != 0 the same initial data are
used (C2 asks for a = 0.5) and only self-convergence is measured.

Inputs only: evaluates the analytic profile; no part of the numerical method lives here.
"""
import numpy as np
from scipy.optimize import brentq, minimize_scalar

from .geometry import grid_coords, mks_to_ks, mks_metric, ucon_to_utilde, bsq_of
from .params import r_horizon


def michel_profile(gam, r_c, r):
    """T = p/rho, rho, u (internal energy), u^r (KS == BL radial component) at the radii r (1D array)."""
    n = 1.0 / (gam - 1.0)
    uc2 = 1.0 / (2.0 * r_c)
    Vc2 = uc2 / (1.0 - 3.0 * uc2)
    Tc = n * Vc2 / ((1.0 + n) * (1.0 - n * Vc2))
    C1 = np.sqrt(uc2) * r_c ** 2 * Tc ** n
    C2 = (1.0 + (1.0 + n) * Tc) ** 2 * (1.0 - 2.0 / r_c + uc2)

    def f(lnT, rr):
        T = np.exp(lnT)
        return (1.0 + (1.0 + n) * T) ** 2 * (1.0 - 2.0 / rr + C1 ** 2 / (rr ** 4 * T ** (2.0 * n))) - C2

    T = np.zeros_like(r)
    for m, rr in enumerate(r):
        res = minimize_scalar(lambda x: f(x, rr), bounds=(np.log(Tc) - 12.0, np.log(Tc) + 12.0), method="bounded",
                              options=dict(xatol=1e-13))
        xm = res.x
        if f(xm, rr) >= 0.0:          # at (or within round-off of) the sonic point
            T[m] = np.exp(xm)
            continue
        if rr >= r_c:                  # subsonic branch: larger T
            T[m] = np.exp(brentq(f, xm, np.log(Tc) + 30.0, args=(rr,), xtol=1e-15, rtol=1e-15))
        else:                          # supersonic branch: smaller T
            T[m] = np.exp(brentq(f, np.log(Tc) - 60.0, xm, args=(rr,), xtol=1e-15, rtol=1e-15))
    rho = T ** n
    u = n * rho * T
    ur = -C1 / (r ** 2 * T ** n)
    return T, rho, u, ur


def bondi(p: dict, r_c=8.0, sigma_h=1.0):
    """Primitive array prim[8, n1g, n2g, n3g], valid in EVERY zone including ghosts (use bc_x1 = 3).

    sigma_h = b^2/rho at the horizon radius fixes the monopole strength (0 -> unmagnetised)."""
    assert p["coords"] == 0
    ng = p["ng"]
    a, gam = p["a"], p["gam"]
    (X1, X2, X3), dx = grid_coords(p)
    r1 = p["R0"] + np.exp(X1)
    T, rho1, u1, ur1 = michel_profile(gam, r_c, r1)
    X1g, X2g = np.meshgrid(X1, X2, indexing="ij")
    r, th, drdX, dthdY = mks_to_ks(p, X1g, X2g)
    gcov, gcon, sqrtg, alpha = mks_metric(p, X1g, X2g)
    n1g, n2g, n3g = r.shape[0], r.shape[1], p["n3"] + 2 * ng
    rho = np.broadcast_to(rho1[:, None], r.shape)
    u = np.broadcast_to(u1[:, None], r.shape)
    uX = np.broadcast_to(ur1[:, None], r.shape) / drdX        # u^{X1} = u^r / r'
    # u^t from u.u = -1 in the MKS metric (only u^t, u^X1 non-zero); root continuous through the horizon
    A = gcov[..., 0, 0]
    B = 2.0 * gcov[..., 0, 1] * uX
    C = gcov[..., 1, 1] * uX ** 2 + 1.0
    disc = np.maximum(B * B - 4.0 * A * C, 0.0)
    with np.errstate(divide="ignore", invalid="ignore"):
        ut = np.where(np.abs(A) > 1e-9, (-B - np.sqrt(disc)) / (2.0 * A), -C / B)
    ucon = np.zeros(r.shape + (4,))
    ucon[..., 0] = ut
    ucon[..., 1] = uX
    util = ucon_to_utilde(ucon, gcon, alpha)
    prim2 = np.zeros((8, n1g, n2g))
    prim2[0], prim2[1] = rho, u
    for i in range(3):
        prim2[2 + i] = util[..., i]
    if sigma_h > 0.0:
        Sig = r * r + a * a * np.cos(th) ** 2
        prim2[5] = 1.0 / (Sig * drdX)                           # B^r = C / Sigma: sqrt(-g) B^1 independent of X1
        # normalise b^2/rho = sigma_h at r = r_h on the equator (interpolate in radius)
        bsq = bsq_of(prim2, gcov, gcon, alpha)
        jeq = np.argmin(np.abs(th[0] - 0.5 * np.pi))
        ratio = np.interp(r_horizon(a), r1, (bsq / rho)[:, jeq])
        prim2[5] *= np.sqrt(sigma_h / ratio)
    prim = np.ascontiguousarray(np.broadcast_to(prim2[:, :, :, None], (8, n1g, n2g, n3g))).copy()
    return prim
