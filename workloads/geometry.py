"""numpy Kerr-Schild / MKS geometry used ONLY to build initial data (eq. 38-39).

Independent of both the oracle and the CUDA path: the generators need u^mu -> modified velocity and
sqrt(-g) to turn a physical set-up into the primitive array both implementations are fed with.
"""
import numpy as np


def _hyper(p: dict):
    return p["coords"] == 0 and p.get("n_x", 0) >= 2 and p.get("r_break", 0.0) > p["R0"]


def radial_x_of_r(p: dict, r):
    """X1 at which eq. 39's radial map (with its hyper-exponential branch, if switched on) reaches the radius r."""
    target = np.log(r - p["R0"])
    if not _hyper(p):
        return target
    xb = np.log(p["r_break"] - p["R0"])
    if target <= xb:
        return target
    from scipy.optimize import brentq
    return brentq(lambda x: x + (x - xb) ** p["n_x"] - target, xb, target, xtol=1e-15, rtol=1e-15)


def grid_coords(p: dict, centred=True):
    """X1, X2, X3 of zone centres over the extended grid (ghosts included)."""
    ng = p["ng"]
    n = (p["n1"], p["n2"], p["n3"])
    if p["coords"] == 0:
        x0 = (np.log(p["r_in"] - p["R0"]), -1.0, 0.0)
        x1 = (radial_x_of_r(p, p["r_out"]), 1.0, 2.0 * np.pi)
    else:
        x0, x1 = p["xmin"], p["xmax"]
    out = []
    dx = []
    for d in range(3):
        h = (x1[d] - x0[d]) / n[d]
        idx = np.arange(-ng, n[d] + ng)
        out.append(x0[d] + (idx + (0.5 if centred else 0.0)) * h)
        dx.append(h)
    return out, dx


def mks_to_ks(p: dict, X1, X2):
    X1 = np.asarray(X1, dtype=float)
    E, E1 = X1, np.ones_like(X1)
    if _hyper(p):                                   # eq. 39, X >= x_b: r = R0 + exp(X + (X - x_b)^n_X)
        xb = np.log(p["r_break"] - p["R0"])
        y = np.maximum(X1 - xb, 0.0)
        E = X1 + y ** p["n_x"]
        E1 = 1.0 + p["n_x"] * y ** (p["n_x"] - 1)
    r = p["R0"] + np.exp(E)
    arg = np.pi * (1.0 + X2)
    th = 0.5 * np.pi * (1.0 + X2) + 0.5 * (1.0 - p["hslope"]) * np.sin(arg)
    drdX = (r - p["R0"]) * E1
    dthdY = 0.5 * np.pi * (1.0 + (1.0 - p["hslope"]) * np.cos(arg))
    return r, th, drdX, dthdY


def ks_metric(a, r, th):
    """g_{mu nu} (KS, eq. 38) with shape r.shape + (4,4)."""
    s2 = np.sin(th) ** 2
    Sig = r * r + a * a * np.cos(th) ** 2
    f = 2.0 * r / Sig
    g = np.zeros(np.shape(r) + (4, 4))
    g[..., 0, 0] = -1.0 + f
    g[..., 0, 1] = g[..., 1, 0] = f
    g[..., 0, 3] = g[..., 3, 0] = -a * s2 * f
    g[..., 1, 1] = 1.0 + f
    g[..., 1, 3] = g[..., 3, 1] = -a * s2 * (1.0 + f)
    g[..., 2, 2] = Sig
    g[..., 3, 3] = s2 * (Sig + a * a * s2 * (1.0 + f))
    return g


def mks_metric(p: dict, X1, X2):
    """gcov, gcon, sqrt(-g), alpha in MKS coordinates at (X1, X2) (arrays broadcast)."""
    if p["coords"] == 1:
        shp = np.broadcast(X1, X2).shape
        g = np.zeros(shp + (4, 4))
        g[..., 0, 0] = -1.0
        for i in (1, 2, 3):
            g[..., i, i] = 1.0
        return g, g.copy(), np.ones(shp), np.ones(shp)
    r, th, drdX, dthdY = mks_to_ks(p, X1, X2)
    g = ks_metric(p["a"], r, th)
    J = np.stack([np.ones_like(r), drdX, dthdY, np.ones_like(r)], axis=-1)
    gcov = g * J[..., :, None] * J[..., None, :]
    gcon = np.linalg.inv(gcov)
    Sig = r * r + p["a"] ** 2 * np.cos(th) ** 2
    sqrtg = Sig * np.abs(np.sin(th)) * np.abs(drdX) * np.abs(dthdY)
    alpha = 1.0 / np.sqrt(-gcon[..., 0, 0])
    return gcov, gcon, sqrtg, alpha


def ucon_to_utilde(ucon, gcon, alpha):
    """Modified velocity of eq. 10: utilde^i = u^i + Gamma beta^i / alpha, Gamma = alpha u^t."""
    lor = alpha * ucon[..., 0]
    beta = gcon[..., 0, 1:] * (alpha ** 2)[..., None]
    return ucon[..., 1:] + (lor / alpha)[..., None] * beta


def bsq_of(prim, gcov, gcon, alpha):
    """b^2 of a primitive array prim[8,...] given the metric at the same points."""
    ut = np.moveaxis(prim[2:5], 0, -1)
    B = np.moveaxis(prim[5:8], 0, -1)
    gij = gcov[..., 1:, 1:]
    qsq = np.einsum("...i,...ij,...j->...", ut, gij, ut)
    lor = np.sqrt(1.0 + qsq)
    ucon = np.zeros(ut.shape[:-1] + (4,))
    ucon[..., 0] = lor / alpha
    beta = gcon[..., 0, 1:] * (alpha ** 2)[..., None]
    ucon[..., 1:] = ut - (lor / alpha)[..., None] * beta
    ucov = np.einsum("...mn,...n->...m", gcov, ucon)
    bt = np.einsum("...i,...i->...", B, ucov[..., 1:])
    bcon = np.zeros_like(ucon)
    bcon[..., 0] = bt
    bcon[..., 1:] = (B + bt[..., None] * ucon[..., 1:]) / ucon[..., :1]
    bcov = np.einsum("...mn,...n->...m", gcov, bcon)
    return np.einsum("...m,...m->...", bcon, bcov)
