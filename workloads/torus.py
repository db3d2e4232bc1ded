"""Fishbone-Moncrief torus with a single poloidal field loop (eq. 54), the synthetic
stand-in for the paper's initial data (which are not in the container).

Pinned by the paper's Table 1: initial mass M (eq. 55) and magnetic energy E_B (eq. 56).
"""
import numpy as np

from .geometry import grid_coords, mks_to_ks, mks_metric, ucon_to_utilde, bsq_of
from .params import SEED


def _l_circular(a, r):
    """l = u^t u_phi of the prograde circular equatorial geodesic at radius r (Boyer-Lindquist)."""
    Om = 1.0 / (r ** 1.5 + a)
    gtt = -(1.0 - 2.0 / r)
    gtp = -2.0 * a / r
    gpp = r * r + a * a + 2.0 * a * a / r
    ut = 1.0 / np.sqrt(-(gtt + 2.0 * Om * gtp + Om * Om * gpp))
    up = (gtp + Om * gpp) * ut
    return ut * up


def _lnh(a, l, r, th):
    s = np.sin(th)
    Sig = r * r + a * a * np.cos(th) ** 2
    Del = r * r - 2.0 * r + a * a
    A = (r * r + a * a) ** 2 - Del * a * a * s * s
    psi = np.sqrt(1.0 + 4.0 * l * l * Sig * Sig * Del / (A * s) ** 2)
    return 0.5 * np.log((1.0 + psi) / (Sig * Del / A)) - 0.5 * psi - 2.0 * a * r * l / A, psi, Sig, Del, A


def fm_torus(p: dict, r_in=6.0, r_max=12.0, beta0=100.0, beta_mode="maxima", perturb=0.04, seed=SEED,
             field=True):
    """Primitive array prim[8, n1g, n2g, n3g] (ghosts NOT valid: the library's bind applies the BCs).

    Returns (prim, info) with info = dict(M=..., E_B=..., rho_max_raw=..., inside=mask, beta_min=...).
    """
    assert p["coords"] == 0
    ng = p["ng"]
    a, gam = p["a"], p["gam"]
    (X1, X2, X3), dx = grid_coords(p)
    X1g, X2g = np.meshgrid(X1, X2, indexing="ij")
    r, th, drdX, dthdY = mks_to_ks(p, X1g, X2g)
    gcov, gcon, sqrtg, alpha = mks_metric(p, X1g, X2g)

    l = _l_circular(a, r_max)
    lnh_in = _lnh(a, l, np.array(r_in), np.array(0.5 * np.pi))[0]
    with np.errstate(invalid="ignore", divide="ignore", over="ignore"):
        lnh, psi, Sig, Del, A = _lnh(a, l, r, th)
        lnh = lnh - lnh_in
    inside = np.isfinite(lnh) & (lnh > 0.0) & (r >= r_in)
    h = np.where(inside, np.exp(np.where(inside, lnh, 0.0)), 1.0)
    # normalise on the interior zones of THIS grid (rho_max = 1)
    interior = np.zeros_like(inside)
    interior[ng:-ng, ng:-ng] = True
    inside &= interior
    hm1_max = (h - 1.0)[inside].max()
    rho = np.where(inside, ((h - 1.0) / hm1_max) ** (1.0 / (gam - 1.0)), 0.0)
    pg = hm1_max * (gam - 1.0) / gam * rho ** gam
    u = pg / (gam - 1.0)
    # azimuthal velocity (BL = KS components because u^r = u^theta = 0)
    with np.errstate(invalid="ignore", divide="ignore"):
        chi2 = 0.5 * (psi - 1.0)
        uphi = 2.0 * a * r * np.sqrt(1.0 + chi2) / np.sqrt(A * Sig * Del) + np.sqrt(Sig / A) * np.sqrt(chi2) / np.sin(th)
    uphi = np.where(inside, uphi, 0.0)
    # u^t from u.u = -1 with the MKS metric (u^X = u^Y = 0, u^Z = u^phi)
    gtt, gtp, gpp = gcov[..., 0, 0], gcov[..., 0, 3], gcov[..., 3, 3]
    AA, BB, CC = gtt, 2.0 * gtp * uphi, gpp * uphi ** 2 + 1.0
    disc = np.maximum(BB * BB - 4.0 * AA * CC, 0.0)
    utime_torus = (-BB - np.sqrt(disc)) / (2.0 * AA)
    # atmosphere: normal observer (utilde = 0): u^mu = n^mu
    ucon = np.zeros(r.shape + (4,))
    ucon[..., 0] = np.where(inside, utime_torus, 1.0 / alpha)
    ucon[..., 3] = uphi
    beta = gcon[..., 0, 1:] * (alpha ** 2)[..., None]
    for i in range(3):
        ucon[..., 1 + i] = np.where(inside, ucon[..., 1 + i], -beta[..., i] / alpha)
    ut = ucon_to_utilde(ucon, gcon, alpha)
    ut[~inside] = 0.0

    rho_fl = np.maximum(p["rho_fl_abs"], p["rho_fl_coef"] * r ** p["rho_fl_pow"])
    u_fl = np.maximum(p["u_fl_abs"], p["u_fl_coef"] * r ** p["u_fl_pow"])

    n1g, n2g, n3g = r.shape[0], r.shape[1], p["n3"] + 2 * ng
    prim2 = np.zeros((8, n1g, n2g))
    prim2[0] = np.where(inside, np.maximum(rho, rho_fl), rho_fl)
    prim2[1] = np.where(inside, np.maximum(u, u_fl), u_fl)
    for i in range(3):
        prim2[2 + i] = ut[..., i]

    info = dict(rho_max_raw=float(hm1_max), inside=inside[ng:-ng, ng:-ng].copy())
    if field:
        # A_phi at the lower-left corner (I-1/2, J-1/2) of every zone from the 4-cell average (eq. 54)
        rbar = np.zeros_like(rho)
        rbar[1:, 1:] = 0.25 * (rho[1:, 1:] + rho[:-1, 1:] + rho[1:, :-1] + rho[:-1, :-1])
        Aphi = np.maximum(rbar / 1.0 - 0.2, 0.0)
        B1 = np.zeros_like(rho); B2 = np.zeros_like(rho)
        B1[:-1, :-1] = ((Aphi[:-1, 1:] + Aphi[1:, 1:]) - (Aphi[:-1, :-1] + Aphi[1:, :-1])) / (2.0 * dx[1] * sqrtg[:-1, :-1])
        B2[:-1, :-1] = -((Aphi[1:, :-1] + Aphi[1:, 1:]) - (Aphi[:-1, :-1] + Aphi[:-1, 1:])) / (2.0 * dx[0] * sqrtg[:-1, :-1])
        prim2[5], prim2[6] = B1, B2
        bsq = bsq_of(prim2, gcov, gcon, alpha)
        bsq_i = bsq[ng:-ng, ng:-ng]
        pg_i = ((gam - 1.0) * prim2[1])[ng:-ng, ng:-ng]
        if beta_mode == "maxima":      # beta0 = p_g,max / p_B,max
            fac = np.sqrt(pg_i.max() / (0.5 * bsq_i.max() * beta0))
        elif beta_mode == "min":       # C1: pointwise minimum of beta (A23)
            m = bsq_i > 0.0
            fac = np.sqrt((pg_i[m] / (0.5 * bsq_i[m])).min() / beta0)
        else:
            raise ValueError(beta_mode)
        prim2[5] *= fac
        prim2[6] *= fac
        bsq = bsq * fac * fac
        m = bsq[ng:-ng, ng:-ng] > 0.0
        info["beta_min"] = float((pg_i[m] / (0.5 * bsq[ng:-ng, ng:-ng][m])).min()) if m.any() else np.inf
        info["E_B"] = float((sqrtg * bsq * inside).sum() * dx[0] * dx[1] * 2.0 * np.pi)
    info["M"] = float((sqrtg * rho * inside).sum() * dx[0] * dx[1] * 2.0 * np.pi)

    prim = np.ascontiguousarray(np.broadcast_to(prim2[:, :, :, None], (8, n1g, n2g, n3g))).copy()
    if perturb:
        rng = np.random.Generator(np.random.PCG64(seed))
        xi = rng.random((p["n1"], p["n2"], p["n3"]))
        fac = 1.0 + perturb * (xi - 0.5)
        ins = inside[ng:-ng, ng:-ng][:, :, None]
        core = prim[1, ng:-ng, ng:-ng, ng:n3g - ng]
        prim[1, ng:-ng, ng:-ng, ng:n3g - ng] = np.where(ins, core * fac, core)
    return prim, info
