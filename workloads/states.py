"""Small synthetic states: Minkowski boxes (waves, shock tubes, uniform), random smooth fields.

Inputs only — no method arithmetic beyond evaluating the initial profile.
"""
import numpy as np

from .params import default_params, SEED


def minkowski_params(n1, n2, n3, xmax=(1.0, 1.0, 1.0), bc=(1, 1, 1), **kw):
    d = default_params(n1=n1, n2=n2, n3=n3, coords=1, xmin=(0.0, 0.0, 0.0), xmax=tuple(xmax),
                       bc_x1=bc[0], bc_x2=bc[1], bc_x3=bc[2],
                       rho_fl_coef=1e-12, rho_fl_pow=0.0, u_fl_coef=1e-14, u_fl_pow=0.0,
                       sigma_max=0.0, b2_over_u_max=0.0)
    d.update(kw)
    return d


def empty_prim(p):
    ng = p["ng"]
    return np.zeros((8, p["n1"] + 2 * ng, p["n2"] + 2 * ng, p["n3"] + 2 * ng))


def centres(p, d):
    ng = p["ng"]
    n = (p["n1"], p["n2"], p["n3"])[d]
    h = (p["xmax"][d] - p["xmin"][d]) / n
    return p["xmin"][d] + (np.arange(-ng, n + ng) + 0.5) * h


def uniform_state(p, q8):
    prim = empty_prim(p)
    for v in range(8):
        prim[v] = q8[v]
    return prim


def sound_wave(p, direction=0, amp=1e-6, rho0=1.0, u0=0.3, B0=(0.0, 0.0, 0.0), t=0.0):
    """Right-going linear sound wave (B along the wave vector allowed) of wavelength = box length.
    Returns prim and the phase speed c_s used for the analytic solution at time t."""
    gam = p["gam"]
    pg = (gam - 1.0) * u0
    w = rho0 + u0 + pg
    cs = np.sqrt(gam * pg / w)
    x = centres(p, direction)
    L = p["xmax"][direction] - p["xmin"][direction]
    shape = [1, 1, 1]
    shape[direction] = -1
    ph = np.sin(2.0 * np.pi * (x - cs * t) / L).reshape(shape)
    prim = empty_prim(p)
    prim[0] = rho0 * (1.0 + amp * ph)
    prim[1] = u0 * (1.0 + gam * amp * ph)           # adiabatic: dp/p = gam drho/rho
    prim[2 + direction] = cs * amp * ph             # dv = cs drho / rho * (rho/w)*(w/rho) -> cs * drho/rho * rho/w * ... see test
    for i in range(3):
        prim[5 + i] = B0[i]
    return prim, cs


def shock_tube(p, left, right, direction=0, x0=0.5):
    """left/right = (rho, p_gas, v) hydrodynamic states; B = 0; discontinuity at x0 along `direction`."""
    gam = p["gam"]
    x = centres(p, direction)
    shape = [1, 1, 1]
    shape[direction] = -1
    L = (x < x0).reshape(shape)
    prim = empty_prim(p)

    def prim_of(s):
        rho, pg, v = s
        lor = 1.0 / np.sqrt(1.0 - v * v)
        return rho, pg / (gam - 1.0), lor * v

    ql, qr = prim_of(left), prim_of(right)
    prim[0] = np.where(L, ql[0], qr[0])
    prim[1] = np.where(L, ql[1], qr[1])
    prim[2 + direction] = np.where(L, ql[2], qr[2])
    return prim


def random_smooth(shape, rng, nmodes=3):
    """A smooth random scalar field on `shape` (sum of a few low Fourier modes), O(1)."""
    out = np.zeros(shape)
    grids = np.meshgrid(*[np.arange(n) / n for n in shape], indexing="ij")
    for _ in range(nmodes):
        k = rng.integers(0, 3, size=len(shape))
        ph = rng.uniform(0, 2 * np.pi)
        out += rng.normal() * np.sin(2 * np.pi * sum(ki * g for ki, g in zip(k, grids)) + ph)
    return out


def rng(seed=SEED):
    return np.random.Generator(np.random.PCG64(seed))


def fast_wave(p, direction=0, bdir=1, amp=1e-6, rho0=1.0, u0=0.3, B0=0.5, t=0.0):
    """Right-going linear fast magnetosonic wave, wave vector along `direction`, uniform field B0 along
    `bdir` (perpendicular), fluid at rest.  Returns prim and the phase speed
    c_f = sqrt((gam p + b^2)/(w + b^2)) (eq. 18 of the paper for k perpendicular to B)."""
    assert bdir != direction
    gam = p["gam"]
    pg = (gam - 1.0) * u0
    w = rho0 + u0 + pg
    bsq = B0 * B0
    cf = np.sqrt((gam * pg + bsq) / (w + bsq))
    x = centres(p, direction)
    L = p["xmax"][direction] - p["xmin"][direction]
    shape = [1, 1, 1]
    shape[direction] = -1
    ph = np.sin(2.0 * np.pi * (x - cf * t) / L).reshape(shape)
    prim = empty_prim(p)
    prim[0] = rho0 * (1.0 + amp * ph)
    prim[1] = u0 * (1.0 + gam * amp * ph)
    prim[2 + direction] = cf * amp * ph
    prim[5 + bdir] = B0 * (1.0 + amp * ph)
    return prim, cf
