"""Parameter dictionaries for the library / oracle parameter blocks and the BASELINE.json configs.

Plain data: every key is a field of the `cuharm_params` block declared in include/cuharm.h.
"""
import math

SEED = 220502484  # numpy PCG64 seed of every synthetic workload


def r_horizon(a: float) -> float:
    """Outer horizon r_h = 1 + sqrt(1 - a^2)."""
    return 1.0 + math.sqrt(1.0 - a * a)


def default_params(**kw) -> dict:
    a = kw.get("a", 0.9375)
    d = dict(
        n1=64, n2=64, n3=1, ng=3,
        coords=0,                      # 0 MKS, 1 Minkowski
        a=a, gam=13.0 / 9.0,
        r_in=0.98 * r_horizon(a), r_out=40.0, R0=0.0, hslope=0.3,
        xmin=(0.0, 0.0, 0.0), xmax=(1.0, 1.0, 1.0),
        recon=0, riemann=0,
        bc_x1=0, bc_x2=2, bc_x3=1,     # outflow / polar-reflect / periodic
        rho_fl_coef=1e-5, rho_fl_pow=-1.5, rho_fl_abs=1e-20,           # eq. 35 (A9)
        u_fl_coef=1e-5 / 3.0, u_fl_pow=-2.5, u_fl_abs=1e-20,
        sigma_max=50.0, b2_over_u_max=2.5e3, gamma_max=50.0,           # eqs. 36-37
        newton_tol=1e-10, newton_maxit=30, newton_extra=0,             # P:L233 (A8: the paper's literal stopping rule)
        fixup_max_passes=4,
        n_x=0, r_break=0.0,            # hyper-exponential radial branch of eq. 39: off; the paper: 4, 400
        inv_chain=0, brent_maxit=200,  # inversion fallback chain: off on the hot path (A33)
        beta_min=1e-2, brent_tol=1e-14,   # eq. 33; Brent's relative tolerance (A40)
        n1_global=0, i_offset=0, slab_lo=0, slab_hi=0,   # slab of a larger grid; 0: the whole grid
        polar_damp=0,                  # P:L311 (A16): polar velocity of the two zones nearest each pole -> 0 at the pole; off
    )
    d.update(kw)
    if "a" in kw and "r_in" not in kw:
        d["r_in"] = 0.98 * r_horizon(d["a"])
    return d


def config(name: str, **kw) -> dict:
    """Grid/scheme parameters of BASELINE.json's configs C1..C5; `kw` overrides
    (e.g. a reduced n1,n2,n3 for a parity-sized copy of the same problem)."""
    if name == "C1":
        d = default_params(n1=64, n2=64, n3=1, a=0.9375, gam=13.0 / 9.0, r_out=40.0, recon=0, riemann=0,
                           rho_fl_coef=1e-4, rho_fl_pow=-1.5, u_fl_coef=1e-6, u_fl_pow=-2.5)
    elif name == "C2":
        d = default_params(n1=64, n2=64, n3=1, a=0.5, gam=4.0 / 3.0, r_out=40.0, recon=0, riemann=0, bc_x1=3)
    elif name == "C3":
        d = default_params(n1=128, n2=128, n3=64, a=0.9375, gam=4.0 / 3.0, r_out=40.0, recon=0, riemann=1)
    elif name == "C4":
        d = default_params(n1=256, n2=256, n3=256, a=0.9375, gam=13.0 / 9.0, r_out=40.0, recon=1, riemann=0)
    elif name == "C5":
        d = default_params(n1=384, n2=256, n3=256, a=0.9375, gam=5.0 / 3.0, r_out=1000.0, recon=1, riemann=1)
    else:
        raise KeyError(name)
    d.update(kw)
    return d


# torus set-up that goes with each config (arguments of workloads.torus.fm_torus)
TORUS = {
    "C1": dict(r_in=6.0, r_max=12.0, beta0=100.0, beta_mode="min", perturb=0.04),
    "C3": dict(r_in=6.0, r_max=12.0, beta0=100.0, beta_mode="maxima", perturb=0.04),
    "C4": dict(r_in=6.0, r_max=12.0, beta0=100.0, beta_mode="maxima", perturb=0.04),
    "C5": dict(r_in=20.0, r_max=41.0, beta0=30.0, beta_mode="maxima", perturb=0.04),
}
