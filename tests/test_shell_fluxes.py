"""Shell (horizon) fluxes, eqs. 43-46: pins of the oracle against closed forms of
the Michel / monopole flow, and GPU-vs-oracle parity of the device reduction."""
import math

import numpy as np
import pytest

import oracle
from workloads import default_params, config
from workloads.bondi import bondi, michel_profile
from workloads.torus import fm_torus


def _michel_constants(gam, r_c):
    n = 1.0 / (gam - 1.0)
    uc2 = 1.0 / (2.0 * r_c)
    Vc2 = uc2 / (1.0 - 3.0 * uc2)
    Tc = n * Vc2 / ((1.0 + n) * (1.0 - n * Vc2))
    C1 = math.sqrt(uc2) * r_c ** 2 * Tc ** n                       # -rho u^r r^2
    C2 = (1.0 + (1.0 + n) * Tc) ** 2 * (1.0 - 2.0 / r_c + uc2)     # (h u_t)^2
    return C1, C2


def _bondi_grid(N, sigma_h):
    p = default_params(n1=N, n2=N, n3=1, a=0.0, gam=4.0 / 3.0, bc_x1=3, hslope=1.0, r_out=20.0)
    prim = bondi(p, sigma_h=sigma_h)
    g = oracle.Grid(p)
    g.bind(prim)
    return p, prim, g


def test_mdot_of_the_michel_flow_is_minus_4_pi_c1_on_every_shell_at_second_order():
    C1, C2 = _michel_constants(4.0 / 3.0, 8.0)
    errs = []
    for N in (16, 32, 64):
        p, prim, g = _bondi_grid(N, 0.0)
        f = np.array([g.shell_fluxes(i) for i in (0, N // 3, N - 1)])
        # a = 0: the quadrature in theta has the same relative error on every shell -> Mdot identical across shells
        assert np.allclose(f[:, 0], f[0, 0], rtol=1e-11)
        errs.append(abs(f[0, 0] / (-4.0 * math.pi * C1) - 1.0))
        # eq. 46 / eq. 43: -T^r_t / (rho u^r) = h (-u_t) = sqrt(C2), pointwise, so the ratio has no quadrature error
        assert np.allclose(f[:, 3] / f[:, 0], math.sqrt(C2), rtol=1e-9)
        # eq. 45: no rotation, a = 0
        assert np.all(np.abs(f[:, 2]) < 1e-13 * np.abs(f[:, 0]))
        # eq. 44: no field
        assert np.all(f[:, 1] == 0.0)
    assert errs[2] < 1e-3 and errs[0] / errs[1] > 3.5 and errs[1] / errs[2] > 3.5, errs    # midpoint rule in theta


def test_phi_b_of_the_monopole_is_2_pi_c_on_every_shell():
    N = 48
    p, prim, g = _bondi_grid(N, 1.0)
    ng = p["ng"]
    f = np.array([g.shell_fluxes(i) for i in range(0, N, 7)])
    assert np.allclose(f[:, 1], f[0, 1], rtol=1e-12)               # sqrt(-g) B^1 does not depend on X1
    # B^1 = c / (Sigma r'), Sigma = r^2 at a = 0, r' = r (R0 = 0): c from any zone
    X1 = math.log(p["r_in"]) + (0 + 0.5) * (math.log(p["r_out"]) - math.log(p["r_in"])) / N
    r = math.exp(X1)
    c = prim[5, ng, ng + N // 2, ng] * r * r * r
    assert abs(f[0, 1] / (2.0 * math.pi * c) - 1.0) < 2e-3          # 1/2 c int |sin th| dth dphi = 2 pi c
    # the radial field is parallel to the flow: no Poynting flux, Edot / Mdot stays the hydrodynamic Bernoulli constant
    C1, C2 = _michel_constants(4.0 / 3.0, 8.0)
    assert np.allclose(f[:, 3] / f[:, 0], math.sqrt(C2), rtol=1e-9)


def test_shell_fluxes_argument_checks():
    p, prim, g = _bondi_grid(8, 0.0)
    out = np.zeros(4)
    import ctypes as C
    assert oracle.lib().oracle_shell_fluxes(g._h, C.c_int32(-1), out.ctypes.data_as(C.POINTER(C.c_double))) != 0
    assert oracle.lib().oracle_shell_fluxes(g._h, C.c_int32(8), out.ctypes.data_as(C.POINTER(C.c_double))) != 0


@pytest.mark.gpu
def test_gpu_shell_fluxes_match_the_oracle():
    import paper_2205_02484_b200 as cu
    for name, kw in (("C3", dict(n1=24, n2=20, n3=12)), ("C4", dict(n1=16, n2=130, n3=140)), ("C1", dict(n1=32, n2=32))):
        p = config(name, **kw)
        prim0, _ = fm_torus(p)
        ref = prim0.copy()
        g = oracle.Grid(p)
        g.bind(ref)
        s = cu.Solver(p, prim0)
        dt = g.cfl_dt(0.45)
        for _ in range(2):
            g.step(dt)
            s.step(dt)
        for i in (0, p["n1"] // 2, p["n1"] - 1):
            a = np.array(s.shell_fluxes(i))
            b = g.shell_fluxes(i)
            # sums of ~1e3..2e4 terms in different orders: compare against the sum of magnitudes' scale
            scale = np.maximum(np.abs(b), 1e-12 * np.max(np.abs(b)))
            assert np.all(np.abs(a - b) <= 1e-10 * scale + 1e-16), (name, i, a, b)
        with pytest.raises(cu.CuharmError):
            s.shell_fluxes(p["n1"])
        s.close()
