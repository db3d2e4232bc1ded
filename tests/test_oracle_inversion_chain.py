"""Pins of the oracle's inversion fallback chain and entropy evolution (eq. 11 P:L94-98, P:L204,
P:L229-239 with eqs. 32-33): the 1D-W Brent method lands on the 2D Newton root; the entropy method round-trips
prim -> (U, sqrt(-g) S u^t) -> prim even when the energy variable is garbage; the entropy equation advanced in place of
the energy equation keeps the Michel flow steady at second order; eq. 33 selects the zones it says; failures are
routed as P:L233 says."""
import math

import numpy as np
import pytest

import oracle
from workloads import default_params, config
from workloads.bondi import bondi
from workloads.states import minkowski_params, uniform_state
from workloads.torus import fm_torus

from test_oracle_point_pins import rand_points, rand_prim, P, RNG


def cons_of(prim, gcov, gcon, sg, gam):
    return oracle.flux_vector(prim, gcov, gcon, sg, gam, 0)


def rel_err(a, b, gam):
    """rho pointwise; u scaled by the conditioning kappa = Gamma^2 (rho + gam u + b^2)/u >= (rho + gam u)/u of the energy
    inversion (pin 5); velocities against their own maximum."""
    kappa = (b[0] + gam * b[1]) / b[1]
    return max(abs(a[0] / b[0] - 1), abs(a[1] / b[1] - 1) / max(1.0, kappa / 100.0),
               np.abs(a[2:5] - b[2:5]).max() / max(np.abs(b[2:5]).max(), 1e-300))


# ------------------------------------------------------------------ (ii) 1D-W by Brent == 2D Newton where both converge
@pytest.mark.parametrize("gam", [4.0 / 3.0, 13.0 / 9.0, 5.0 / 3.0])
def test_1dw_brent_lands_on_the_2d_newton_root(gam):
    worst = 0.0
    for X1, X2 in rand_points(150):
        gcov, gcon, sg, al = oracle.metric_at(P, X1, X2)
        prim = rand_prim(Gmax=3.0, uor=(0.05, 1.0), sig=(1e-3, 10.0), gcov=gcov)
        U = cons_of(prim, gcov, gcon, sg, gam)
        guess = prim.copy()
        guess[:5] *= 1.0 + 0.3 * (RNG.random(5) - 0.5)
        p2, f2, _ = oracle.invert_2d(U, gcov, gcon, sg, gam, guess, extra=2)
        p1, f1 = oracle.invert_1dw(U, gcov, gcon, sg, gam, guess)
        assert f2 == 0 and f1 == 0, (f1, f2)
        worst = max(worst, rel_err(p1, p2, gam), rel_err(p1, prim, gam))
    assert worst < 1e-12, worst


def test_1dw_recovers_where_newton_gives_up():
    """'If the numerical method fails to produce results' (flag 2: the iteration cap, here 2 updates from a
    far guess) the 1D method by Brent takes over -- it needs a bracket, not a good guess."""
    gam = 4.0 / 3.0
    n1d = 0
    for X1, X2 in rand_points(60):
        gcov, gcon, sg, al = oracle.metric_at(P, X1, X2)
        prim = rand_prim(Gmax=2.0, uor=(0.05, 1.0), sig=(1e-3, 1.0), gcov=gcov)
        U = cons_of(prim, gcov, gcon, sg, gam)
        guess = prim.copy()
        guess[0] *= 300.0
        guess[1] *= 1e-3
        guess[2:5] = 0.0
        p2, f2, _ = oracle.invert_2d(U, gcov, gcon, sg, gam, guess, maxit=2)
        if f2 != 2:
            continue
        p1, f1 = oracle.invert_1dw(U, gcov, gcon, sg, gam, guess)
        assert f1 == 0
        assert rel_err(p1, prim, gam) < 1e-12
        n1d += 1
    assert n1d >= 30


# ------------------------------------------------------------------ (iii) the entropy method
@pytest.mark.parametrize("gam", [4.0 / 3.0, 5.0 / 3.0])
def test_entropy_inversion_round_trip_needs_no_energy(gam):
    """prim -> (U, U_S = sqrt(-g) S u^t) -> prim with S = p_g / rho^(gam-1) (A36), from a guess the method never
    uses, and with the energy variable replaced by garbage: by P:L213 the entropy method must not need it -- so it works
    exactly where eq. 30 has no root."""
    worst = 0.0
    for X1, X2 in rand_points(150):
        gcov, gcon, sg, al = oracle.metric_at(P, X1, X2)
        prim = rand_prim(Gmax=4.0, uor=(1e-3, 1.0), sig=(1e-3, 100.0), gcov=gcov)
        U = cons_of(prim, gcov, gcon, sg, gam)
        US = oracle.entropy_cons(prim, gcov, gcon, sg, gam)
        # closed form of the conserved entropy: sqrt(-g) (gam-1) u rho^(1-gam) Gamma / alpha
        lor = math.sqrt(1.0 + prim[2:5] @ gcov[1:, 1:] @ prim[2:5])
        assert abs(US / (sg * (gam - 1.0) * prim[1] * prim[0] ** (1.0 - gam) * lor / al) - 1.0) < 1e-14
        for bad_energy in (U[1], -7.0 * abs(U[1]), 1e30 * abs(U[1]), float("nan")):
            Ub = U.copy()
            Ub[1] = bad_energy
            got, flag = oracle.invert_entropy(Ub, US, gcov, gcon, sg, gam, np.ones(8))
            assert flag == 0
            e = max(abs(got[0] / prim[0] - 1), abs(got[1] / prim[1] - 1),
                    np.abs(got[2:5] - prim[2:5]).max() / np.abs(prim[2:5]).max())
            worst = max(worst, e)
        # with the energy variable of the wrong sign the energy equation has no physical root: Newton and 1D-W give up
        Ub = U.copy()
        Ub[1] = 7.0 * abs(U[1])              # T^t_t > 0: negative energy density for the normal observer
        f2d = oracle.invert_2d(Ub, gcov, gcon, sg, gam, prim)[1]
        f1d = oracle.invert_1dw(Ub, gcov, gcon, sg, gam, prim)[1]
        assert f2d != 0 and f1d != 0, (f2d, f1d)
    # u is recovered from S rho^(gam-1), whose only amplification is that of Gamma: d ln(Gamma) = Gamma^2 d(v^2) / 2
    assert worst < 1e-11, worst


def test_entropy_inversion_rejects_unphysical_conserved_states():
    """D < 0 or S < 0 'prevents the use of any of the aforementioned inversion methods'."""
    gam = 4.0 / 3.0
    X1, X2 = rand_points(1)[0]
    gcov, gcon, sg, al = oracle.metric_at(P, X1, X2)
    prim = rand_prim(gcov=gcov)
    U = cons_of(prim, gcov, gcon, sg, gam)
    US = oracle.entropy_cons(prim, gcov, gcon, sg, gam)
    assert oracle.invert_entropy(U, -US, gcov, gcon, sg, gam, prim)[1] == 1
    Ub = U.copy(); Ub[0] = -U[0]
    assert oracle.invert_entropy(Ub, US, gcov, gcon, sg, gam, prim)[1] == 1
    assert oracle.invert_1dw(Ub, gcov, gcon, sg, gam, prim)[1] == 1


# ------------------------------------------------------------------ eq. 11: the entropy flux and its evolution
def test_entropy_flux_of_a_uniform_state_is_s_u():
    """F_S(q, q) = sqrt(-g) S u^d: a uniform Minkowski state moving with velocity v has F_S = S Gamma v."""
    p = minkowski_params(6, 5, 4, gam=5.0 / 3.0)
    v = np.array([0.3, -0.2, 0.5])
    lor = 1.0 / math.sqrt(1.0 - v @ v)
    q = np.array([0.7, 0.4, *(lor * v), 0.3, 0.1, -0.2])
    prim = uniform_state(p, q)
    g = oracle.Grid(p)
    g.bind(prim)
    S = (p["gam"] - 1.0) * q[1] / q[0] ** (p["gam"] - 1.0)
    ng = p["ng"]
    for d in (1, 2, 3):
        FS = g.entropy_flux_dir(prim, d)
        assert abs(FS[ng + 2, ng + 2, ng + 2] - S * lor * v[d - 1]) < 1e-15


def _bondi_entropy_err(N):
    # beta_min = 2 > any beta: EVERY zone is inverted with the entropy method, first and only (eq. 33), i.e. the scheme
    # advances eq. 11 in place of the energy equation everywhere
    p = default_params(n1=N, n2=N, n3=1, a=0.0, gam=4.0 / 3.0, bc_x1=3, hslope=1.0, r_out=20.0, newton_extra=2,
                       inv_chain=1, beta_min=2.0)
    prim = bondi(p, sigma_h=0.0)
    P0 = prim.copy()
    g = oracle.Grid(p)
    g.bind(prim)
    dt = g.cfl_dt(0.45)
    ns = int(math.ceil(4.0 / dt))
    for _ in range(ns):
        g.step(4.0 / ns)
    ng = p["ng"]
    sl = (slice(ng, -ng), slice(ng, -ng), ng)
    ch = g.get_chain_stats()
    assert ch[3] == 2 * ns * N * N and ch[2] == ch[3] and g.get_stats()[0] == 0     # all zones, all recovered
    S0 = P0[1][sl] / P0[0][sl] ** p["gam"]
    S1 = prim[1][sl] / prim[0][sl] ** p["gam"]
    return np.array([np.mean(np.abs(prim[v][sl] / P0[v][sl] - 1.0)) for v in (0, 1)] + [np.mean(np.abs(S1 / S0 - 1.0))])


def test_entropy_evolution_keeps_michel_flow_steady_at_second_order():
    """The Michel flow is isentropic and steady: with eq. 11 advanced in place of the energy equation in every zone
    (flux of S, update of sqrt(-g) S u^t, eq. 32 inversion) it must stay put with second-order errors, and the
    specific entropy p / rho^gam must stay constant to second order."""
    e16 = _bondi_entropy_err(16)
    e32 = _bondi_entropy_err(32)
    order = np.log2(e16 / e32)
    assert (e32 < 2e-3).all() and (order > 1.7).all(), (e16, e32, order)


# ------------------------------------------------------------------ eq. 33 and the routing of P:L233
def test_beta_switch_selects_the_zones_eq33_says():
    p = config("C4", n1=24, n2=24, n3=4, inv_chain=1)
    prim, _ = fm_torus(p)
    prim[5:8] *= 200.0                      # beta0 = 100 -> 2.5e-3 at its minimum: below 1e-2 in part of the torus
    g = oracle.Grid(p)
    g.bind(prim)
    ng = p["ng"]
    # beta of every interior zone from the oracle's own fluid state (b^2) at the previous time level
    geo = g.get_geom(0)
    pm = [0, 0, 0, 0, 1, 1, 1, 2, 2, 3]
    pn = [0, 1, 2, 3, 1, 2, 3, 2, 3, 3]
    count = 0
    for i in range(ng, ng + p["n1"]):
        for j in range(ng, ng + p["n2"]):
            gcov = np.zeros((4, 4)); gcon = np.zeros((4, 4))
            for s in range(10):
                gcov[pm[s], pn[s]] = gcov[pn[s], pm[s]] = geo[s, i, j]
                gcon[pm[s], pn[s]] = gcon[pn[s], pm[s]] = geo[10 + s, i, j]
            for k in range(ng, ng + p["n3"]):
                q = prim[:, i, j, k]
                bsq = oracle.fluid_state(q, gcov, gcon)["bsq"]
                pg = (p["gam"] - 1.0) * q[1]
                count += pg / (pg + 0.5 * bsq) < 1e-2
    assert 0 < count < p["n1"] * p["n2"] * p["n3"]
    dt = g.cfl_dt(0.45)
    before = prim.copy()
    # predictor only sees P^n: one step = predictor (counted from P^n) + corrector (also keyed on P^n, A37)
    g.step(dt)
    ch = g.get_chain_stats()
    assert ch[3] == 2 * count, (ch, count)
    # with the switch off the same step takes the 2D route in those zones
    p_off = dict(p, beta_min=0.0)
    g2 = oracle.Grid(p_off)
    prim2 = before.copy()
    g2.bind(prim2)
    g2.step(dt)
    assert g2.get_chain_stats()[3] == 0
    # the switch changes the result (it is not a no-op) and both runs stay finite
    assert np.isfinite(prim).all() and np.isfinite(prim2).all()
    assert np.abs(prim[1] - prim2[1]).max() > 0.0


def test_chain_reduces_the_zones_that_reach_the_averaging():
    """the parity-size C5 copy sends 860 Newton failures per step straight to eq. 34; with the chain of
    P:L233 most of them are recovered by the 1D-W or the entropy method."""
    kw = dict(n1=40, n2=24, n3=16)
    tk = dict(r_in=20.0, r_max=41.0, beta0=30.0)
    res = {}
    for chain in (0, 1):
        p = config("C5", **kw, inv_chain=chain, beta_min=0.0)
        prim, _ = fm_torus(p, **tk)
        g = oracle.Grid(p)
        g.bind(prim)
        g.step(g.cfl_dt(0.45))
        res[chain] = (int(g.get_stats()[0]), [int(x) for x in g.get_chain_stats()])
        assert np.isfinite(prim).all()
    assert res[0][0] > 100 and res[0][1] == [0, 0, 0, 0]
    sent, by_1dw, by_ent, _ = res[1][1]
    assert abs(sent - res[0][0]) < 0.3 * res[0][0]            # about the same zones fail the 2D method (the corrector sees
    # a predictor state with recovered instead of averaged zones, so the counts are close, not equal)
    assert res[1][0] == sent - by_1dw - by_ent                # what is left for eq. 34
    assert res[1][0] < 0.2 * res[0][0], res
