"""Pins 9-11, 13, 15 of DESIGN.md: the oracle's grid-level scheme against what the mathematics fixes —
exact Riemann solutions, linear waves, the Michel (Bondi) steady state, flux-CT's algebraic identity,
symmetries, the CFL closed form, the boundary rules the paper states."""
import math

import numpy as np
import pytest

import oracle
from workloads import default_params, config
from workloads.bondi import bondi, michel_profile
from workloads.states import minkowski_params, sound_wave, fast_wave, shock_tube, uniform_state, rng
from workloads.torus import fm_torus

import exact_riemann as er

NG = 3


def interior(p, a):
    ng = p["ng"]
    return a[..., ng:ng + p["n1"], ng:ng + p["n2"], ng:ng + p["n3"]]


def run(p, prim, t_end=None, nsteps=None, xi=0.45):
    g = oracle.Grid(p)
    g.bind(prim)
    dt = g.cfl_dt(xi)
    if t_end is not None:
        nsteps = int(math.ceil(t_end / dt))
        dt = t_end / nsteps
    for _ in range(nsteps):
        g.step(dt)
    return g, dt, nsteps


# ------------------------------------------------------------------ the exact Riemann solver pins itself
@pytest.mark.parametrize("gam,left,right", [(5.0 / 3.0, (10.0, 13.33, 0.0), (1.0, 1e-6, 0.0)),
                                            (4.0 / 3.0, (1.0, 1.0, 0.5), (1.0, 1.0, -0.5)),
                                            (5.0 / 3.0, (1.0, 1000.0, 0.0), (1.0, 0.01, 0.0))])
def test_exact_riemann_solver_satisfies_jump_conditions_and_invariants(gam, left, right):
    sol = er.solve(gam, left, right)
    gas = sol["gas"]
    assert abs(sol["dv"]) < 1e-10                      # v continuous at the contact (p is by construction)
    for a, sign, rho_s in ((left, -1, sol["rhoLstar"]), (right, +1, sol["rhoRstar"])):
        ps, vs = sol["pstar"], sol["vstar"]
        if ps > a[1]:   # shock: Rankine-Hugoniot in the lab frame, [F] = V_s [U] for D, S, tau
            _, _, Vs = er._shock(gas, a, ps, sign)

            def cons(rho, p, v):
                W = 1.0 / math.sqrt(1 - v * v)
                h = gas.h(rho, p)
                D, S, E = rho * W, rho * h * W * W * v, rho * h * W * W - p
                return np.array([D, S, E]), np.array([D * v, S * v + p, S])
            Ua, Fa = cons(*a)
            Ub, Fb = cons(rho_s, ps, vs)
            assert np.allclose(Fb - Fa, Vs * (Ub - Ua), rtol=1e-9, atol=1e-11 * np.abs(Fa).max())
        else:           # rarefaction: entropy and the Riemann invariant constant
            assert abs(ps / rho_s ** gam - a[1] / a[0] ** gam) < 1e-12 * a[1] / a[0] ** gam
            sq = math.sqrt(gam - 1.0)

            def J(rho, p, v):
                cs = gas.cs(rho, p)
                return 0.5 * math.log((1 + v) / (1 - v)) - sign * (1.0 / sq) * math.log((sq + cs) / (sq - cs))
            assert abs(J(*a) - J(rho_s, ps, vs)) < 1e-11


# ------------------------------------------------------------------ pin 11: Minkowski shock tubes
@pytest.mark.parametrize("direction", [0, 1, 2])
def test_shock_tube_against_exact_riemann_solution(direction):
    gam = 5.0 / 3.0
    left, right = (10.0, 13.33, 0.0), (1.0, 1e-6 * 1e4, 0.0)     # mildly relativistic blast (p_R = 1e-2)
    sol = er.solve(gam, left, right)
    errs = []
    for N in (100, 200):
        n = [1, 1, 1]
        n[direction] = N
        bc = [1, 1, 1]
        bc[direction] = 0
        p = minkowski_params(*n, bc=bc, gam=gam, recon=0, riemann=1, newton_extra=2)
        prim = shock_tube(p, left, right, direction=direction, x0=0.5)
        t_end = 0.4
        g, dt, ns = run(p, prim, t_end=t_end, xi=0.4)
        x = (np.arange(N) + 0.5) / N
        ex = er.sample(sol, (x - 0.5) / t_end)
        rho = interior(p, prim)[0].reshape(-1)
        pg = (gam - 1.0) * interior(p, prim)[1].reshape(-1)
        ut = interior(p, prim)[2 + direction].reshape(-1)
        v = ut / np.sqrt(1 + ut * ut)
        e = np.mean(np.abs(rho - ex[0])) / np.mean(ex[0]) + np.mean(np.abs(pg - ex[1])) / np.mean(ex[1]) + np.mean(np.abs(v - ex[2]))
        errs.append(e)
        assert g.get_stats()[0] == 0                  # no inversion failures
    assert errs[1] < 0.06 and errs[1] < 0.75 * errs[0], errs      # converging (first order at the shock)
    # plateau between contact and shock: p*, v* to 2 %
    x = (np.arange(200) + 0.5) / 200
    xi_mid = 0.5 * (sol["vstar"] + er._shock(sol["gas"], right, sol["pstar"], +1)[2])
    m = np.argmin(np.abs((x - 0.5) / 0.4 - xi_mid))
    assert abs(pg[m] / sol["pstar"] - 1) < 0.02 and abs(v[m] / sol["vstar"] - 1) < 0.02


# ------------------------------------------------------------------ pin 11: linear waves, second order
@pytest.mark.parametrize("kind,direction,recon,riemann", [("sound", 0, 0, 0), ("sound", 1, 1, 1), ("sound", 2, 0, 1),
                                                          ("fast", 0, 0, 0), ("fast", 2, 1, 0), ("fast", 1, 0, 1)])
def test_linear_wave_second_order_convergence(kind, direction, recon, riemann):
    errs = []
    for N in (16, 32, 64):
        n = [1, 1, 1]
        n[direction] = N
        p = minkowski_params(*n, gam=5.0 / 3.0, recon=recon, riemann=riemann, newton_extra=2)
        amp = 1e-6
        if kind == "sound":
            prim, c = sound_wave(p, direction=direction, amp=amp, B0=tuple(0.3 if i == direction else 0.0 for i in range(3)))
        else:
            prim, c = fast_wave(p, direction=direction, bdir=(direction + 1) % 3, amp=amp)
        t_end = 0.5 / c                                # half a period
        run(p, prim, t_end=t_end, xi=0.4)
        if kind == "sound":
            ref, _ = sound_wave(p, direction=direction, amp=amp, t=t_end,
                                B0=tuple(0.3 if i == direction else 0.0 for i in range(3)))
        else:
            ref, _ = fast_wave(p, direction=direction, bdir=(direction + 1) % 3, amp=amp, t=t_end)
        e = np.mean(np.abs(interior(p, prim)[0] - interior(p, ref)[0])) / amp
        errs.append(e)
    order = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    # PLM-MC: clean second order.  PPM (A20, basic CW84): its monotonisation flattens every smooth extremum, which
    # is known to cost accuracy there; on a sine wave the L1 rate settles near 1.5-1.7 (still converging fast).
    if recon == 0:
        assert errs[-1] < 5e-3 and order[-1] > 1.8 and order[0] > 1.5, (errs, order)
    else:
        assert errs[-1] < 8e-3 and order[-1] > 1.45 and order[0] > 1.2, (errs, order)


def test_uniform_moving_magnetised_state_is_preserved():
    p = minkowski_params(6, 5, 4, newton_extra=2)
    q = [1.0, 0.7, 0.3, -0.2, 0.5, 0.4, 0.1, -0.3]
    prim = uniform_state(p, q)
    run(p, prim, nsteps=3)
    for v in range(8):
        assert np.allclose(prim[v], q[v], rtol=0, atol=2e-14)


# ------------------------------------------------------------------ pin 15: CFL closed form
def test_cfl_closed_form_uniform_minkowski():
    gam = 4.0 / 3.0
    p = minkowski_params(8, 4, 2, xmax=(1.0, 2.0, 0.5), gam=gam)
    rho, u, vx = 1.0, 0.5, 0.3
    lor = 1.0 / math.sqrt(1 - vx * vx)
    prim = uniform_state(p, [rho, u, lor * vx, 0, 0, 0, 0, 0])
    g = oracle.Grid(p)
    g.bind(prim)
    pg = (gam - 1) * u
    cs = math.sqrt(gam * pg / (rho + u + pg))
    # x: relativistic velocity addition; y, z: transverse sound speed cs/(Gamma sqrt(1 - vx^2 cs^2)) ... use the
    # textbook transverse formula lambda = +- cs sqrt(1-v^2) / sqrt(1 - v^2 cs^2)
    cx = (abs(vx) + cs) / (1 + abs(vx) * cs)
    ct = cs * math.sqrt(1 - vx * vx) / math.sqrt(1 - vx * vx * cs * cs)
    xi = 0.45
    dx = (1.0 / 8, 2.0 / 4, 0.5 / 2)
    inv = cx / (xi * dx[0]) + ct / (xi * dx[1]) + ct / (xi * dx[2])
    assert abs(g.cfl_dt(xi) * inv - 1.0) < 1e-13


def test_divb_normalised_measure_skips_subnormal_range_corners():
    """A4 (addition): corners whose terms sum to < 1e-290 do not enter max |D| / sum|terms| (rounding is absolute in
    the subnormal range, so the ratio is O(1) there for any field); max |D| still sees them, and a field of ordinary
    magnitude with the same non-solenoidal pattern is reported as O(1)."""
    p = minkowski_params(6, 5, 4)
    prim = uniform_state(p, [1.0, 1.0, 0, 0, 0, 0, 0, 0])
    rng = np.random.Generator(np.random.PCG64(7))
    pattern = rng.uniform(0.5, 1.0, size=prim[5].shape)
    prim[5] = 1e-300 * pattern          # not solenoidal, subnormal-range terms
    g = oracle.Grid(p)
    g.bind(prim)
    mabs, mnorm = g.divb()
    assert mnorm == 0.0 and 0.0 < mabs < 1e-295
    prim[5] = 1e-3 * pattern
    g.bind(prim)
    mabs, mnorm = g.divb()
    assert mnorm > 1e-2 and mabs > 1e-4


# ------------------------------------------------------------------ pin 9: flux-CT keeps eq. 23 for ARBITRARY fluxes
@pytest.mark.parametrize("kind", ["minkowski", "mks"])
def test_flux_ct_preserves_divb_for_arbitrary_fluxes(kind):
    r = rng(9)
    if kind == "minkowski":
        p = minkowski_params(8, 6, 10)
    else:
        p = default_params(n1=8, n2=6, n3=10)
    g = oracle.Grid(p)
    prim = np.zeros((8,) + g.shape)
    # a divergence-free start: B = 0 plus whatever flux-CT adds; then a second random update on top of it
    prim[0] = 1.0
    prim[1] = 1.0
    g.bind(prim)
    def periodic_wrap(F):
        # the fluxes of a periodic direction are themselves periodic (they come from periodic primitives); random
        # ones must be made so, or the wrap-around corners would compare two different values of the same edge
        ng = p["ng"]
        bcs = (p["bc_x1"], p["bc_x2"], p["bc_x3"])
        nn = (p["n1"], p["n2"], p["n3"])
        for d in range(3):
            if bcs[d] == 1:
                idx = ng + (np.arange(-ng, nn[d] + ng) % nn[d])
                F = np.take(F, idx, axis=1 + d)
        return np.ascontiguousarray(F)

    for rep in range(2):
        F = [periodic_wrap(r.normal(size=(8,) + g.shape)) for _ in range(3)]
        F1, F2, F3, E = g.flux_ct(*F)
        g.update_B_only(prim, F1, F2, F3, 0.37)
        g.apply_bc(prim)
        mabs, mnorm = g.divb()
        assert np.abs(interior(p, prim)[5:8]).max() > 0.1
        assert mnorm < 5e-14, (rep, mabs, mnorm)
    # negative control: the raw (unreplaced) fluxes do NOT preserve it
    g.update_B_only(prim, *F, 0.37)
    assert g.divb()[1] > 1e-3


def test_flux_ct_emf_is_the_four_face_average_eq21():
    p = minkowski_params(4, 4, 4)
    g = oracle.Grid(p)
    r = rng(21)
    F = [r.normal(size=(8,) + g.shape) for _ in range(3)]
    F1, F2, F3, E = g.flux_ct(*F)
    i, j, k = 4, 5, 3
    # E^3 at (I-1/2, J-1/2, K): eq. 21 (cyclic): 1/4 [F1(B2)_{J} + F1(B2)_{J-1} - F2(B1)_{I} - F2(B1)_{I-1}]
    e3 = 0.25 * (F[0][6, i, j, k] + F[0][6, i, j - 1, k] - F[1][5, i, j, k] - F[1][5, i - 1, j, k])
    assert abs(E[2, i, j, k] - e3) < 1e-15
    assert abs(F1[6, i, j, k] - 0.5 * (E[2, i, j, k] + E[2, i, j + 1, k])) < 1e-15       # eq. 22 (A3)
    assert abs(F2[5, i, j, k] + 0.5 * (E[2, i, j, k] + E[2, i + 1, j, k])) < 1e-15
    assert F1[5, i, j, k] == 0.0 and F2[6, i, j, k] == 0.0 and F3[7, i, j, k] == 0.0
    # hydrodynamic components untouched
    assert np.array_equal(F1[:5], F[0][:5])


# ------------------------------------------------------------------ pin 10/11: Michel (Bondi) steady state, a = 0
def _bondi_err(N, sigma_h, t_end=4.0):
    p = default_params(n1=N, n2=N, n3=1, a=0.0, gam=4.0 / 3.0, bc_x1=3, hslope=1.0, r_out=20.0, newton_extra=2)
    prim = bondi(p, sigma_h=sigma_h)
    P0 = prim.copy()
    g, dt, ns = run(p, prim, t_end=t_end)
    assert g.get_stats()[0] == 0
    rel = [np.mean(np.abs(interior(p, prim)[v] / interior(p, P0)[v] - 1.0)) for v in (0, 1)]
    dv = np.mean(np.abs(interior(p, prim)[2] - interior(p, P0)[2])) / np.abs(interior(p, P0)[2]).mean()
    return np.array(rel + [dv]), g


def test_michel_profile_is_a_solution():
    r = np.array([2.0, 3.0, 7.9, 8.0, 8.1, 15.0, 40.0])
    gam = 4.0 / 3.0
    T, rho, u, ur = michel_profile(gam, 8.0, r)
    n = 3.0
    assert np.allclose(rho * ur * r * r, (rho * ur * r * r)[0], rtol=1e-12)          # mass flux constant
    bern = (1 + (1 + n) * T) ** 2 * (1 - 2 / r + ur ** 2)                           # relativistic Bernoulli constant
    assert np.allclose(bern, bern[0], rtol=1e-10)
    cs2 = gam * T / (1 + (1 + n) * T)                                               # sound speed^2 = gam p / w
    # squared Mach number of the radial flow seen by a static observer: (u^r)^2 / (1 - 2/r + (u^r)^2) is its squared
    # proper velocity.  Supersonic inside the critical radius, subsonic outside, and exactly sonic AT r_c = 8, where
    # 1 - 2/r_c + u_c^2 = 1 - 3 u_c^2 and c_s^2 = u_c^2 / (1 - 3 u_c^2) (the Michel critical-point conditions)
    mach2 = ur ** 2 / (1 - 2 / r + ur ** 2) / cs2
    assert mach2[0] > 1 and mach2[1] > 1 and mach2[2] > 1 and mach2[4] < 1 and mach2[-1] < 1
    assert (np.diff(mach2) < 0).all()
    assert abs(mach2[3] - 1.0) < 1e-6, mach2[3]
    assert abs(ur[3] ** 2 - 1.0 / 16.0) < 1e-8           # u_c^2 = 1 / (2 r_c); a double root of the T equation: sqrt(eps)


def test_bondi_hydro_steady_state_second_order():
    e16, _ = _bondi_err(16, 0.0)
    e32, _ = _bondi_err(32, 0.0)
    order = np.log2(e16 / e32)
    assert (e32 < 2e-3).all() and (order > 1.7).all(), (e16, e32, order)


def test_bondi_magnetised_monopole_steady_and_divb():
    e16, _ = _bondi_err(16, 1.0)
    e32, g = _bondi_err(32, 1.0)
    order = np.log2(e16 / e32)
    # b^2/rho = 1 at the horizon: the magnetic terms dominate the inner zones and the rate is pre-asymptotic at
    # these sizes (measured: 1.2 at 32->64, 1.7 at 64->128 for u); require convergence, not the asymptotic rate
    assert (e32 < np.array([1e-3, 2e-3, 2e-2])).all() and (order > 0.8).all(), (e16, e32, order)
    assert g.divb()[1] < 1e-13


# ------------------------------------------------------------------ torus: div B, symmetry (pin 13), steadiness (pin 10)
def test_torus_divb_stays_at_roundoff_and_counts():
    p = config("C1", n1=32, n2=32, newton_extra=2)
    prim, info = fm_torus(p, beta0=100.0, beta_mode="min")
    g = oracle.Grid(p)
    g.bind(prim)
    assert g.divb()[1] < 1e-13
    dt = g.cfl_dt(0.9)
    for _ in range(10):
        g.step(dt)
    assert g.divb()[1] < 1e-12, g.divb()
    assert np.isfinite(prim).all() and (prim[0] > 0).all() and (prim[1] > 0).all()


@pytest.mark.parametrize("name,kw,perturb", [("C3", dict(n1=24, n2=16, n3=6), 0.0), ("C4", dict(n1=32, n2=32, n3=5), 0.04)])
def test_k_invariant_input_stays_bitwise_k_invariant_and_matches_2d(name, kw, perturb):
    """SURVEY 8(c) pin 13 / A31: phi-independent 3D input stays bitwise phi-independent, and every k-plane (ghost
    planes included) equals, bit for bit, the run of the same (r, theta) data at N3 = 1.  The full-size GPU test
    (test_gpu_parity.py::test_full_size_c4_...) leans on the second half, so it is pinned here for the oracle itself.
    Both schemes: PLM + HLL (C3) and PPM + LLF (C4, with the seeded perturbation of u drawn once per (i, j))."""
    p2 = config(name, **dict(kw, n3=1), newton_extra=2)
    prim2, _ = fm_torus(p2, perturb=perturb)
    p3 = config(name, **kw, newton_extra=2)
    ng = p3["ng"]
    prim3 = np.ascontiguousarray(np.broadcast_to(prim2[:, :, :, ng:ng + 1], prim2.shape[:3] + (p3["n3"] + 2 * ng,)))
    g2 = oracle.Grid(p2); g2.bind(prim2)
    dt = g2.cfl_dt(0.4)
    g3 = oracle.Grid(p3); g3.bind(prim3)
    # the k-sweep sees equal left and right states: its c_w is finite but its flux differences cancel exactly; dt is
    # taken from the 2D grid for both (the X3 CFL term differs: dx3 = 2 pi vs 2 pi / n3)
    for _ in range(2):
        g2.step(dt)
        g3.step(dt)
    for k in range(prim3.shape[3]):
        assert np.array_equal(prim3[..., k], prim3[..., 0])
        assert np.array_equal(prim3[..., k], prim2[..., min(k, prim2.shape[3] - 1)]), k
    assert np.array_equal(g3.get_stats()[:6] // p3["n3"], g2.get_stats()[:6])


def test_equatorial_mirror_symmetry_is_kept():
    p = config("C1", n1=24, n2=16, newton_extra=2)
    prim, _ = fm_torus(p, perturb=0.0, beta_mode="maxima")
    run(p, prim, nsteps=3, xi=0.5)
    sgn = np.array([1, 1, 1, -1, 1, 1, -1, 1.0])       # a polar vector's theta component flips; for B^i of a
    # single loop symmetric about the equator B^1 is ODD and B^2 EVEN in (theta - pi/2): use its own parity
    sgn[5], sgn[6], sgn[7] = -1, 1, -1       # B^3 is wound up from B^1: odd as well
    for v in range(8):
        a = prim[v][:, ::-1, :] * sgn[v]
        scale = np.abs(prim[v]).max() + 1e-300
        assert np.abs(a - prim[v]).max() / scale < 1e-11, v


def test_unmagnetised_torus_is_steady_at_second_order():
    errs = []
    for N in (32, 64):
        p = default_params(n1=N, n2=N, n3=1, gam=4.0 / 3.0, r_out=40.0, newton_extra=2)
        prim, info = fm_torus(p, perturb=0.0, field=False)
        P0 = prim.copy()
        g, dt, ns = run(p, prim, t_end=1.0, xi=0.4)
        ins = info["inside"]
        core = ins & (interior(p, P0)[0][:, :, 0] > 0.2)          # away from the torus surface (a kink: first order)
        e = np.abs(interior(p, prim)[0][:, :, 0] - interior(p, P0)[0][:, :, 0])[core].mean()
        errs.append(e)
    assert errs[1] < 2e-3 and np.log2(errs[0] / errs[1]) > 1.6, errs


# ------------------------------------------------------------------ boundary rules (A15)
def test_boundary_conditions_reflect_periodic_outflow():
    p = default_params(n1=6, n2=5, n3=4)
    g = oracle.Grid(p)
    r = rng(311)
    prim = r.uniform(0.5, 1.5, size=(8,) + g.shape)
    prim[2:5] = r.normal(size=(3,) + g.shape) * 0.1
    before = prim.copy()
    g.apply_bc(prim)
    ng, n1, n2, n3 = p["ng"], p["n1"], p["n2"], p["n3"]
    assert np.array_equal(interior(p, prim), interior(p, before))          # interior untouched
    sg = g.get_geom(0)[20]
    for m in range(ng):
        # polar reflection with u^2, B^2 sign flip
        for v in range(8):
            s = -1.0 if v in (3, 6) else 1.0
            assert np.array_equal(prim[v, ng:ng + n1, ng - 1 - m, ng:ng + n3], s * prim[v, ng:ng + n1, ng + m, ng:ng + n3])
            assert np.array_equal(prim[v, ng:ng + n1, ng + n2 + m, ng:ng + n3], s * prim[v, ng:ng + n1, ng + n2 - 1 - m, ng:ng + n3])
        # periodic in X3 (n3 >= ng here)
        assert np.array_equal(prim[:, :, :, ng - 1 - m], prim[:, :, :, ng + n3 - 1 - m])
        assert np.array_equal(prim[:, :, :, ng + n3 + m], prim[:, :, :, ng + m])
        # radial outflow: rho, u copied; sqrt(-g) B^i constant across the copy
        for v in (0, 1):
            assert np.array_equal(prim[v, ng - 1 - m, ng:ng + n2, ng:ng + n3], prim[v, ng, ng:ng + n2, ng:ng + n3])
        for v in (5, 6, 7):
            lhs = prim[v, ng + n1 + m, ng:ng + n2, ng:ng + n3] * sg[ng + n1 + m, ng:ng + n2, None]
            rhs = prim[v, ng + n1 - 1, ng:ng + n2, ng:ng + n3] * sg[ng + n1 - 1, ng:ng + n2, None]
            assert np.allclose(lhs, rhs, rtol=1e-14)
    # inflow check: no ghost zone at the inner edge moves outwards (u^1 <= 0), none at the outer edge inwards
    gc = g.get_geom(0)
    for i, sign in ((ng - 1, +1), (ng + n1, -1)):
        for j in range(ng, ng + n2):
            gcov = np.zeros((4, 4)); gcon = np.zeros((4, 4))
            pm = [0, 0, 0, 0, 1, 1, 1, 2, 2, 3]; pn = [0, 1, 2, 3, 1, 2, 3, 2, 3, 3]
            for s in range(10):
                gcov[pm[s], pn[s]] = gcov[pn[s], pm[s]] = gc[s, i, j]
                gcon[pm[s], pn[s]] = gcon[pn[s], pm[s]] = gc[10 + s, i, j]
            for k in range(ng, ng + n3):
                st = oracle.fluid_state(prim[:, i, j, k], gcov, gcon)
                assert sign * st["ucon"][1] <= 1e-14


def test_fixup_replaces_a_failed_zone_by_the_mean_of_its_four_face_neighbours_eq34():
    p = minkowski_params(6, 6, 2)
    g = oracle.Grid(p)
    r = rng(34)
    prim = r.uniform(0.5, 1.5, size=(8,) + g.shape)
    g.apply_bc(prim)
    before = prim.copy()
    flag = np.zeros(g.shape, dtype=np.int32)
    i, j, k = 5, 6, 3
    flag[i, j, k] = 2
    flag[7, 4, 4] = 2; flag[8, 4, 4] = 2        # a pair: face stencil blocked -> diagonal stencil (eq. 34, second form)
    g.fixup(prim, flag)
    for v in range(5):
        want = 0.25 * (before[v, i + 1, j, k] + before[v, i - 1, j, k] + before[v, i, j + 1, k] + before[v, i, j - 1, k])
        assert abs(prim[v, i, j, k] - want) < 1e-15
        want = 0.25 * (before[v, 8, 5, 4] + before[v, 8, 3, 4] + before[v, 6, 5, 4] + before[v, 6, 3, 4])
        assert abs(prim[v, 7, 4, 4] - want) < 1e-15
    assert np.array_equal(prim[5:], before[5:])                               # B untouched
    mask = np.ones(g.shape, bool); mask[i, j, k] = False; mask[7, 4, 4] = False; mask[8, 4, 4] = False
    assert np.array_equal(prim[:, mask], before[:, mask])
