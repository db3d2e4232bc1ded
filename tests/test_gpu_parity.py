"""GPU parity tests: libcuharm.so (through its C ABI / the thin binding) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances are `north_star`'s: <= 1e-11 per primitive after one RK2 step,
<= 1e-9 after 100 steps on smooth flows, <= 1e-8 after 10 steps on the perturbed torus, normalised div B
<= 1e-12.  Error measure: pointwise |dq|/|q_ref| for rho and u; for utilde^i and B^i
(which cross zero) max|dq| / max_grid|q_ref|."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
import paper_2205_02484_b200 as cu  # noqa: E402
from workloads import default_params, config  # noqa: E402
from workloads.bondi import bondi  # noqa: E402
from workloads.states import minkowski_params, shock_tube, sound_wave, rng  # noqa: E402
from workloads.torus import fm_torus  # noqa: E402


def interior(p, a):
    ng = p["ng"]
    return a[..., ng:ng + p["n1"], ng:ng + p["n2"], ng:ng + p["n3"]]


def prim_errors(p, got, ref, whole=False, tol=1e-11, vel_floor=0.0):
    """Per-primitive error in the parity-policy measure: pointwise relative for rho and u, max-norm
    relative to the grid maximum for utilde^i and B^i.  The internal energy is recovered from the total energy with
    the intrinsic condition number kappa = Gamma^2 (rho + gam u + b^2)/u (SURVEY 8(c) pin 5; the oracle's own round
    trip shows 2e-15..6e-15 kappa): where 1e-14 kappa exceeds `tol` the u error is measured against 1e-14 kappa
    instead, i.e. it is returned rescaled so that `< tol` is still the test.  kappa is taken at its lower bound
    (rho + gam u)/u (Gamma = 1, b = 0), which only makes the test stricter.  vel_floor: for Minkowski tests with
    |utilde| << 1 the velocity error is measured against max(max|utilde|, vel_floor) (the speed of light)."""
    g = got if whole else interior(p, got)
    r = ref if whole else interior(p, ref)
    out = []
    for v in range(8):
        if v == 0:
            out.append(float(np.max(np.abs(g[v] - r[v]) / np.abs(r[v]))))
        elif v == 1:
            kappa = (r[0] + p["gam"] * r[1]) / r[1]
            e = np.abs(g[v] - r[v]) / np.abs(r[v])
            out.append(float(np.max(e / np.maximum(1.0, 1e-14 * kappa / tol))))
        else:
            # a component that vanishes identically in the reference (utilde^2, B^3 of the unperturbed-in-theta torus)
            # is pure round-off of its siblings: never measure it against less than 1e-3 of their largest maximum
            grp = slice(2, 5) if v < 5 else slice(5, 8)
            scale = max(float(np.max(np.abs(r[v]))), 1e-3 * float(np.max(np.abs(r[grp]))))
            if v < 5:
                scale = max(scale, vel_floor)
            out.append(float(np.max(np.abs(g[v] - r[v])) / scale) if scale > 0 else float(np.max(np.abs(g[v]))))
    return np.array(out)


def both(p, prim0, nsteps, xi=0.45, graph=False):
    """Run nsteps on both implementations with the oracle's dt; returns (gpu prim, oracle prim, solver, grid, dt)."""
    ref = prim0.copy()
    g = oracle.Grid(p)
    g.bind(ref)
    dt = g.cfl_dt(xi)
    s = cu.Solver(p, prim0)
    if graph:
        s.use_graph(True)
    for _ in range(nsteps):
        g.step(dt)
        s.step(dt)
    return s.prim.cpu().numpy(), ref, s, g, dt


# ------------------------------------------------------------------ S0 geometry
@pytest.mark.parametrize("name,kw", [("C1", dict(n1=40, n2=36)), ("C5", dict(n1=48, n2=20, n3=1)), ("C2", dict(n1=16, n2=16))])
def test_geometry_tables_match(name, kw):
    p = config(name, **kw)
    prim = np.ones((8, p["n1"] + 6, p["n2"] + 6, p["n3"] + 6))
    s = cu.Solver(p, prim)
    g = oracle.Grid(p)
    for loc in range(4):
        a = s.geom(loc).cpu().numpy()
        b = g.get_geom(loc)
        scale = np.maximum(np.abs(b), 1e-300)
        err = np.abs(a - b) / scale
        if loc == 2:
            # on the axis itself g_33, g^33 are round-off of zero / its floored inverse (A32): never used, not compared
            ng = p["ng"]
            for jj in (ng, ng + p["n2"]):
                err[[9, 19], :, jj] = 0.0
        if loc == 3:
            # components that vanish analytically are round-off residue of O(1) cancellations on both sides
            big = np.max(np.abs(b), axis=0, keepdims=True)
            err = np.abs(a - b) / np.maximum(np.abs(b), 1e-3 * big)
            assert err.max() < 1e-10, (loc, err.max())
        else:
            assert err.max() < 1e-12, (loc, np.unravel_index(err.argmax(), err.shape), err.max())


def test_minkowski_geometry_is_flat():
    p = minkowski_params(4, 4, 4)
    s = cu.Solver(p, np.ones((8, 10, 10, 10)))
    g = oracle.Grid(p)
    for loc in range(4):
        assert np.array_equal(s.geom(loc).cpu().numpy(), g.get_geom(loc))


# ------------------------------------------------------------------ prim <-> cons
@pytest.mark.parametrize("gam", [4.0 / 3.0, 13.0 / 9.0, 5.0 / 3.0])
def test_prim_to_cons_and_inversion_round_trip(gam):
    p = config("C3", n1=20, n2=18, n3=37, gam=gam)     # 37+6 = 43: ragged tail of the 128-wide k tiling
    prim, _ = fm_torus(p)
    g = oracle.Grid(p)
    g.bind(prim)
    s = cu.Solver(p, prim)
    U_ref = g.prim_to_cons(prim)
    U = s.prim_to_cons().cpu().numpy()
    scale = np.max(np.abs(U_ref), axis=(1, 2, 3), keepdims=True)
    scale[5:8] = scale[5:8].max()                       # B^3 = 0 initially: its conserved image is round-off of B^1, B^2
    assert (np.abs(U - U_ref) / scale).max() < 1e-14
    # inversion of the ORACLE's conserved variables from a perturbed guess, against the oracle's own inversion
    r = rng(5)
    guess = prim.copy()
    guess[:5] *= 1.0 + 0.1 * (r.random(guess[:5].shape) - 0.5)
    ref, fref = g.cons_to_prim(U_ref, guess)
    got, fgot = s.cons_to_prim(torch.as_tensor(U_ref).cuda(), torch.as_tensor(guess).cuda())
    got, fgot = got.cpu().numpy(), fgot.cpu().numpy()
    assert np.array_equal(fgot, fref) and (fref == 0).all()
    assert (prim_errors(p, got, ref, whole=True) < 1e-11).all(), prim_errors(p, got, ref, whole=True)
    # and the round trip itself (north_star: 1e-12 where the inversion is well conditioned; kappa-scaled elsewhere)
    kappa = (prim[0] + gam * prim[1]) / prim[1]
    rt = np.abs(got[1] - prim[1]) / prim[1]
    assert (rt < np.maximum(1e-12, 1e-14 * kappa)).all()


def test_inversion_failure_flags_match():
    p = minkowski_params(4, 4, 4, newton_maxit=3)
    r = rng(7)
    prim = np.zeros((8, 10, 10, 10))
    prim[0] = 1.0; prim[1] = 1.0
    prim[2:5] = r.normal(size=(3, 10, 10, 10))
    prim[5:8] = r.normal(size=(3, 10, 10, 10))
    g = oracle.Grid(p); g.bind(prim)
    s = cu.Solver(p, prim)
    U = g.prim_to_cons(prim)
    U[0, 2, 2, 2] = -1.0                # D <= 0          -> 1
    U[1, 3, 3, 3] = np.nan              # non-finite      -> 1
    guess = prim.copy(); guess[0] *= 50.0; guess[2:5] = 0.0   # far guess + 3 iterations -> some 2s
    ref, fref = g.cons_to_prim(U, guess)
    got, fgot = s.cons_to_prim(torch.as_tensor(U).cuda(), torch.as_tensor(guess).cuda())
    assert np.array_equal(fgot.cpu().numpy(), fref)
    assert fref[2, 2, 2] == 1 and fref[3, 3, 3] == 1 and (fref == 2).any()


# ------------------------------------------------------------------ S2+S3 stage: face fluxes per direction
@pytest.mark.parametrize("recon", [0, 1])
@pytest.mark.parametrize("riemann", [0, 1])
def test_face_fluxes_match_per_direction(recon, riemann):
    p = config("C3", n1=20, n2=18, n3=12, recon=recon, riemann=riemann)
    prim, _ = fm_torus(p)
    g = oracle.Grid(p); g.bind(prim)
    s = cu.Solver(p, prim)
    ng = p["ng"]
    for d in (1, 2, 3):
        F_ref, cw_ref, cwmax = g.flux_dir(prim, d)
        F, cw = s.flux_dir(s.prim, d)
        F, cw = F.cpu().numpy(), cw.cpu().numpy()
        lo = [ng - 1] * 3; lo[d - 1] = ng
        sl = tuple(slice(lo[c], ng + (p["n1"], p["n2"], p["n3"])[c] + 1) for c in range(3))
        for v in range(8):
            a, b = F[(v,) + sl], F_ref[(v,) + sl]
            scale = np.abs(b).max()
            if scale > 0:
                assert np.abs(a - b).max() / scale < 1e-13, (d, v, np.abs(a - b).max() / scale)
        assert np.abs(cw[sl] - cw_ref[sl]).max() < 1e-13


# ------------------------------------------------------------------ one full RK2 step: <= 1e-11
CASES_1STEP = [
    ("C1", dict(), dict(beta_mode="min"), 0.9),                                   # 64x64x1, PLM+LLF
    ("C3", dict(n1=32, n2=24, n3=40), dict(), 0.45),                              # PLM+HLL, ragged k
    ("C4", dict(n1=32, n2=32, n3=20), dict(), 0.45),                              # PPM+LLF
    ("C5", dict(n1=40, n2=24, n3=16), dict(r_in=20.0, r_max=41.0, beta0=30.0), 0.45),   # PPM+HLL, r_out = 1000
]


@pytest.mark.parametrize("name,kw,tkw,xi", CASES_1STEP, ids=[c[0] for c in CASES_1STEP])
def test_one_rk2_step_matches_oracle(name, kw, tkw, xi):
    p = config(name, **kw)
    prim0, _ = fm_torus(p, **tkw)
    got, ref, s, g, dt = both(p, prim0, 1, xi=xi)
    err = prim_errors(p, got, ref)
    assert (err < 1e-11).all(), err
    # ghost zones too (boundary kernels), same measure over the whole array
    assert (prim_errors(p, got, ref, whole=True) < 1e-11).all()
    assert list(s.stats()) == list(g.get_stats())
    assert abs(s.last_cfl_dt(0.45) / g.last_cfl_dt(0.45) - 1) < 1e-13
    a, n = s.divb(); ar, nr = g.divb()
    assert n < 1e-12 and nr < 1e-12


def test_ten_steps_perturbed_torus_and_divb():
    p = config("C3", n1=32, n2=32, n3=16)
    prim0, _ = fm_torus(p)
    got, ref, s, g, dt = both(p, prim0, 10)
    err = prim_errors(p, got, ref, tol=1e-8)
    assert (err < 1e-8).all(), err
    assert s.divb()[1] < 1e-12
    assert list(s.stats()[:6]) == list(g.get_stats()[:6])


def test_c1_config_100_steps_reported_bound_not_a_north_star_tolerance_and_divb():
    p = config("C1")
    prim0, _ = fm_torus(p, beta_mode="min")
    got, ref, s, g, dt = both(p, prim0, 100, xi=0.9)
    err = prim_errors(p, got, ref, tol=1e-6)
    # C1 is the perturbed (turbulent) torus: the stated bound is 1e-8 at 10 steps; at 100 steps report and bound loosely
    assert (err < 1e-6).all(), err
    assert s.divb()[1] < 1e-12 and g.divb()[1] < 1e-12


def test_hundred_steps_smooth_bondi():
    p = config("C2", n1=64, n2=64)
    prim0 = bondi(p)
    got, ref, s, g, dt = both(p, prim0, 100)
    err = prim_errors(p, got, ref, tol=1e-9)
    assert (err < 1e-9).all(), err


def test_minkowski_shock_tube_and_wave_steps():
    p = minkowski_params(64, 1, 1, bc=(0, 1, 1), gam=5.0 / 3.0, riemann=1)
    prim0 = shock_tube(p, (10.0, 13.33, 0.0), (1.0, 1e-2, 0.0))
    got, ref, s, g, dt = both(p, prim0, 20, xi=0.4)
    assert (prim_errors(p, got, ref, tol=1e-10) < 1e-10).all(), prim_errors(p, got, ref)
    p = minkowski_params(1, 1, 48, gam=5.0 / 3.0, recon=1)
    prim0, _ = sound_wave(p, direction=2, amp=1e-3, B0=(0.0, 0.0, 0.3))
    got, ref, s, g, dt = both(p, prim0, 20, xi=0.4)
    # |utilde| ~ 4e-4 here: absolute round-off of the momentum/enthalpy ratio is ~ulp(1); measure against c = 1
    e = prim_errors(p, got, ref, tol=1e-10, vel_floor=1.0)
    assert (e < 1e-10).all(), e


def test_cfl_dt_and_divb_values_match():
    p = config("C3", n1=24, n2=20, n3=12)
    prim0, _ = fm_torus(p)
    ref = prim0.copy()
    g = oracle.Grid(p); g.bind(ref)
    s = cu.Solver(p, prim0)
    assert abs(s.cfl_dt(0.45) / g.cfl_dt(0.45) - 1) < 1e-13
    # a field that is NOT divergence-free: both must report the same (large) numbers
    r = rng(23)
    bad = ref.copy(); bad[5:8] += 0.01 * r.normal(size=bad[5:8].shape)
    g.bind(bad)
    s.load(bad)
    a, n = s.divb(); ar, nr = g.divb()
    assert abs(a / ar - 1) < 1e-12 and abs(n / nr - 1) < 1e-12 and nr > 1e-3
    # the same pattern scaled into the subnormal range: skipped by the normalised measure on both sides (A4)
    tiny = ref.copy(); tiny[5:8] = 1e-300 * r.uniform(0.5, 1.0, size=tiny[5:8].shape)
    g.bind(tiny)
    s.load(tiny)
    a, n = s.divb(); ar, nr = g.divb()
    assert n == 0.0 and nr == 0.0 and 0.0 < ar < 1e-290 and abs(a / ar - 1) < 1e-9


# ------------------------------------------------------------------ S8: repair of failed zones (eq. 34)
def test_failed_zones_are_repaired_like_the_oracle():
    p = config("C3", n1=24, n2=20, n3=8)
    prim0, _ = fm_torus(p)
    ng = p["ng"]
    # poison a few interior zones so that their inversion fails in the first substep: a huge field-aligned
    # momentum with tiny density gives D > 0 but no physical root within the iteration cap / v^2 range
    prim0[0, ng + 5, ng + 7, ng + 2] = np.nan
    prim0[0, ng + 10, ng + 9, ng + 3] = np.nan
    prim0[0, ng + 11, ng + 9, ng + 3] = np.nan          # a pair: face stencil blocked -> diagonal stencil
    prim0[1, ng + 15, ng + 4, ng + 6] = np.nan
    ref = prim0.copy()
    g = oracle.Grid(p); g.bind(ref)
    s = cu.Solver(p, prim0)
    dt = 0.01
    g.step(dt); s.step(dt)
    st, sr = s.stats(), g.get_stats()
    assert sr[0] > 0 and sr[1] > 0
    assert list(st) == list(sr), (st, list(sr))
    got = s.prim.cpu().numpy()
    assert np.isfinite(interior(p, ref)).all() and np.isfinite(interior(p, got)).all()
    assert (prim_errors(p, got, ref, tol=1e-10) < 1e-10).all(), prim_errors(p, got, ref)


# ------------------------------------------------------------------ S1: ghost fill, every combination of rules
def test_ghost_fill_matches_the_oracle_for_every_rule_combination():
    """cuharm_apply_bc (one launch composing X1 -> X2 -> X3) against the oracle's three sequential fills, whole arrays
    including edges and corners: MKS with outflow(+inflow check) / reflect / periodic and with `fixed` directions,
    Minkowski with periodic / outflow everywhere, and grids with fewer zones than ghost layers."""
    r = rng(31)
    cases = []
    for bcs in ((0, 2, 1), (3, 2, 1), (0, 3, 1), (0, 2, 3), (0, 2, 0), (3, 3, 1)):
        cases.append(default_params(n1=9, n2=8, n3=5, bc_x1=bcs[0], bc_x2=bcs[1], bc_x3=bcs[2]))
    for bcs in ((1, 1, 1), (0, 0, 0), (1, 0, 1), (0, 1, 3)):
        cases.append(minkowski_params(7, 6, 4, bc=bcs))
    cases.append(minkowski_params(2, 1, 1, bc=(1, 1, 1)))        # wraps repeatedly: n < ng
    cases.append(default_params(n1=5, n2=4, n3=1))
    for p in cases:
        shape = (8, p["n1"] + 6, p["n2"] + 6, p["n3"] + 6)
        prim = np.empty(shape)
        prim[0] = 1.0 + r.random(shape[1:]); prim[1] = 0.5 + r.random(shape[1:])
        prim[2:5] = 0.3 * r.normal(size=(3,) + shape[1:])
        prim[5:8] = r.normal(size=(3,) + shape[1:])
        ref = prim.copy()
        g = oracle.Grid(p)
        g.apply_bc(ref)
        s = cu.Solver(p, prim)            # bind applies the ghost fill once
        got = s.prim.cpu().numpy()
        scale = np.maximum(np.abs(ref), 1e-300)
        # copies, sign flips and periodic images are exact; the sqrt(-g) ratios and the inflow check (a square root and
        # two divisions, ill-conditioned in the ghost rows beyond the axis) differ by rounding: 1e-11 is far below the
        # O(1) error of any wrong source zone or missed rule
        assert np.max(np.abs(got - ref) / scale) < 1e-11, (p["bc_x1"], p["bc_x2"], p["bc_x3"], p["coords"])
        s.close()


# ------------------------------------------------------------------ full size, in the launch configuration bench.py times
def test_full_size_c4_k_invariant_torus_matches_the_2d_oracle():
    """BASELINE.json's headline size (C4: 256^3, PPM + LLF) through the same path bench.py times (graph replay, bulk-
    copy kernels with two 128-zone chunks per row, strip-ordered tiles).  The oracle cannot do 1.7e7 zones in
    seconds, but a property that holds at any size lets it check EVERY zone: phi-independent input stays phi-
    independent and equals the run at N3 = 1 (SURVEY 8(c) pin 13 / A31, pinned for the oracle itself in
    test_oracle_scheme_pins.py).  So the GPU steps the 2D perturbed, magnetised torus replicated along phi at
    256^3; the oracle steps the 256 x 256 x 1 original; tolerances as for one RK2 step."""
    p2 = config("C4", n3=1)
    prim2, _ = fm_torus(p2)                       # seeded +-2 % perturbation of u, one draw per (i, j)
    ref = prim2.copy()
    g = oracle.Grid(p2)
    g.bind(ref)
    dt = g.cfl_dt(0.45)
    g.step(dt)
    p3 = config("C4")
    ng = p3["ng"]
    assert (p3["n1"], p3["n2"], p3["n3"]) == (256, 256, 256)
    prim3 = np.ascontiguousarray(np.broadcast_to(prim2[:, :, :, ng:ng + 1], prim2.shape[:3] + (p3["n3"] + 2 * ng,)))
    s = cu.Solver(p3, prim3)
    s.use_graph(True)
    s.step(dt)
    got = s.prim.cpu().numpy()
    gi = interior(p3, got)
    assert (gi == gi[..., :1]).all(), "phi-invariant input must stay bitwise phi-invariant"
    err = prim_errors(p2, np.ascontiguousarray(got[..., :2 * ng + 1]), ref)   # the k = 0 plane, shaped like the 2D array
    assert (err < 1e-11).all(), err
    assert s.divb()[1] < 1e-12
    st = s.stats()
    assert st[0] == 0          # no inversion failures
    s.close()


# ------------------------------------------------------------------ launch modes, errors, edge shapes
def test_graph_replay_is_bitwise_identical_to_plain_launches():
    p = config("C4", n1=24, n2=16, n3=12)
    prim0, _ = fm_torus(p)
    a, _, s1, _, _ = both(p, prim0, 0)
    s2 = cu.Solver(p, prim0); s2.use_graph(True)
    for _ in range(3):
        s1.step(0.01); s2.step(0.01)
    assert torch.equal(s1.prim, s2.prim)
    assert s1.launch_count() > 0 and s2.launch_count() > 0


def test_tiny_and_ragged_grids():
    # n3 odd -> generic kernels; even -> bulk-copy kernels: 64-zone tiles (n3 <= 64), one ragged 128-zone chunk, two and
    # three chunks with a ragged tail; n2 prime / composite -> strip widths 1 and 6 of the tile order
    for n in ((1, 1, 1), (3, 2, 1), (5, 7, 129), (2, 3, 130), (6, 17, 50), (3, 5, 64), (3, 5, 66), (5, 18, 100), (4, 7, 258)):
        p = minkowski_params(*n)
        r = rng(n[2])
        shape = (8, n[0] + 6, n[1] + 6, n[2] + 6)
        prim0 = np.zeros(shape)
        prim0[0] = 1.0 + 0.1 * r.random(shape[1:]); prim0[1] = 0.5 + 0.1 * r.random(shape[1:])
        prim0[2:5] = 0.1 * r.normal(size=(3,) + shape[1:])
        B = r.normal(size=3)
        for i in range(3):
            prim0[5 + i] = B[i]                      # uniform field: divergence-free
        got, ref, s, g, dt = both(p, prim0, 2, xi=0.3)
        assert (prim_errors(p, got, ref, whole=True) < 1e-11).all(), (n, prim_errors(p, got, ref, whole=True))


def test_error_codes():
    import ctypes as C
    L = cu.lib()
    h = C.c_void_p()
    bad = cu.make_params(default_params(ng=2))
    assert L.cuharm_grid_init(C.byref(h), C.byref(bad), None) == -1
    bad = cu.make_params(default_params()); bad.struct_bytes = 8
    assert L.cuharm_grid_init(C.byref(h), C.byref(bad), None) == -1
    ok = cu.make_params(default_params(n1=8, n2=8))
    assert L.cuharm_grid_init(C.byref(h), C.byref(ok), None) == 0
    assert L.cuharm_step(h, 0.1) == -2                      # not bound
    need = L.cuharm_workspace_bytes(h)
    prim = torch.ones((8, 14, 14, 7), dtype=torch.float64, device="cuda")
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    assert L.cuharm_bind(h, C.c_void_p(prim.data_ptr()), C.c_void_p(ws.data_ptr()), need - 1) == -4
    assert L.cuharm_bind(h, C.c_void_p(prim.data_ptr()), C.c_void_p(ws.data_ptr()), need) == 0
    assert L.cuharm_step(h, 0.1) == -2                      # no geometry yet
    assert L.cuharm_metric_precompute(h) == 0
    assert L.cuharm_step(h, -1.0) == -1
    assert L.cuharm_step(h, float("nan")) == -1
    # split step: order is enforced; options are validated
    assert L.cuharm_substep(h, 0) == -2                     # no cuharm_set_dt yet
    assert L.cuharm_set_dt(h, 0.0) == -1
    assert L.cuharm_set_dt(h, 1e-3) == 0
    assert L.cuharm_substep(h, 1) == -2                     # corrector before predictor
    assert L.cuharm_substep(h, 2) == -1
    assert L.cuharm_substep(h, 0) == 0 and L.cuharm_substep(h, 1) == 0
    out2 = (C.c_int64 * 2)()
    assert L.cuharm_repair_pass(h, 0, 99, out2) == -1       # pass beyond fixup_max_passes
    assert L.cuharm_invert_fallback(h, 3, C.c_void_p(prim.data_ptr()), None, C.c_void_p(prim.data_ptr()), None) == -1
    assert L.cuharm_shell_fluxes(h, 99, (C.c_double * 4)()) == -1
    torch.cuda.synchronize()
    L.cuharm_destroy(h)
    for kw in (dict(polar_damp=1, bc_x2=1), dict(n1_global=8, i_offset=4, n1=8), dict(inv_chain=1, brent_maxit=0),
               dict(fixup_max_passes=99), dict(reserved=1)):
        bad = cu.make_params(default_params(**kw))
        assert L.cuharm_grid_init(C.byref(h), C.byref(bad), None) == -1, kw
