"""GPU parity, second set: the paths the first set (test_gpu_parity.py) never reached — ceilings and Lorentz cap
(eqs. 36-37), phi-VARYING data on 256-zone rows in the launch configuration bench.py times, the
headline scheme (PPM + LLF) at 10 steps, 100 steps of the unperturbed torus, even ghost-layer counts, and a step
size that changes every step under graph replay (eq. 26).  Same error measure and tolerances as the
first set."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
import paper_2205_02484_b200 as cu  # noqa: E402
from workloads import config  # noqa: E402
from workloads.states import minkowski_params, rng  # noqa: E402
from workloads.torus import fm_torus  # noqa: E402

from test_gpu_parity import both, interior, prim_errors  # noqa: E402


# ------------------------------------------------------------------ S9: ceilings and Lorentz cap
def strong_field_state(p, bscale, gamma_patch):
    """A magnetised torus with B scaled by `bscale` and a 3 x 3 x 6 patch moving outwards with Lorentz factor
    `gamma_patch` (utilde^1 = sqrt((Gamma^2 - 1) / g_11))."""
    prim, _ = fm_torus(p)
    ng = p["ng"]
    prim[5:8] *= bscale
    g11 = oracle.Grid(p).get_geom(0)[4]
    i0, j0 = ng + 20, ng + 6
    for di in range(3):
        for dj in range(3):
            prim[2, i0 + di, j0 + dj, ng + 2:ng + 8] = np.sqrt((gamma_patch ** 2 - 1.0) / g11[i0 + di, j0 + dj])
    return prim


CEIL_CASES = [
    # the paper's ceilings (50, 2.5e3) on a field 300x the torus': b^2/rho > 50 at the torus edge, ~700 failed
    # inversions per step (repairs incl. the last-resort rule ride along)
    ("strong field", dict(gamma_max=1.5), 300.0, 2.0),
    # the torus' own field against tight limits: ceilings fire in ~1e3 zones, few failures
    ("tight limits", dict(sigma_max=1e-4, b2_over_u_max=1e-2, gamma_max=1.5), 1.0, 2.0),
]
# Here the Lorentz cap is exercised with Gamma_max = 1.5 against a Gamma = 2 patch; the paper's 50 against Gamma = 80 inside a
# step is test_lorentz_cap_inside_a_step_at_the_papers_gamma_max_50 below (a conditioning-aware comparison), and the rescale
# formula (A12) at Gamma_max = 50 is compared zone by zone in test_floors_stage_matches_the_oracle_zone_by_zone.


@pytest.mark.parametrize("label,kw,bscale,gpatch", CEIL_CASES, ids=[c[0] for c in CEIL_CASES])
def test_ceilings_and_lorentz_cap_fire_and_match(label, kw, bscale, gpatch):
    p = config("C4", n1=32, n2=32, n3=20, **kw)
    prim0 = strong_field_state(p, bscale, gpatch)
    ref = prim0.copy()
    g = oracle.Grid(p)
    g.bind(ref)
    dt = g.cfl_dt(0.45)
    s = cu.Solver(p, prim0)
    g.step(dt)
    s.step(dt)
    st, sr = list(s.stats()), [int(x) for x in g.get_stats()]
    assert sr[4] > 0 and sr[5] > 0, sr                      # ceilings applied, Lorentz caps applied
    assert st == sr, (st, sr)
    got = s.prim.cpu().numpy()
    err = prim_errors(p, got, ref)
    assert (err < 1e-11).all(), err
    for _ in range(4):
        g.step(dt)
        s.step(dt)
    st, sr = list(s.stats()), [int(x) for x in g.get_stats()]
    assert st[:6] == sr[:6], (st, sr)
    err = prim_errors(p, s.prim.cpu().numpy(), ref, tol=1e-8)
    assert (err < 1e-8).all(), err
    assert s.divb()[1] < 1e-12
    s.close()


def _zone_errors(p, got, ref):
    """The parity-policy measure zone by zone (interior): pointwise relative for rho and u, |dq| / max_grid|q_ref| for
    utilde^i and B^i."""
    g, r = interior(p, got), interior(p, ref)
    e = np.zeros_like(r)
    for v in range(8):
        if v < 2:
            e[v] = np.abs(g[v] - r[v]) / np.abs(r[v])
        else:
            grp = slice(2, 5) if v < 5 else slice(5, 8)
            scale = max(float(np.max(np.abs(r[v]))), 1e-3 * float(np.max(np.abs(r[grp]))))
            e[v] = np.abs(g[v] - r[v]) / scale
    return e


def test_lorentz_cap_inside_a_step_at_the_papers_gamma_max_50():
    """P:L265 (A12) at the paper's own Gamma_max = 50 against a Gamma = 80 patch, inside a full RK2 step.  The patch sits
    next to floor-density zones at rest, whose update is then a difference of terms ~1e5 times the result: in a few tens of
    zones the two sides differ by more than 1e-11 (up to ~1e-9 in rho).  That this is conditioning and not a difference
    of method is SHOWN here, not asserted in a comment: the oracle is run again on inputs wiggled by 1e-15 relative (four
    seeds), and in every zone and primitive where library and oracle differ by more than 1e-11 the oracle's own answer
    moves by at least a tenth as much (measured: 0.37 at the least).  Everywhere else the one-step tolerance holds; counters are equal; caps fire."""
    p = config("C4", n1=32, n2=32, n3=20)
    assert p["gamma_max"] == 50.0
    prim0 = strong_field_state(p, 1.0, 80.0)
    ref = prim0.copy()
    g = oracle.Grid(p)
    g.bind(ref)
    dt = g.cfl_dt(0.45)
    s = cu.Solver(p, prim0)
    g.step(dt)
    s.step(dt)
    st, sr = list(s.stats()), [int(x) for x in g.get_stats()]
    assert sr[5] > 0 and st[:6] == sr[:6], (st, sr)
    diff = _zone_errors(p, s.prim.cpu().numpy(), ref)
    s.close()
    kappa = (interior(p, ref)[0] + p["gam"] * interior(p, ref)[1]) / interior(p, ref)[1]
    diff[1] /= np.maximum(1.0, 1e-14 * kappa / 1e-11)             # prim_errors' kappa rule for u
    loose = diff >= 1e-11
    nz = int(np.count_nonzero(loose.any(axis=0)))
    sens = np.zeros_like(diff)
    for seed in (31, 32, 33, 34):
        w = prim0 * (1.0 + 1e-15 * rng(seed).choice([-1.0, 1.0], size=prim0.shape))
        gw = oracle.Grid(p)
        gw.bind(w)
        gw.step(dt)
        e = _zone_errors(p, w, ref)
        e[1] /= np.maximum(1.0, 1e-14 * kappa / 1e-11)
        sens = np.maximum(sens, e)
    print(f"Gamma_max = 50, Gamma = 80 patch: {nz} zones beyond 1e-11 (worst {diff.max():.2e}); the oracle's own response "
          f"to a 1e-15 input wiggle there: min ratio {np.min(sens[loose] / diff[loose]) if nz else float('nan'):.2f}, "
          f"caps applied {sr[5]}")
    assert nz < 200, nz
    assert (sens[loose] >= 0.1 * diff[loose]).all(), (diff[loose], sens[loose])


def test_floors_stage_matches_the_oracle_zone_by_zone():
    """cuharm_apply_floors against the oracle's C-12 on random states, a third of which violate a floor, a ceiling or
    the Lorentz cap (Gamma = 70 against the paper's 50): masks bit-exact, primitives to 1e-11.  The states are kept
    where the ceiling's re-inversion is well conditioned (kappa = Gamma^2 (rho + gam u + b^2)/u <~ 100: u/rho >= 0.03,
    Gamma <= 1.5, b^2/u <= 30 after the ceiling; zones pushed below the u floor and zones beyond the cap carry no
    field), checked with the oracle itself: a 1e-15 relative perturbation of the input moves its output by < 1e-13."""
    p = config("C4", n1=24, n2=20, n3=36, sigma_max=10.0, b2_over_u_max=30.0)
    r = rng(41)
    shape = (8, p["n1"] + 6, p["n2"] + 6, p["n3"] + 6)
    g = oracle.Grid(p)
    geo = g.get_geom(0)
    sq = [np.sqrt(geo[c])[:, :, None] for c in (4, 7, 9)]            # sqrt(g_11), sqrt(g_22), sqrt(g_33)

    def vectors(amplitude):
        n = r.normal(size=(3,) + shape[1:])
        n /= np.sqrt((n ** 2).sum(0))
        return [amplitude * n[c] / sq[c] for c in range(3)]

    prim = np.empty(shape)
    prim[0] = 10.0 ** r.uniform(-8, 0, shape[1:])                    # a third below the eq. 35 density floor
    prim[1] = prim[0] * 10.0 ** r.uniform(-1.5, 0, shape[1:])
    low = r.random(shape[1:]) < 0.1
    prim[1][low] *= 1e-6                                             # below the internal-energy floor
    prim[2:5] = vectors(10.0 ** r.uniform(-2, 0.0, shape[1:]))       # Gamma <= 1.5
    prim[5:8] = vectors(np.sqrt(prim[1] * 10.0 ** r.uniform(-2, 2.0, shape[1:])))   # b^2/u from 1e-2 to 1e2
    hot = r.random(shape[1:]) < 0.02
    prim[2][hot] = (np.sqrt(70.0 ** 2 - 1.0) / sq[0] * np.ones(shape[1:]))[hot]    # beyond the Lorentz cap
    prim[3][hot] = 0.0
    prim[4][hot] = 0.0
    prim[5:8, hot | low] = 0.0
    ref = prim.copy()
    mref = g.apply_floors(ref)
    wiggled = prim * (1.0 + 1e-15 * r.normal(size=prim.shape))
    g.apply_floors(wiggled)
    assert (prim_errors(p, wiggled, ref) < 1e-13).all()              # conditioning of the inputs, by the oracle itself
    s = cu.Solver(p, prim)
    d = torch.as_tensor(prim).cuda()
    mgot = s.apply_floors(d).cpu().numpy()
    got = d.cpu().numpy()
    assert np.array_equal(interior(p, mgot), interior(p, mref))
    mi = interior(p, mref)
    for bit in (1, 2, 4, 8):
        assert (mi & bit).sum() > 100, bit                 # every branch taken in many zones
    err = prim_errors(p, got, ref)
    assert (err < 1e-11).all(), err
    s.close()


# ------------------------------------------------------------------ phi-varying data on 256-zone rows (bench launch configuration)
def test_phi_varying_256_deep_slab_ppm_llf_one_and_ten_steps():
    """C4's scheme (MKS, PPM + LLF) on a 48 x 40 x 256 slab of the C4 grid with the seeded 3D perturbation, graph
    replay: two 128-zone tiles per row in update_tma_kernel with their k+-1 halo, nine 29-face chunks per row in the
    X3 flux kernel, strip-ordered tiles, E^1 / E^2 edges with non-cancelling X3 flux differences."""
    p = config("C4", n1=48, n2=40, n3=256)
    prim0, _ = fm_torus(p)
    ng = p["ng"]
    assert np.ptp(prim0[1, ng + 24, ng + 20, ng:-ng]) > 0          # phi-dependent input
    got, ref, s, g, dt = both(p, prim0, 1, graph=True)
    err = prim_errors(p, got, ref)
    assert (err < 1e-11).all(), err
    assert (prim_errors(p, got, ref, whole=True) < 1e-11).all()
    assert list(s.stats()) == [int(x) for x in g.get_stats()]
    for _ in range(9):
        g.step(dt)
        s.step(dt)
    err = prim_errors(p, s.prim.cpu().numpy(), ref, tol=1e-8)
    assert (err < 1e-8).all(), err
    assert s.divb()[1] < 1e-12
    assert list(s.stats()[:6]) == [int(x) for x in g.get_stats()[:6]]
    s.close()


def test_hundred_steps_unperturbed_torus():
    """SURVEY 8(c) parity policy: <= 1e-9 after 100 steps on smooth flows -- the unperturbed (magnetised) torus."""
    p = config("C4", n1=48, n2=48, n3=4)
    prim0, _ = fm_torus(p, perturb=0.0)
    got, ref, s, g, dt = both(p, prim0, 100, graph=True)
    err = prim_errors(p, got, ref, tol=1e-9)
    assert (err < 1e-9).all(), err
    assert s.divb()[1] < 1e-12
    s.close()


# ------------------------------------------------------------------ even ghost-layer count (generic update path)
@pytest.mark.parametrize("ng", [4, 5])
def test_other_ghost_layer_counts(ng):
    p = config("C4", n1=20, n2=16, n3=40, ng=ng)
    base = config("C4", n1=20, n2=16, n3=40)
    prim3, _ = fm_torus(base)
    # re-pad the ng = 3 array to ng layers (the ghost fill overwrites the padding)
    pad = ng - 3
    prim0 = np.ascontiguousarray(np.pad(prim3, ((0, 0), (pad, pad), (pad, pad), (pad, pad)), mode="edge"))
    ref = prim0.copy()
    g = oracle.Grid(p)
    g.bind(ref)
    dt = g.cfl_dt(0.45)
    s = cu.Solver(p, prim0)
    s.use_graph(True)
    for _ in range(2):
        g.step(dt)
        s.step(dt)
    got = s.prim.cpu().numpy()
    err = prim_errors(p, got, ref)
    assert (err < 2e-11).all(), err
    assert (prim_errors(p, got, ref, whole=True) < 2e-11).all()
    assert s.divb()[1] < 1e-12
    s.close()


# ------------------------------------------------------------------ a new dt every step, one graph
def test_changing_dt_under_graph_replay_is_bitwise_plain_and_follows_eq26():
    """cuharm_step_cfl takes dt on the device from eq. 26; under graph replay the same recorded graph serves every
    dt.  (i) graph replay == plain launches bit for bit over 10 steps with 10 different dt; (ii) the device dt equals
    the host formula (cuharm_last_cfl_dt) bit for bit; (iii) the run follows the oracle stepped with its own eq. 26."""
    p = config("C4", n1=32, n2=24, n3=12)
    prim0, _ = fm_torus(p)
    ref = prim0.copy()
    g = oracle.Grid(p)
    g.bind(ref)
    dt0 = g.cfl_dt(0.45)
    s1 = cu.Solver(p, prim0)
    s2 = cu.Solver(p, prim0)
    s2.use_graph(True)
    g.step(dt0); s1.step(dt0); s2.step(dt0)
    dts, t_sum = [dt0], dt0
    for n in range(10):
        expect = s1.last_cfl_dt(0.45)
        s1.step_cfl(0.45)
        s2.step_cfl(0.45)
        t1, d1 = s1.time()
        t2, d2 = s2.time()
        assert d1 == expect and d2 == expect, (n, d1, d2, expect)
        dto = g.last_cfl_dt(0.45)
        assert abs(dto / d1 - 1.0) < 1e-9
        g.step(dto)
        dts.append(d1)
        t_sum += d1
        assert t1 == t_sum and t2 == t_sum
    # dt really changed every step (the first eq. 26 value repeats dt0: the first predictor saw the initial state)
    assert dts[1] == dts[0] and len(set(dts[1:])) == len(dts) - 1
    assert torch.equal(s1.prim, s2.prim)
    n_graph = s2.launch_count()
    err = prim_errors(p, s1.prim.cpu().numpy(), ref, tol=1e-8)
    assert (err < 1e-8).all(), err
    # a host-chosen dt through the same graph, and a capped device dt
    s1.step(0.5 * dt0); s2.step(0.5 * dt0)
    s1.step_cfl(0.45, 0.25 * dt0); s2.step_cfl(0.45, 0.25 * dt0)
    assert s2.time()[1] == 0.25 * dt0
    assert torch.equal(s1.prim, s2.prim)
    assert s2.launch_count() > n_graph
    s1.close(); s2.close()


def test_non_finite_wave_speed_gives_zero_dt():
    p = minkowski_params(8, 8, 8)
    prim = np.zeros((8, 14, 14, 14))
    prim[0] = 1.0; prim[1] = 1.0
    prim[1, 6, 6, 6] = np.nan
    s = cu.Solver(p, prim)
    assert s.cfl_dt(0.45) == 0.0
    with pytest.raises(cu.CuharmError):
        s.step(0.0)
    s.close()


def test_device_side_eq26_carries_the_host_guard_and_repair_keeps_the_face_speeds():
    """(i) cuharm_step_cfl takes dt on the device; where the host formula answers 0 (a non-finite face speed)
    the device must answer 0 too -- a step that leaves the clock where it is -- not 1/0 or NaN; (ii) cuharm_repair as a
    stage of its own must not wipe the face-speed maxima of the last predictor, which cuharm_step_cfl reads next."""
    p = minkowski_params(8, 8, 8)
    prim = np.zeros((8, 14, 14, 14))
    prim[0] = 1.0; prim[1] = 1.0
    prim[1, 6, 6, 6] = np.nan
    s = cu.Solver(p, prim)
    s.step(1e-3)                                   # its predictor records a non-finite c_w
    assert s.last_cfl_dt(0.45) == 0.0
    t_before = s.time()[0]
    s.step_cfl(0.45)
    t_after, dt_last = s.time()
    assert dt_last == 0.0 and t_after == t_before
    s.close()
    p = config("C4", n1=24, n2=20, n3=12)
    prim0, _ = fm_torus(p)
    s = cu.Solver(p, prim0)
    s.step(s.cfl_dt(0.45))
    cw = s.last_cw()
    expect = s.last_cfl_dt(0.45)
    flag = torch.zeros(s.shape[1:], dtype=torch.int32, device=s.device)
    flag[10, 9, 7] = 2
    work = s.prim.clone()
    s.repair(work, flag)
    assert s.last_cw() == cw and min(cw) > 0.0
    s.step_cfl(0.45)
    assert s.time()[1] == expect and expect > 0.0
    s.close()


# ------------------------------------------------------------------ tensor-map vs one-dimensional bulk-copy staging
def test_tensor_map_update_kernel_is_bitwise_the_row_copy_kernel(monkeypatch):
    """update_tmap_kernel (12 tensor-map boxes per tile) against update_tma_kernel (63 row copies per tile; selected by
    CUHARM_NO_TMAP=1 at grid_init, the fallback when the driver's tensor-map encoder is unavailable): same tiles, same
    arithmetic, same expression per edge EMF -> identical bits, for both tile widths and a ragged last tile."""
    for name, kw in (("C4", dict(n1=20, n2=16, n3=150)), ("C3", dict(n1=24, n2=16, n3=40))):
        p = config(name, **kw)
        prim0, _ = fm_torus(p)
        res = []
        for no_tmap in (False, True):
            if no_tmap:
                monkeypatch.setenv("CUHARM_NO_TMAP", "1")
            else:
                monkeypatch.delenv("CUHARM_NO_TMAP", raising=False)
            s = cu.Solver(p, prim0)
            dt = s.cfl_dt(0.45)
            for _ in range(3):
                s.step(dt)
            res.append((s.prim.cpu().numpy().copy(), list(s.stats()), s.divb()))
            s.close()
        monkeypatch.delenv("CUHARM_NO_TMAP", raising=False)
        assert np.array_equal(res[0][0], res[1][0]) and res[0][1] == res[1][1] and res[0][2] == res[1][2]


# ------------------------------------------------------------------ the headline workload itself, every zone
def test_full_size_c4_workload_two_steps_every_zone_against_the_oracle():
    """BASELINE.json's headline config as bench.py runs it -- C4, 256 x 256 x 256, the seeded 3D-perturbed magnetised
    torus, PPM + LLF, graph replay, tensor-map update kernel with two 128-zone tiles per row -- against the oracle on ALL
    16.8 million zones (the oracle needs ~6 s per full step on 16 cores): <= 1e-11 per primitive after one RK2 step,
    <= 1e-10 after two, div B at round-off, counters equal."""
    p = config("C4")
    assert (p["n1"], p["n2"], p["n3"]) == (256, 256, 256)
    prim0, _ = fm_torus(p)
    ref = prim0.copy()
    g = oracle.Grid(p)
    g.bind(ref)
    dt = g.cfl_dt(0.45)
    s = cu.Solver(p, torch.from_numpy(prim0))
    assert abs(s.cfl_dt(0.45) / dt - 1.0) < 1e-13
    s.use_graph(True)
    for n, tol in ((1, 1e-11), (2, 1e-10)):
        g.step(dt)
        s.step(dt)
        got = s.prim.cpu().numpy()
        err = prim_errors(p, got, ref, whole=True, tol=tol)
        assert (err < tol).all(), (n, err)
        assert list(s.stats()) == [int(x) for x in g.get_stats()]
    assert s.divb()[1] < 1e-12 and g.divb()[1] < 1e-12
    assert abs(s.last_cfl_dt(0.45) / g.last_cfl_dt(0.45) - 1.0) < 1e-13
    s.close()
