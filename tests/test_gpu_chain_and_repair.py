"""GPU parity of the inversion fallback chain (eqs. 11, 32, 33) and of the grid-wide
eq. 34 repair (A13) against the oracle: the two fallback methods as stages of their own, zone by zone;
whole RK2 steps with the chain on (flags, statistics, chain counters exact; primitives to the one-step tolerance);
a step in which thousands of zones fail, so that the repair runs on many blocks with its grid barrier."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
import paper_2205_02484_b200 as cu  # noqa: E402
from workloads import config  # noqa: E402
from workloads.states import rng  # noqa: E402
from workloads.torus import fm_torus  # noqa: E402

from test_gpu_parity import interior, prim_errors  # noqa: E402

PAIRS = [(0, 0), (0, 1), (0, 2), (0, 3), (1, 1), (1, 2), (1, 3), (2, 2), (2, 3), (3, 3)]


def full_metric(geom, i, j):
    """4x4 g_cov, g^con, sqrt(-g) of column (i, j) from the oracle's exported table (10 + 10 + 2 components)."""
    gcov, gcon = np.zeros((4, 4)), np.zeros((4, 4))
    for n, (a, b) in enumerate(PAIRS):
        gcov[a, b] = gcov[b, a] = geom[n, i, j]
        gcon[a, b] = gcon[b, a] = geom[10 + n, i, j]
    return gcov, gcon, geom[20, i, j]


def state_errors(got, ref, gam):
    """rho pointwise; u against the conditioning kappa of the energy inversion; velocities against their maximum."""
    kappa = (ref[0] + gam * ref[1]) / ref[1]
    return max(abs(got[0] / ref[0] - 1.0), abs(got[1] / ref[1] - 1.0) / max(1.0, kappa / 100.0),
               np.abs(got[2:5] - ref[2:5]).max() / max(np.abs(ref[2:5]).max(), 1e-300))


# ------------------------------------------------------------------ the two fallback methods, stage by stage
@pytest.mark.parametrize("gam", [4.0 / 3.0, 5.0 / 3.0])
def test_fallback_inversions_match_the_oracle_zone_by_zone(gam):
    p = config("C3", n1=10, n2=8, n3=2, gam=gam, inv_chain=1)
    prim, _ = fm_torus(p)
    r = rng(11)
    # well-conditioned random states at every zone (the ranges of the oracle's own pins: Gamma <= 3, u/rho in
    # [0.05, 1], b^2/rho in [1e-3, 10]); outside them the recovery of u amplifies round-off by kappa >> 100 on both sides
    geom0 = oracle.Grid(p).get_geom(0)
    for i in range(prim.shape[1]):
        for j in range(prim.shape[2]):
            gij = full_metric(geom0, i, j)[0][1:, 1:]
            for k in range(prim.shape[3]):
                rho = 10.0 ** r.uniform(-1, 1)
                v = r.normal(size=3) / np.sqrt(np.diag(gij))
                v *= np.sqrt((r.uniform(1.0, 3.0) ** 2 - 1.0) / (v @ gij @ v))
                B = r.normal(size=3) / np.sqrt(np.diag(gij))
                B *= np.sqrt(rho * 10.0 ** r.uniform(-3, 1) / (B @ gij @ B))
                prim[:, i, j, k] = [rho, rho * 10.0 ** r.uniform(np.log10(0.05), 0), *v, *B]
    g = oracle.Grid(p); g.bind(prim.copy())
    s = cu.Solver(p, prim)
    geom = g.get_geom(0)
    U = g.prim_to_cons(prim)
    n1g, n2g, n3g = prim.shape[1:]
    guess = prim.copy()
    guess[:5] *= 1.0 + 0.3 * (r.random(guess[:5].shape) - 0.5)
    US = np.zeros(prim.shape[1:])
    for i in range(n1g):
        for j in range(n2g):
            gcov, gcon, sg = full_metric(geom, i, j)
            for k in range(n3g):
                US[i, j, k] = oracle.entropy_cons(prim[:, i, j, k], gcov, gcon, sg, gam)
    Ud, gd, USd = torch.as_tensor(U).cuda(), torch.as_tensor(guess).cuda(), torch.as_tensor(US).cuda()
    got1, f1 = s.invert_fallback(1, Ud, gd)
    got2, f2 = s.invert_fallback(2, Ud, gd, USd)
    got1, f1, got2, f2 = got1.cpu().numpy(), f1.cpu().numpy(), got2.cpu().numpy(), f2.cpu().numpy()
    worst1 = worst2 = 0.0
    for i in range(n1g):
        for j in range(n2g):
            gcov, gcon, sg = full_metric(geom, i, j)
            for k in range(n3g):
                q = (slice(None), i, j, k)
                r1, fr1 = oracle.invert_1dw(U[q], gcov, gcon, sg, gam, guess[q])
                r2, fr2 = oracle.invert_entropy(U[q], US[i, j, k], gcov, gcon, sg, gam, guess[q])
                assert f1[i, j, k] == fr1 and f2[i, j, k] == fr2, (i, j, k, f1[i, j, k], fr1, f2[i, j, k], fr2)
                if fr1 == 0:
                    worst1 = max(worst1, state_errors(got1[q], r1, gam))
                if fr2 == 0:
                    worst2 = max(worst2, state_errors(got2[q], r2, gam))
    assert (f1 == 0).mean() > 0.95 and (f2 == 0).mean() > 0.95
    assert worst1 < 1e-11 and worst2 < 1e-11, (worst1, worst2)


def test_1d_method_takes_over_where_newton_gives_up_on_the_gpu_too():
    """Flag 2 of the 2D method (iteration cap from a far guess) -> the 1D method by Brent recovers the state."""
    gam = 4.0 / 3.0
    p = config("C3", n1=10, n2=8, n3=2, gam=gam, inv_chain=1, newton_maxit=2)
    prim, _ = fm_torus(p)
    g = oracle.Grid(p); g.bind(prim.copy())
    s = cu.Solver(p, prim)
    U = g.prim_to_cons(prim)
    guess = prim.copy()
    guess[0] *= 300.0; guess[1] *= 1e-3; guess[2:5] = 0.0
    Ud, gd = torch.as_tensor(U).cuda(), torch.as_tensor(guess).cuda()
    _, f2d = s.cons_to_prim(Ud, gd)
    got, f1d = s.invert_fallback(1, Ud, gd)
    f2d, f1d, got = f2d.cpu().numpy(), f1d.cpu().numpy(), got.cpu().numpy()
    _, f2d_ref = g.cons_to_prim(U, guess)
    assert np.array_equal(f2d, f2d_ref) and (f2d == 2).sum() >= 100
    assert (f1d[f2d == 2] == 0).all()
    sel = f2d == 2
    assert np.abs(got[0][sel] / prim[0][sel] - 1.0).max() < 1e-11
    assert np.abs(got[2:5][:, sel] - prim[2:5][:, sel]).max() < 1e-11 * max(np.abs(prim[2:5]).max(), 1.0)


# ------------------------------------------------------------------ whole steps with the chain on
CHAIN_CASES = [
    ("C4 failures only", "C4", dict(n1=32, n2=32, n3=20), dict(), 0.0, 1.0),
    ("C5 failures only", "C5", dict(n1=40, n2=24, n3=16), dict(r_in=20.0, r_max=41.0, beta0=30.0), 0.0, 1.0),
    ("C5 eq.33 zones", "C5", dict(n1=40, n2=24, n3=16), dict(r_in=20.0, r_max=41.0, beta0=30.0), 1e-2, 30.0),
    ("C3 PLM+HLL eq.33", "C3", dict(n1=32, n2=24, n3=40), dict(), 1e-2, 150.0),
]


@pytest.mark.parametrize("label,name,kw,tkw,beta_min,bscale", CHAIN_CASES, ids=[c[0] for c in CHAIN_CASES])
def test_steps_with_the_fallback_chain_match_the_oracle(label, name, kw, tkw, beta_min, bscale):
    p = config(name, inv_chain=1, beta_min=beta_min, **kw)
    prim0, _ = fm_torus(p, **tkw)
    prim0[5:8] *= bscale
    ref = prim0.copy()
    g = oracle.Grid(p); g.bind(ref)
    dt = g.cfl_dt(0.45)
    s = cu.Solver(p, prim0)
    s.use_graph(True)
    for n in range(2):
        g.step(dt); s.step(dt)
        cs, cr = s.chain_stats(), [int(x) for x in g.get_chain_stats()]
        assert cs == cr, (n, cs, cr)
        assert list(s.stats()) == [int(x) for x in g.get_stats()], (n, s.stats(), list(g.get_stats()))
    assert cr[0] + cr[3] > 0, "the case must exercise the chain"
    if beta_min > 0:
        assert cr[3] > 0, "the case must have eq. 33 zones"
    got = s.prim.cpu().numpy()
    # zones that went through Brent carry its tolerance (1e-14 relative on W or v^2) times the conditioning of the
    # recovery; everything else is the plain one-step parity
    err = prim_errors(p, got, ref, tol=1e-10)
    assert (err < 1e-10).all(), err
    assert s.divb()[1] < 1e-12


# ------------------------------------------------------------------ the repair on thousands of failed zones
@pytest.mark.parametrize("frac,patches", [(0.02, 0), (0.15, 40), (0.6, 0)])
def test_repair_stage_on_thousands_of_failed_zones_matches_the_oracle(frac, patches):
    """cuharm_repair against oracle_fixup on the same primitives and the same pattern of failed zones: isolated
    zones (face stencil), clusters (diagonal stencil, later passes, the last-resort rule) and a grid that is mostly
    failed.  0.15 x 46080 zones = ~7000 list entries = 27 blocks of the repair kernel: the grid barrier between the
    passes is exercised.  The repaired values are sums of 4 (or up to 8) neighbours: equal to round-off."""
    p = config("C3", n1=48, n2=40, n3=24)
    prim0, _ = fm_torus(p)
    ng = p["ng"]
    r = rng(29)
    bad = r.random((p["n1"], p["n2"], p["n3"])) < frac
    for _ in range(patches):
        i, j, k = r.integers(0, 36, size=3)
        bad[i:i + 4, j:j + 3, k % p["n3"]] = True
    flag = np.zeros(prim0.shape[1:], dtype=np.int32)
    flag[ng:-ng, ng:-ng, ng:-ng][bad] = 2
    g = oracle.Grid(p); g.bind(prim0.copy())
    s = cu.Solver(p, prim0)
    ref = s.prim.cpu().numpy().copy()          # with ghosts filled (identical fills: tested elsewhere)
    ref[:5, ng:-ng, ng:-ng, ng:-ng][:, bad] *= 1e6     # junk in the failed zones: it must not leak into any result
    work = torch.as_tensor(ref).cuda()
    st0, sr0 = s.stats(), [int(x) for x in g.get_stats()]
    g.fixup(ref, flag)
    s.repair(work, torch.as_tensor(flag).cuda())
    st, sr = s.stats(), [int(x) for x in g.get_stats()]
    for c in (0, 1, 7):
        assert st[c] - st0[c] == sr[c] - sr0[c] == (int(bad.sum()) if c < 2 else sr[c] - sr0[c]), (c, st, sr)
    if patches or frac > 0.5:
        assert sr[7] - sr0[7] > 0
    got = work.cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-14 * np.abs(ref).max()
    assert np.abs(got[:2] / ref[:2] - 1.0).max() < 1e-13
