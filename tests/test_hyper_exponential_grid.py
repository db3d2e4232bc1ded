"""The hyper-exponential radial branch of eq. 39:
r = R0 + exp(X) for X < x_b, R0 + exp(X + (X - x_b)^n_X) beyond, x_b = ln(r_break - R0).
Pins of the oracle's map, metric and connection on that branch, and GPU-vs-oracle parity on such a grid."""
import math

import numpy as np
import pytest

import oracle
from workloads import default_params, config
from workloads.geometry import grid_coords, mks_to_ks
from workloads.torus import fm_torus

PH = default_params(n_x=4, r_break=10.0, r_out=200.0)
XB = math.log(10.0)
RNG = np.random.default_rng(39)


def test_radial_map_branches_join_smoothly_and_reach_r_out():
    m = oracle.radial_map(PH, XB - 0.3)
    assert m["r"] == pytest.approx(math.exp(XB - 0.3), rel=1e-15) and m["d1"] == pytest.approx(m["r"], rel=1e-15) \
        and m["d2"] == pytest.approx(m["r"], rel=1e-15)                      # plain exponential below x_b
    lo, hi = oracle.radial_map(PH, XB - 1e-9), oracle.radial_map(PH, XB + 1e-9)
    for k in ("r", "d1", "d2"):                                              # n_X = 4: C^3 at the junction
        assert abs(hi[k] / lo[k] - 1.0) < 1e-8
    y = 0.7
    m = oracle.radial_map(PH, XB + y)                                        # the definition, written out
    assert m["r"] == pytest.approx(math.exp(XB + y + y ** 4), rel=1e-14)
    assert m["d1"] == pytest.approx(m["r"] * (1 + 4 * y ** 3), rel=1e-14)
    assert m["d2"] == pytest.approx(m["r"] * ((1 + 4 * y ** 3) ** 2 + 12 * y ** 2), rel=1e-14)
    e = 1e-5                                                                 # derivatives against centred differences
    f = lambda x, k: oracle.radial_map(PH, x)[k]
    assert (f(XB + y + e, "r") - f(XB + y - e, "r")) / (2 * e) == pytest.approx(m["d1"], rel=1e-8)
    assert (f(XB + y + e, "d1") - f(XB + y - e, "d1")) / (2 * e) == pytest.approx(m["d2"], rel=1e-8)
    Xo = m["X_out"]
    assert oracle.radial_map(PH, Xo)["r"] == pytest.approx(200.0, rel=1e-13)
    assert XB < Xo < math.log(200.0)                                         # fewer e-folds of X than a pure log grid
    # switched off: the plain logarithmic grid
    assert oracle.radial_map(default_params(r_out=200.0), 1.0)["X_out"] == pytest.approx(math.log(200.0), rel=1e-15)


def test_grid_outer_edge_and_generator_geometry_agree_with_the_oracle():
    p = default_params(n1=32, n2=8, n3=1, n_x=4, r_break=10.0, r_out=200.0)
    (X1, X2, X3), dx = grid_coords(p, centred=False)
    ng = p["ng"]
    assert oracle.radial_map(p, X1[ng + p["n1"]])["r"] == pytest.approx(200.0, rel=1e-12)   # last face = r_out
    assert oracle.radial_map(p, X1[ng])["r"] == pytest.approx(p["r_in"], rel=1e-14)
    (C1, C2, C3), _ = grid_coords(p)
    r, th, drdX, dthdY = mks_to_ks(p, C1, 0.3)
    for i in (ng, ng + 10, ng + 31):
        m = oracle.coord_map(p, C1[i], 0.3)
        assert m["r"] == pytest.approx(r[i], rel=1e-13) and m["drdX"] == pytest.approx(drdX[i], rel=1e-13)
    g = oracle.Grid(p)
    geo = g.get_geom(0)
    # sqrt(-g) of the centre table = Sigma sin(th) r' th' with the hyper-exponential r' (closed form)
    i, j = ng + 28, ng + 3
    m = oracle.coord_map(p, C1[i], C2[j])
    assert m["r"] > 10.0
    Sig = m["r"] ** 2 + p["a"] ** 2 * math.cos(m["th"]) ** 2
    assert geo[20, i, j] == pytest.approx(Sig * math.sin(m["th"]) * m["drdX"] * m["dthdY"], rel=1e-13)


def _points(n):
    return list(zip(RNG.uniform(XB + 0.05, oracle.radial_map(PH, 0.0)["X_out"], n), RNG.uniform(-0.99, 0.99, n)))


def test_metric_on_the_hyper_exponential_branch_is_eq38_pushed_through_the_map():
    for X1, X2 in _points(25):
        gcov, gcon, sg, al = oracle.metric_at(PH, X1, X2)
        I = gcov @ gcon
        assert np.all(np.abs(I - np.eye(4)) <= 1e-13 * np.maximum(np.abs(gcov) @ np.abs(gcon), 1.0))
        assert abs(sg - math.sqrt(-np.linalg.det(gcov))) < 1e-10 * sg
        c = oracle.coord_map(PH, X1, X2)
        mr = oracle.radial_map(PH, X1)
        assert c["r"] == mr["r"] and c["drdX"] == mr["d1"] and c["r"] > 10.0
        r, th, a = c["r"], c["th"], PH["a"]
        rho2 = r * r + a * a * math.cos(th) ** 2
        dX = RNG.normal(size=4)
        dt, dr, dth, dph = dX[0], c["drdX"] * dX[1], c["dthdY"] * dX[2], dX[3]
        s2 = math.sin(th) ** 2
        ds2 = (-(1 - 2 * r / rho2) * dt * dt + (4 * r / rho2) * dr * dt + (1 + 2 * r / rho2) * dr * dr + rho2 * dth * dth
               + s2 * (rho2 + a * a * (1 + 2 * r / rho2) * s2) * dph * dph - (4 * a * r * s2 / rho2) * dph * dt
               - 2 * a * (1 + 2 * r / rho2) * s2 * dr * dph)
        assert abs(dX @ gcov @ dX - ds2) < 1e-12 * (np.abs(dX) @ np.abs(gcov) @ np.abs(dX))


def test_connection_on_the_hyper_exponential_branch():
    def g(X1, X2):
        return oracle.metric_at(PH, X1, X2)[0]

    def lnsg(X1, X2):
        return math.log(oracle.metric_at(PH, X1, X2)[2])

    for X1, X2 in _points(12):
        G = oracle.conn_at(PH, X1, X2)
        assert np.allclose(G, np.transpose(G, (0, 2, 1)), rtol=0, atol=1e-13 * np.abs(G).max())
        e = 1e-4
        tr = np.einsum("mmn->n", G)
        d1 = (-lnsg(X1 + 2 * e, X2) + 8 * lnsg(X1 + e, X2) - 8 * lnsg(X1 - e, X2) + lnsg(X1 - 2 * e, X2)) / (12 * e)
        assert abs(tr[1] - d1) < 1e-8 * max(1, abs(d1))            # Gamma^mu_{mu 1} = d_1 ln sqrt(-g): sees r''
        dg = np.zeros((4, 4, 4))
        dg[:, :, 1] = (-g(X1 + 2 * e, X2) + 8 * g(X1 + e, X2) - 8 * g(X1 - e, X2) + g(X1 - 2 * e, X2)) / (12 * e)
        dg[:, :, 2] = (-g(X1, X2 + 2 * e) + 8 * g(X1, X2 + e) - 8 * g(X1, X2 - e) + g(X1, X2 - 2 * e)) / (12 * e)
        gcon = oracle.metric_at(PH, X1, X2)[1]
        ref = 0.5 * (np.einsum("ls,skn->lnk", gcon, dg) + np.einsum("ls,snk->lnk", gcon, dg) - np.einsum("ls,nks->lnk", gcon, dg))
        assert np.all(np.abs(G - ref) < 1e-6 * max(1.0, np.abs(ref).max())), np.abs(G - ref).max()


@pytest.mark.gpu
def test_gpu_matches_the_oracle_on_a_hyper_exponential_grid():
    import paper_2205_02484_b200 as cu
    p = config("C4", n1=40, n2=24, n3=12, n_x=4, r_break=15.0, r_out=300.0)
    prim0, _ = fm_torus(p)
    s = cu.Solver(p, prim0)
    g = oracle.Grid(p)
    for loc in range(4):                       # geometry tables: centres, 1-faces, 2-faces, connection
        a = s.geom(loc).cpu().numpy()
        b = g.get_geom(loc)
        big = np.max(np.abs(b), axis=0, keepdims=True)
        err = np.abs(a - b) / np.maximum(np.abs(b), 1e-3 * big + 1e-300)
        if loc == 2:
            ng = p["ng"]
            for jj in (ng, ng + p["n2"]):
                err[[9, 19], :, jj] = 0.0
        assert err.max() < (1e-10 if loc == 3 else 1e-11), (loc, err.max())
    ref = prim0.copy()
    g.bind(ref)
    dt = g.cfl_dt(0.45)
    assert abs(s.cfl_dt(0.45) / dt - 1) < 1e-12
    for _ in range(2):
        g.step(dt)
        s.step(dt)
    got = s.prim.cpu().numpy()
    ng = p["ng"]
    sl = (slice(None), slice(ng, -ng), slice(ng, -ng), slice(ng, -ng))
    for v in range(8):
        a, b = got[sl][v], ref[sl][v]
        if v == 0:
            e = np.max(np.abs(a - b) / np.abs(b))
        elif v == 1:
            kappa = (ref[sl][0] + p["gam"] * b) / b
            e = np.max(np.abs(a - b) / np.abs(b) / np.maximum(1.0, 1e-14 * kappa / 2e-11))
        else:
            grp = slice(2, 5) if v < 5 else slice(5, 8)
            e = np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-3 * np.max(np.abs(ref[sl][grp])))
        assert e < 2e-11, (v, e)
    assert s.divb()[1] < 1e-12
    s.close()
