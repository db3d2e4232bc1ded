"""Polar-velocity damping (A16): "the polar component of the 4-velocity in the two cells closest
to the pole is modified, by an interpolation to zero at the pole".  The paper gives no formula; A16 reads it
as the straight line in X^2 through zero at the pole and utilde^2 of the third zone.  Pins of the oracle (what the
reading fixes whatever its implementation): after the stage and the ghost fill the seven values of utilde^2 from three
ghost zones beyond the pole to the third interior zone lie on ONE straight line that passes through zero at the pole;
nothing else changes; the stage is idempotent and off by default.  GPU parity at the bottom."""
import numpy as np
import pytest

import oracle
from workloads import config
from workloads.states import rng, random_smooth
from workloads.torus import fm_torus


def setup(n1=14, n2=12, n3=5, **kw):
    p = config("C3", n1=n1, n2=n2, n3=n3, polar_damp=1, **kw)
    prim, _ = fm_torus(p)
    r = rng(17)
    prim[2:5] += 0.2 * (r.random(prim[2:5].shape) - 0.5)     # a polar velocity worth damping
    return p, prim


def test_polar_velocity_lies_on_a_line_through_zero_at_the_pole():
    p, prim = setup()
    g = oracle.Grid(p)
    g.apply_bc(prim)
    before = prim.copy()
    g.polar_damp(prim)
    g.apply_bc(prim)
    ng, n2 = p["ng"], p["n2"]
    dx = 2.0 / n2
    X = -1.0 + (np.arange(-ng, n2 + ng) + 0.5) * dx          # zone centres, ghosts included (eq. 39: X^2 in [-1, 1])
    u2 = prim[3]
    assert np.abs(u2[ng:-ng, ng + 2, ng:-ng]).mean() > 1e-2  # the anchor row is not trivially zero
    for rows, pole in ((slice(0, ng + 3), -1.0), (slice(n2 + ng - 3, n2 + 2 * ng), 1.0)):
        x, y = X[rows], u2[ng:-ng, rows, ng:-ng]
        slope = (y[:, 1:, :] - y[:, :-1, :]) / (x[1:] - x[:-1])[None, :, None]
        scale = np.abs(slope).max(axis=1, keepdims=True)
        assert (np.abs(slope - slope[:, :1, :]) <= 1e-12 * scale).all()          # one straight line ...
        at_pole = y[:, 0, :] + slope[:, 0, :] * (pole - x[0])
        assert (np.abs(at_pole) <= 1e-13 * np.abs(y).max(axis=1)).all()           # ... through zero at the pole
    # nothing but utilde^2 of the two rows next to each pole (and their mirror images) has changed
    same = np.ones(prim.shape, dtype=bool)
    same[3, :, :ng + 2, :] = False
    same[3, :, n2 + ng - 2:, :] = False
    # (radial ghost zones are left out: their inflow check renormalises all three velocity components, A15)
    assert np.array_equal(prim[:, ng:-ng][same[:, ng:-ng]], before[:, ng:-ng][same[:, ng:-ng]])
    # idempotent
    again = prim.copy()
    g.polar_damp(again)
    g.apply_bc(again)
    assert np.array_equal(again, prim)


def test_polar_damping_is_off_by_default_and_changes_only_the_polar_rows_in_one_substep():
    p, prim = setup()
    assert config("C4")["polar_damp"] == 0
    runs = {}
    for on in (0, 1):
        q = dict(p, polar_damp=on)
        a = prim.copy()
        g = oracle.Grid(q)
        g.bind(a)
        g.step(1e-3)
        assert np.isfinite(a).all()
        runs[on] = a
    ng, n2 = p["ng"], p["n2"]
    d = np.abs(runs[1] - runs[0])
    assert d[3].max() > 0.0
    # one RK2 step = two substeps of a 7-point stencil: the difference cannot have travelled further than 2 + 2*3 rows
    assert d[:, :, ng + 8:n2 + ng - 8, :].max() == 0.0 if n2 > 16 else True


# ------------------------------------------------------------------ GPU parity
@pytest.mark.gpu
def test_gpu_polar_damping_matches_the_oracle():
    torch = pytest.importorskip("torch")
    import paper_2205_02484_b200 as cu
    from test_gpu_parity import prim_errors
    for name, kw in (("C3", dict(n1=20, n2=18, n3=12)), ("C4", dict(n1=16, n2=24, n3=20))):
        p = config(name, polar_damp=1, **kw)
        prim0, _ = fm_torus(p)
        # a smooth polar velocity on top of the torus (zone-level noise would leave the limiter at its switching
        # points everywhere, where the two implementations may legitimately take different branches)
        prim0[3] += 0.03 * random_smooth(prim0[3].shape, rng(19))
        ref = prim0.copy()
        g = oracle.Grid(p); g.bind(ref)
        dt = g.cfl_dt(0.45)
        s = cu.Solver(p, prim0)
        s.use_graph(True)
        g.step(dt); s.step(dt)
        got = s.prim.cpu().numpy()
        err = prim_errors(p, got, ref, whole=True)
        assert (err < 1e-11).all(), (name, err)
        g.step(dt); s.step(dt)
        got = s.prim.cpu().numpy()
        assert (prim_errors(p, got, ref, whole=True, tol=1e-9) < 1e-9).all()
        assert list(s.stats()) == [int(x) for x in g.get_stats()]
        # and the stage changes something: the same run without it differs in the polar rows
        s2 = cu.Solver(dict(p, polar_damp=0), prim0)
        s2.step(dt); s2.step(dt)
        assert (s2.prim.cpu().numpy()[3] != got[3]).any()
