"""BASELINE.json's configurations AS WRITTEN, at their full sizes, libcuharm against the CPU oracle:

  C3  128 x 128 x 64, PLM + HLL: one step <= 1e-11, ten steps <= 1e-8 (north_star), 100 steps reported
  C5  384 x 256 x 256, PPM + HLL, r_out = 1000 M: one step <= 1e-11
  C4  256^3, PPM + LLF: ten steps <= 1e-8 (one and two steps: tests/test_gpu_parity_wide.py)

Every zone is compared, ghosts included, in the parity-policy measure of tests/test_gpu_parity.py.  The oracle steps
C3 in ~0.3 s, C4 in ~6 s and C5 in ~9 s on 16 host cores.  Collected after the stage-level parity tests so that
`pytest -x` reports those first."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
import paper_2205_02484_b200 as cu  # noqa: E402
from workloads import config  # noqa: E402
from workloads.params import TORUS  # noqa: E402
from workloads.torus import fm_torus  # noqa: E402

from test_gpu_parity import prim_errors  # noqa: E402


def start(name):
    p = config(name)
    prim0, _ = fm_torus(p, **TORUS[name])
    ref = prim0.copy()
    g = oracle.Grid(p)
    g.bind(ref)
    dt = g.cfl_dt(0.45)
    s = cu.Solver(p, torch.from_numpy(prim0))
    assert abs(s.cfl_dt(0.45) / dt - 1.0) < 1e-13
    s.use_graph(True)
    return p, ref, g, s, dt


def kappa_rescaled_zones(p, ref, tol):
    """Zones whose internal-energy error is measured against 1e-14 kappa instead of tol (prim_errors' docstring)."""
    kappa = (ref[0] + p["gam"] * ref[1]) / ref[1]
    return int(np.count_nonzero(1e-14 * kappa > tol))


def test_c3_as_written_1_10_100_steps():
    p, ref, g, s, dt = start("C3")
    assert (p["n1"], p["n2"], p["n3"], p["recon"], p["riemann"]) == (128, 128, 64, 0, 1)
    done = 0
    for upto, tol in ((1, 1e-11), (10, 1e-8), (100, None)):
        while done < upto:
            g.step(dt)
            s.step(dt)
            done += 1
        got = s.prim.cpu().numpy()
        if tol is not None:
            err = prim_errors(p, got, ref, whole=True, tol=tol)
            assert (err < tol).all(), (upto, err)
            assert list(s.stats()[:6]) == [int(x) for x in g.get_stats()[:6]]
        else:
            # no north_star tolerance covers 100 steps of the perturbed torus: the number is REPORTED (pytest -s / -rP);
            # the bound below only catches a path that has come apart
            err = prim_errors(p, got, ref, whole=True, tol=1e-6)
            print(f"C3 128x128x64 PLM+HLL after 100 steps: max parity error per primitive {err}")
            assert (err < 1e-6).all(), err
        assert s.divb()[1] < 1e-12 and g.divb()[1] < 1e-12
    s.close()


def test_c5_as_written_one_step():
    p, ref, g, s, dt = start("C5")
    assert (p["n1"], p["n2"], p["n3"], p["recon"], p["riemann"], p["r_out"]) == (384, 256, 256, 1, 1, 1000.0)
    g.step(dt)
    s.step(dt)
    got = s.prim.cpu().numpy()
    err = prim_errors(p, got, ref, whole=True, tol=1e-11)
    print(f"C5 384x256x256 PPM+HLL r_out=1000: one step, max parity error per primitive {err}; "
          f"{kappa_rescaled_zones(p, ref, 1e-11)} of {ref[0].size} zones have 1e-14 kappa > 1e-11 (u measured against that)")
    assert (err < 1e-11).all(), err
    st, so = list(s.stats()), [int(x) for x in g.get_stats()]
    assert st[:6] == so[:6] and st[7] == so[7]
    # counter 6 is the total of Newton iterations.  The exit test |dW/W| < newton_tol is a floating-point decision: among
    # 25 million zones a few sit within an ulp of the threshold and take one iteration more or less on one side
    # (measured: 4 iterations in 9.4e7); the converged values agree to 1e-11 either way, which is what is asserted above
    print(f"Newton iterations: library {st[6]}, oracle {so[6]}")
    assert abs(st[6] - so[6]) <= 1e-6 * so[6]
    assert s.divb()[1] < 1e-12 and g.divb()[1] < 1e-12
    assert abs(s.last_cfl_dt(0.45) / g.last_cfl_dt(0.45) - 1.0) < 1e-13
    s.close()


def test_c4_as_written_ten_steps():
    p, ref, g, s, dt = start("C4")
    assert (p["n1"], p["n2"], p["n3"], p["recon"], p["riemann"]) == (256, 256, 256, 1, 0)
    for _ in range(10):
        g.step(dt)
        s.step(dt)
    got = s.prim.cpu().numpy()
    err = prim_errors(p, got, ref, whole=True, tol=1e-8)
    print(f"C4 256^3 PPM+LLF after 10 steps: max parity error per primitive {err}")
    assert (err < 1e-8).all(), err
    assert list(s.stats()[:6]) == [int(x) for x in g.get_stats()[:6]]
    assert s.divb()[1] < 1e-12 and g.divb()[1] < 1e-12
    s.close()


# ------------------------------------------------------------------ C2: Bondi + monopole at 64^2 / 128^2 / 256^2 to t = 50 M
def _bondi_run(p, sigma_h, t_end=50.0, xi=0.45):
    from workloads.bondi import bondi
    prim0 = bondi(p, sigma_h=sigma_h)
    s = cu.Solver(p, prim0)
    ns = int(np.ceil(t_end / s.cfl_dt(xi)))
    dt = t_end / ns
    s.use_graph(True)
    for _ in range(ns):
        s.step(dt)
    out = s.prim.cpu().numpy()
    assert s.stats()[0] == 0 and s.divb()[1] < 1e-11
    s.close()
    return prim0, out, ns, dt


def _interior2d(p, a):
    ng = p["ng"]
    return a[:, ng:ng + p["n1"], ng:ng + p["n2"], ng]


def _coarsen(a):
    return 0.25 * (a[:, 0::2, 0::2] + a[:, 1::2, 0::2] + a[:, 0::2, 1::2] + a[:, 1::2, 1::2])


def test_c2_as_written_three_resolutions_to_t50_and_the_oracle_at_64():
    """BASELINE.json configs[1]: a = 0.5, gam = 4/3, sonic radius 8 M, monopole field with b^2/rho = 1 at the horizon, MKS
    grids 64^2, 128^2, 256^2, integrated to t = 50 M (3 266 / 6 464 / 12 863 RK2 steps), all on the library.
    (i) The 64^2 run against the oracle stepped the same 3 266 steps, every zone: north_star's bound for smooth flows
    (1e-9, stated at 100 steps) is asserted here at 3 266 (measured 1.2e-11).
    (ii) L1 self-convergence 64 -> 128 -> 256 (2 x 2 zone averages of the finer run against the coarser one).  The initial
    data are the a = 0 Michel solution put on an a = 0.5 hole (A38), so the flow evolves and there is no exact
    solution to compare with; with b^2/rho = 1 at the horizon the rate at these sizes is pre-asymptotic (the oracle's
    own pin tests/test_oracle_scheme_pins.py::test_bondi_magnetised_monopole_steady_and_divb says the same of 16 -> 64).
    The orders are REPORTED; asserted is that every primitive converges at better than first order - 10 %.
    (iii) The scheme's second order at these sizes is shown where an exact solution exists: the unmagnetised Michel flow
    on a = 0 with the same grid family, 64^2 -> 128^2 against the exact steady state: order > 1.7."""
    runs = {}
    for N in (64, 128, 256):
        p = config("C2", n1=N, n2=N)
        runs[N] = (p,) + _bondi_run(p, 1.0)
    # (i)
    p, prim0, out, ns, dt = runs[64]
    assert (p["a"], p["n1"], p["n2"], p["n3"]) == (0.5, 64, 64, 1)
    ref = prim0.copy()
    g = oracle.Grid(p)
    g.bind(ref)
    for _ in range(ns):
        g.step(dt)
    err = prim_errors(p, out, ref, whole=True, tol=1e-9)
    print(f"C2 64^2 after {ns} steps (t = 50 M): max parity error per primitive {err}")
    assert (err < 1e-9).all(), err
    # (ii)
    I = {N: _interior2d(runs[N][0], runs[N][2]) for N in runs}
    e64 = np.array([np.mean(np.abs(I[64][v] - _coarsen(I[128])[v])) for v in (0, 1, 2, 3, 4, 5, 6, 7)])
    e128 = np.array([np.mean(np.abs(I[128][v] - _coarsen(I[256])[v])) for v in (0, 1, 2, 3, 4, 5, 6, 7)])
    order = np.log2(e64 / e128)
    print(f"C2 L1 self-convergence at t = 50 M: |64-128| {e64}\n |128-256| {e128}\n order {order}")
    assert (order > 0.9).all(), order
    # (iii)
    errs = []
    for N in (64, 128):
        p = config("C2", n1=N, n2=N, a=0.0)
        prim0, out, ns, dt = _bondi_run(p, 0.0)
        a, b = _interior2d(p, out), _interior2d(p, prim0)
        errs.append(np.array([np.mean(np.abs(a[0] / b[0] - 1.0)), np.mean(np.abs(a[1] / b[1] - 1.0)),
                              np.mean(np.abs(a[2] - b[2])) / np.mean(np.abs(b[2]))]))
    order0 = np.log2(errs[0] / errs[1])
    print(f"Michel flow, a = 0, to t = 50 M: L1 error vs the exact steady state 64^2 {errs[0]}, 128^2 {errs[1]}, order {order0}")
    assert (order0 > 1.7).all(), (errs, order0)


# ------------------------------------------------------------------ the fallback chain at the headline size
def test_c4_full_size_one_step_with_the_fallback_chain_busy():
    """256^3 with inv_chain = 1, beta_min = 1e-2 (eq. 33) and the torus field scaled x100, so that about 3 % of
    the zones (half a million per substep) take the entropy method: chain counters equal, every zone against the oracle to
    the tolerance of the small chain cases (1e-10: Brent's 1e-14 times the conditioning of the recovery)."""
    p = config("C4", inv_chain=1, beta_min=1e-2)
    prim0, _ = fm_torus(p, **TORUS["C4"])
    prim0[5:8] *= 100.0
    ref = prim0.copy()
    g = oracle.Grid(p)
    g.bind(ref)
    dt = g.cfl_dt(0.45)
    s = cu.Solver(p, torch.from_numpy(prim0))
    s.use_graph(True)
    g.step(dt)
    s.step(dt)
    cs, cr = s.chain_stats(), [int(x) for x in g.get_chain_stats()]
    print(f"C4 256^3, chain on, field x100: chain counters library {cs}, oracle {cr}")
    assert cs == cr and cr[3] > 2e5, (cs, cr)
    st, so = list(s.stats()), [int(x) for x in g.get_stats()]
    assert st[:6] == so[:6] and st[7] == so[7], (st, so)
    err = prim_errors(p, s.prim.cpu().numpy(), ref, whole=True, tol=1e-10)
    print(f"max parity error per primitive {err}")
    assert (err < 1e-10).all(), err
    assert s.divb()[1] < 1e-12 and g.divb()[1] < 1e-12
    s.close()
