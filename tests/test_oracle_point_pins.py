"""Pins 1-8, 12 of DESIGN.md: the oracle's point-level functions against what the paper and the
mathematics fix (closed forms, invariants, textbook special cases, brute force)."""
import math

import numpy as np
import pytest

import oracle
from workloads import default_params

P = default_params()
RNG = np.random.default_rng(2205)


def rand_points(n, pole=False):
    X1 = RNG.uniform(math.log(1.1), math.log(40.0), n)
    X2 = RNG.uniform(-0.999, 0.999, n) if not pole else RNG.choice([-1, 1], n) * RNG.uniform(0.97, 0.9999, n)
    return list(zip(X1, X2))


def rand_prim(Gmax=2.0, uor=(0.1, 1.0), sig=(1e-3, 1.0), gcov=None):
    rho = 10 ** RNG.uniform(-4, 1)
    u = rho * 10 ** RNG.uniform(math.log10(uor[0]), math.log10(uor[1]))
    # random direction, magnitude from the target Lorentz factor using gcov
    d = RNG.normal(size=3)
    q2 = d @ gcov[1:, 1:] @ d
    lor = RNG.uniform(1.0, Gmax)
    ut = d * math.sqrt((lor * lor - 1.0) / q2)
    B = RNG.normal(size=3)
    B2 = B @ gcov[1:, 1:] @ B
    B *= math.sqrt(rho * 10 ** RNG.uniform(math.log10(sig[0]), math.log10(sig[1])) / B2)
    return np.array([rho, u, *ut, *B])


# ------------------------------------------------------------------ pin 3: coordinate map
def test_coord_map_fixed_points_and_symmetry():
    for h in (0.3, 1.0, 0.6):
        p = default_params(hslope=h)
        assert oracle.coord_map(p, 0.0, -1.0)["th"] == 0.0
        assert abs(oracle.coord_map(p, 0.0, 0.0)["th"] - math.pi / 2) < 1e-15
        assert abs(oracle.coord_map(p, 0.0, 1.0)["th"] - math.pi) < 1e-15
        for Y in RNG.uniform(0, 1, 20):
            s = oracle.coord_map(p, 0.3, Y)["th"] + oracle.coord_map(p, 0.3, -Y)["th"]
            assert abs(s - math.pi) < 1e-14
    # derivatives against central differences
    for X1, X2 in rand_points(10):
        c = oracle.coord_map(P, X1, X2)
        e = 1e-5
        dr = (oracle.coord_map(P, X1 + e, X2)["r"] - oracle.coord_map(P, X1 - e, X2)["r"]) / (2 * e)
        dth = (oracle.coord_map(P, X1, X2 + e)["th"] - oracle.coord_map(P, X1, X2 - e)["th"]) / (2 * e)
        d2 = (oracle.coord_map(P, X1, X2 + e)["dthdY"] - oracle.coord_map(P, X1, X2 - e)["dthdY"]) / (2 * e)
        assert abs(dr - c["drdX"]) < 1e-8 * c["r"]
        assert abs(dth - c["dthdY"]) < 1e-8
        assert abs(d2 - c["d2thdY2"]) < 1e-7
    # equator-concentrated: d theta / dY at the equator is h * pi/2 (eq. 39 with A14)
    assert abs(oracle.coord_map(P, 0.0, 0.0)["dthdY"] - 0.3 * math.pi / 2) < 1e-15


# ------------------------------------------------------------------ pin 1: metric
def test_metric_inverse_determinant_and_line_element():
    for X1, X2 in rand_points(40) + rand_points(10, pole=True):
        gcov, gcon, sg, al = oracle.metric_at(P, X1, X2)
        assert np.allclose(gcov, gcov.T, rtol=0, atol=0)
        I = gcov @ gcon
        scale = np.abs(gcov) @ np.abs(gcon)
        assert np.all(np.abs(I - np.eye(4)) <= 1e-14 * np.maximum(scale, 1.0))
        det = np.linalg.det(gcov)
        assert abs(sg - math.sqrt(-det)) < 1e-11 * sg
        assert abs(al - 1 / math.sqrt(-gcon[0, 0])) < 1e-15
        # eq. 38 written out term by term for a random displacement (KS), pushed through the map
        c = oracle.coord_map(P, X1, X2)
        r, th, a = c["r"], c["th"], P["a"]
        rho2 = r * r + a * a * math.cos(th) ** 2
        dX = RNG.normal(size=4)
        dt, dr, dth, dph = dX[0], c["drdX"] * dX[1], c["dthdY"] * dX[2], dX[3]
        s2 = math.sin(th) ** 2
        ds2 = (-(1 - 2 * r / rho2) * dt * dt + (4 * r / rho2) * dr * dt + (1 + 2 * r / rho2) * dr * dr + rho2 * dth * dth
               + s2 * (rho2 + a * a * (1 + 2 * r / rho2) * s2) * dph * dph - (4 * a * r * s2 / rho2) * dph * dt
               - 2 * a * (1 + 2 * r / rho2) * s2 * dr * dph)
        assert abs(dX @ gcov @ dX - ds2) < 1e-12 * (np.abs(dX) @ np.abs(gcov) @ np.abs(dX))


def test_metric_polar_face_and_minkowski():
    gcov, gcon, sg, al = oracle.metric_at(P, 1.0, -1.0, polar_face=1)
    assert sg == 0.0 and np.all(np.isfinite(gcon)) and np.all(np.isfinite(gcov))
    pm = default_params(coords=1)
    gcov, gcon, sg, al = oracle.metric_at(pm, 0.3, 0.2)
    eta = np.diag([-1.0, 1, 1, 1])
    assert np.array_equal(gcov, eta) and np.array_equal(gcon, eta) and sg == 1.0 and al == 1.0
    assert np.all(oracle.conn_at(pm, 0.3, 0.2) == 0.0)


# ------------------------------------------------------------------ pin 2: connection
def test_connection_symmetry_trace_and_finite_differences():
    def lnsg(X1, X2):
        return math.log(oracle.metric_at(P, X1, X2)[2])

    for X1, X2 in rand_points(25):
        G = oracle.conn_at(P, X1, X2)
        assert np.allclose(G, np.transpose(G, (0, 2, 1)), rtol=0, atol=1e-13 * np.abs(G).max())
        # Gamma^mu_{mu nu} = d_nu ln sqrt(-g)
        e = 1e-4
        tr = np.einsum("mmn->n", G)
        d1 = (-lnsg(X1 + 2 * e, X2) + 8 * lnsg(X1 + e, X2) - 8 * lnsg(X1 - e, X2) + lnsg(X1 - 2 * e, X2)) / (12 * e)
        d2 = (-lnsg(X1, X2 + 2 * e) + 8 * lnsg(X1, X2 + e) - 8 * lnsg(X1, X2 - e) + lnsg(X1, X2 - 2 * e)) / (12 * e)
        assert abs(tr[0]) < 1e-12 and abs(tr[3]) < 1e-12
        assert abs(tr[1] - d1) < 1e-9 * max(1, abs(d1)) and abs(tr[2] - d2) < 1e-8 * max(1, abs(d2))
        # full Christoffel from 4th-order differences of the metric
        def g(X1_, X2_):
            return oracle.metric_at(P, X1_, X2_)[0]
        dg = np.zeros((4, 4, 4))  # dg[s,k,n]
        dg[:, :, 1] = (-g(X1 + 2 * e, X2) + 8 * g(X1 + e, X2) - 8 * g(X1 - e, X2) + g(X1 - 2 * e, X2)) / (12 * e)
        dg[:, :, 2] = (-g(X1, X2 + 2 * e) + 8 * g(X1, X2 + e) - 8 * g(X1, X2 - e) + g(X1, X2 - 2 * e)) / (12 * e)
        gcon = oracle.metric_at(P, X1, X2)[1]
        ref = 0.5 * (np.einsum("ls,skn->lnk", gcon, dg) + np.einsum("ls,snk->lnk", gcon, dg) - np.einsum("ls,nks->lnk", gcon, dg))
        assert np.all(np.abs(G - ref) < 3e-8 * max(1.0, np.abs(ref).max())), np.abs(G - ref).max()


# ------------------------------------------------------------------ pin 4: fluid state
def test_fluid_state_invariants():
    for X1, X2 in rand_points(50):
        gcov, gcon, sg, al = oracle.metric_at(P, X1, X2)
        q = rand_prim(Gmax=10.0, gcov=gcov, sig=(1e-3, 10))
        S = oracle.fluid_state(q, gcov, gcon)
        assert abs(S["ucon"] @ S["ucov"] + 1.0) < 1e-12 * (np.abs(S["ucon"]) @ np.abs(S["ucov"]))
        assert abs(S["bcon"] @ S["ucov"]) < 1e-12 * (np.abs(S["bcon"]) @ np.abs(S["ucov"]))
        # B^i = b^i u^t - b^t u^i (eq. 4 with nu = t)
        Bi = S["bcon"][1:] * S["ucon"][0] - S["bcon"][0] * S["ucon"][1:]
        assert np.allclose(Bi, q[5:], rtol=1e-12, atol=1e-13 * np.abs(q[5:]).max())
        # modified velocity: u^i + Gamma beta^i / alpha with Gamma = alpha u^t (eq. 10)
        beta = gcon[0, 1:] * al * al
        assert np.allclose(S["ucon"][1:] + al * S["ucon"][0] * beta / al, q[2:5], rtol=1e-12, atol=1e-14)
        assert np.allclose(S["ucov"], gcov @ S["ucon"], rtol=1e-13) and abs(S["bsq"] - S["bcon"] @ S["bcov"]) < 1e-13 * abs(S["bsq"])


def test_flux_vector_against_contravariant_definition():
    """U and F from T^{mu nu} of eq. 5 built with upper indices and lowered by hand."""
    gam = P["gam"]
    for X1, X2 in rand_points(30):
        gcov, gcon, sg, al = oracle.metric_at(P, X1, X2)
        q = rand_prim(Gmax=5.0, gcov=gcov)
        S = oracle.fluid_state(q, gcov, gcon)
        rho, u = q[0], q[1]
        pg = (gam - 1) * u
        h = rho + u + pg
        Tup = (h + S["bsq"]) * np.outer(S["ucon"], S["ucon"]) + (pg + 0.5 * S["bsq"]) * gcon - np.outer(S["bcon"], S["bcon"])
        Tmix = Tup @ gcov  # T^mu_nu
        for d in range(4):
            F = oracle.flux_vector(q, gcov, gcon, sg, gam, d)
            ref = np.zeros(8)
            ref[0] = sg * rho * S["ucon"][d]
            ref[1:5] = sg * Tmix[d]
            ref[5:8] = sg * (S["bcon"][1:] * S["ucon"][d] - S["bcon"][d] * S["ucon"][1:])
            tol = 1e-12 * sg * (np.abs(Tup) @ np.abs(gcov)).max()
            assert np.all(np.abs(F - ref) <= tol)
        # the conserved B is sqrt(-g) B^i
        U = oracle.flux_vector(q, gcov, gcon, sg, gam, 0)
        assert np.allclose(U[5:], sg * q[5:], rtol=1e-12, atol=1e-14 * sg * np.abs(q[5:]).max())


# ------------------------------------------------------------------ pin 6: wave speeds
def test_wave_speeds_special_cases_and_dispersion_residual():
    eta = np.diag([-1.0, 1, 1, 1])
    gam = 5.0 / 3.0
    # fluid at rest in Minkowski -> +- c_ms
    q = np.array([1.0, 0.3, 0, 0, 0, 0.4, -0.2, 0.7])
    pg = (gam - 1) * q[1]; w = q[0] + q[1] + pg; b2 = q[5:] @ q[5:]
    cs2 = gam * pg / w; va2 = b2 / (b2 + w); cms = math.sqrt(va2 + cs2 * (1 - va2))
    for d in (1, 2, 3):
        c1, c2 = oracle.wave_speeds(q, eta, eta, gam, d)
        assert abs(c1 - cms) < 1e-14 and abs(c2 + cms) < 1e-14
    # B = 0, fluid moving along x: relativistic velocity addition (v +- cs)/(1 +- v cs)
    for v in (0.0, 0.3, -0.8, 0.99):
        lor = 1 / math.sqrt(1 - v * v)
        q = np.array([1.0, 0.3, lor * v, 0, 0, 0, 0, 0])
        cs = math.sqrt(cs2)
        c1, c2 = oracle.wave_speeds(q, eta, eta, gam, 1)
        assert abs(c1 - (v + cs) / (1 + v * cs)) < 1e-13 and abs(c2 - (v - cs) / (1 - v * cs)) < 1e-13
    # general: residual of eq. 18 with k_mu = (-omega, k_d), omega = k.u, k^2 = K.K
    for X1, X2 in rand_points(40):
        gcov, gcon, sg, al = oracle.metric_at(P, X1, X2)
        q = rand_prim(Gmax=4.0, gcov=gcov)
        S = oracle.fluid_state(q, gcov, gcon)
        pg = (P["gam"] - 1) * q[1]; w = q[0] + q[1] + pg
        cs2_ = P["gam"] * pg / w; va2_ = S["bsq"] / (S["bsq"] + w); cms2 = va2_ + cs2_ * (1 - va2_)
        for d in (1, 2, 3):
            c1, c2 = oracle.wave_speeds(q, gcov, gcon, P["gam"], d)
            assert c1 >= c2
            for c in (c1, c2):
                k = np.zeros(4); k[0] = -c; k[d] = 1.0
                om = k @ S["ucon"]
                kk = k @ gcon @ k
                K2 = kk + om * om
                scale = abs(om * om) + cms2 * (np.abs(k) @ np.abs(gcon) @ np.abs(k) + om * om)
                assert abs(om * om - cms2 * K2) < 1e-11 * scale


# ------------------------------------------------------------------ pin 7: reconstruction
def eq15_literal(qm, q0, qp):
    """eq. 15 typed as printed with the A2 correction (signed last branch)."""
    if (q0 - qm) * (qp - q0) < 0:
        return 0.0
    if abs(q0 - qm) < abs(qp - q0) and 2 * abs(q0 - qm) < 0.5 * abs(qp - qm):
        return 2 * (q0 - qm)
    if 2 * abs(qp - q0) < 0.5 * abs(qp - qm):
        return 2 * (qp - q0)
    return 0.5 * (qp - qm)


def minmod3(a, b, c):
    if a > 0 and b > 0 and c > 0:
        return min(a, b, c)
    if a < 0 and b < 0 and c < 0:
        return max(a, b, c)
    return 0.0


def test_mc_slope_is_minmod_and_exact_on_linear_data():
    for _ in range(20000):
        qm, q0, qp = RNG.normal(size=3) * 10 ** RNG.uniform(-3, 3)
        s = oracle.slope_mc(qm, q0, qp)
        ref = minmod3(2 * (q0 - qm), 2 * (qp - q0), 0.5 * (qp - qm))
        assert s == eq15_literal(qm, q0, qp)
        assert abs(s - ref) <= 1e-15 * max(abs(qm), abs(q0), abs(qp))
    assert oracle.slope_mc(1.0, 2.0, 1.5) == 0.0 and oracle.slope_mc(1.0, 0.0, 1.0) == 0.0
    assert oracle.slope_mc(1.0, 3.0, 5.0) == 2.0


@pytest.mark.parametrize("recon", [0, 1])
def test_reconstruction_linear_exact_and_bounded(recon):
    for _ in range(2000):
        a, b = RNG.normal(size=2)
        y = a + b * np.arange(-2, 3)
        l, r = oracle.recon_cell(recon, y)
        assert abs(l - (a - 0.5 * b)) < 1e-14 * (abs(a) + abs(b)) and abs(r - (a + 0.5 * b)) < 1e-14 * (abs(a) + abs(b))
        y = RNG.normal(size=5)
        l, r = oracle.recon_cell(recon, y)
        lo, hi = min(y[1:4]), max(y[1:4])
        assert lo - 1e-14 <= l <= hi + 1e-14 and lo - 1e-14 <= r <= hi + 1e-14
        # local extremum -> flat
        if (y[2] - y[1]) * (y[3] - y[2]) < 0:
            assert l == y[2] and r == y[2]


def test_ppm_exact_on_parabola_cell_averages():
    # cell averages of q(x) = a + b x + c x^2 over unit cells centred on x = -2..2; monotone on [-2.5, 2.5]
    for _ in range(2000):
        a, c = RNG.normal(size=2)
        b = (abs(c) * 5.0 + 0.1 + abs(RNG.normal())) * RNG.choice([-1, 1])
        x = np.arange(-2, 3.0)
        y = a + b * x + c * (x * x + 1.0 / 12.0)
        l, r = oracle.recon_cell(1, y)
        qe = lambda t: a + b * t + c * t * t
        assert abs(l - qe(-0.5)) < 1e-13 * (abs(a) + abs(b) + abs(c)) and abs(r - qe(0.5)) < 1e-13 * (abs(a) + abs(b) + abs(c))


# ------------------------------------------------------------------ pin 8: Riemann fluxes
def test_llf_hll_consistency():
    for X1, X2 in rand_points(20):
        gcov, gcon, sg, al = oracle.metric_at(P, X1, X2)
        q = rand_prim(Gmax=3.0, gcov=gcov)
        for d in (1, 2, 3):
            F = oracle.flux_vector(q, gcov, gcon, sg, P["gam"], d)
            for riem in (0, 1):
                Fb, cw = oracle.face_flux(q, q, gcov, gcon, sg, P["gam"], d, riem)
                assert np.allclose(Fb, F, rtol=1e-13, atol=1e-14 * np.abs(F).max())
            c1, c2 = oracle.wave_speeds(q, gcov, gcon, P["gam"], d)
            assert abs(cw - max(0, c1, -c2)) < 1e-15
    # eq. 20 -> eq. 17 when c_max = c_min: a static symmetric pair in Minkowski
    eta = np.diag([-1.0, 1, 1, 1])
    ql = np.array([1.0, 1.0, 0, 0, 0, 0.1, 0.2, 0.0]); qr = np.array([0.5, 0.2, 0, 0, 0, 0.1, -0.2, 0.1])
    # equalise the two fast speeds by hand: same c_ms needs same (cs2, va2); use identical thermodynamics, different B direction
    qr[:2] = ql[:2]; qr[5:] = [0.1, -0.2, 0.0]
    F0, cw0 = oracle.face_flux(ql, qr, eta, eta, 1.0, 4 / 3, 1, 0)
    F1, cw1 = oracle.face_flux(ql, qr, eta, eta, 1.0, 4 / 3, 1, 1)
    assert cw0 == cw1 and np.allclose(F0, F1, rtol=1e-14, atol=1e-16)


def test_llf_formula_on_random_pair():
    """eq. 17 retyped from the paper around the oracle's own U, F and c_w definition."""
    gam = P["gam"]
    for X1, X2 in rand_points(20):
        gcov, gcon, sg, al = oracle.metric_at(P, X1, X2)
        ql = rand_prim(Gmax=3.0, gcov=gcov); qr = rand_prim(Gmax=3.0, gcov=gcov)
        for d in (1, 2, 3):
            Fl = oracle.flux_vector(ql, gcov, gcon, sg, gam, d); Fr = oracle.flux_vector(qr, gcov, gcon, sg, gam, d)
            Ul = oracle.flux_vector(ql, gcov, gcon, sg, gam, 0); Ur = oracle.flux_vector(qr, gcov, gcon, sg, gam, 0)
            c1l, c2l = oracle.wave_speeds(ql, gcov, gcon, gam, d); c1r, c2r = oracle.wave_speeds(qr, gcov, gcon, gam, d)
            cmax = abs(max(0, c1r, c1l)); cmin = abs(max(0, -c2r, -c2l)); cw = max(cmax, cmin)
            Fb, cwo = oracle.face_flux(ql, qr, gcov, gcon, sg, gam, d, 0)
            assert cwo == cw
            assert np.allclose(Fb, 0.5 * (Fl + Fr - cw * (Ur - Ul)), rtol=1e-14, atol=1e-15 * np.abs(Fl).max())
            Fh, _ = oracle.face_flux(ql, qr, gcov, gcon, sg, gam, d, 1)
            ref = (cmax * Fl + cmin * Fr - cmax * cmin * (Ur - Ul)) / (cmax + cmin)
            assert np.allclose(Fh, ref, rtol=1e-13, atol=1e-15 * np.abs(Fl).max())


# ------------------------------------------------------------------ pin 5: inversion round trip
@pytest.mark.parametrize("gam", [4 / 3, 13 / 9, 5 / 3])
def test_prim_cons_prim_round_trip(gam):
    """north_star: prim -> cons -> prim to 1e-12 (well-conditioned states), max(1e-12, 1e-14 kappa) beyond."""
    nfail = 0
    its = []
    for X1, X2 in rand_points(300) + rand_points(60, pole=True):
        gcov, gcon, sg, al = oracle.metric_at(P, X1, X2)
        wide = RNG.random() < 0.4
        q = rand_prim(Gmax=3.0 if wide else 2.0, uor=(1e-2, 1.0) if wide else (0.1, 1.0), sig=(1e-3, 10.0 if wide else 1.0), gcov=gcov)
        U = oracle.flux_vector(q, gcov, gcon, sg, gam, 0)
        guess = q.copy()
        guess[:5] *= 1.0 + 0.1 * RNG.uniform(-1, 1, 5)
        out, flag, it = oracle.invert_2d(U, gcov, gcon, sg, gam, guess, tol=1e-10, maxit=30, extra=0)
        nfail += flag != 0
        its.append(it)
        S = oracle.fluid_state(q, gcov, gcon)
        lor2 = 1 + q[2:5] @ gcov[1:, 1:] @ q[2:5]
        kappa = lor2 * (q[0] + gam * q[1] + S["bsq"]) / q[1]
        tol = max(1e-12, 1e-14 * kappa)
        assert abs(out[0] - q[0]) <= tol * q[0]
        assert abs(out[1] - q[1]) <= tol * q[1]
        vs = np.abs(q[2:5]).max()
        assert np.all(np.abs(out[2:5] - q[2:5]) <= tol * max(vs, 1e-3))
        assert np.all(np.abs(out[5:] - q[5:]) <= 1e-14 * np.abs(q[5:]).max())
    assert nfail == 0
    assert max(its) <= 12


def test_inversion_residuals_eq29_eq30_with_documented_sign():
    """A6: eq. 30 holds with MINUS B^2(1+v^2)/2; the printed plus sign leaves an O(1) residual."""
    gam = 13 / 9
    X1, X2 = 1.2, 0.3
    gcov, gcon, sg, al = oracle.metric_at(P, X1, X2)
    q = rand_prim(Gmax=2.0, gcov=gcov, sig=(0.5, 1.0))
    U = oracle.flux_vector(q, gcov, gcon, sg, gam, 0)
    S = oracle.fluid_state(q, gcov, gcon)
    Qcov = al * U[1:5] / sg; Bc = np.array([0, *(al * U[5:] / sg)]); D = al * U[0] / sg
    ncon = np.array([1 / al, *(-al * gcon[0, 1:])])
    Qcon = gcon @ Qcov
    Bsq = Bc @ gcov @ Bc; QdB = Qcov @ Bc; Qdn = Qcov @ ncon
    Qt2 = Qcon @ Qcov + Qdn ** 2
    lor = al * S["ucon"][0]; v2 = 1 - 1 / lor ** 2
    pg = (gam - 1) * q[1]; W = lor ** 2 * (q[0] + q[1] + pg)
    assert abs(D - lor * q[0]) < 1e-13 * D  # A7: D = Gamma rho = alpha rho u^t
    f1 = Qt2 - v2 * (Bsq + W) ** 2 + QdB ** 2 * (Bsq + 2 * W) / W ** 2
    f2m = -Qdn - 0.5 * Bsq * (1 + v2) + QdB ** 2 / (2 * W * W) - W + pg
    f2p = -Qdn + 0.5 * Bsq * (1 + v2) + QdB ** 2 / (2 * W * W) - W + pg
    assert abs(f1) < 1e-12 * (Bsq + W) ** 2 and abs(f2m) < 1e-12 * W
    assert abs(f2p) > 1e-2 * Bsq
    # eq. 31
    assert abs(pg - (gam - 1) / gam * (W * (1 - v2) - D * math.sqrt(1 - v2))) < 1e-13 * W


def test_inversion_failure_codes():
    eta = np.diag([-1.0, 1, 1, 1])
    q = np.array([1.0, 0.1, 0.2, 0, 0, 0.1, 0, 0])
    U = oracle.flux_vector(q, eta, eta, 1.0, 4 / 3, 0)
    Ub = U.copy(); Ub[0] = -1.0
    out, flag, _ = oracle.invert_2d(Ub, eta, eta, 1.0, 4 / 3, q)
    assert flag == 1 and np.array_equal(out[:5], q[:5])
    Ub = U.copy(); Ub[1] = np.nan
    assert oracle.invert_2d(Ub, eta, eta, 1.0, 4 / 3, q)[1] == 1
    # energy too small for the momentum: negative internal energy
    Ub = U.copy(); Ub[1] = U[1] * 0.2   # U[1] = T^t_t < 0; shrinking |T^t_t| removes energy
    out, flag, _ = oracle.invert_2d(Ub, eta, eta, 1.0, 4 / 3, q)
    assert flag != 0 and np.array_equal(out[:5], q[:5]) and np.allclose(out[5:], Ub[5:])


# ------------------------------------------------------------------ pin 12: floors
def test_floors_postconditions_idempotence_and_lorentz_cap():
    p = default_params()
    for X1, X2 in rand_points(60):
        gcov, gcon, sg, al = oracle.metric_at(p, X1, X2)
        r = oracle.coord_map(p, X1, X2)["r"]
        q = rand_prim(Gmax=2.0, gcov=gcov, sig=(1e-2, 1.0))
        kind = RNG.integers(0, 4)
        if kind == 0:
            q[0] = 1e-12; q[1] = 1e-14
        elif kind == 1:   # strongly magnetised -> ceilings
            q[0] *= 1e-3; q[1] = q[0] * 1e-4
        elif kind == 2:   # too fast
            q[2:5] *= 80.0 / math.sqrt(1 + q[2:5] @ gcov[1:, 1:] @ q[2:5])
        out, mask = oracle.apply_floors(p, r, gcov, gcon, sg, q)
        S = oracle.fluid_state(out, gcov, gcon)
        rfl = max(p["rho_fl_abs"], p["rho_fl_coef"] * r ** p["rho_fl_pow"]); ufl = max(p["u_fl_abs"], p["u_fl_coef"] * r ** p["u_fl_pow"])
        assert out[0] >= rfl * (1 - 1e-12) and out[1] >= ufl * (1 - 1e-12)
        lor = math.sqrt(1 + out[2:5] @ gcov[1:, 1:] @ out[2:5])
        assert lor <= p["gamma_max"] * (1 + 1e-12)
        if mask & 8:
            assert abs(lor - p["gamma_max"]) < 1e-10 * p["gamma_max"]
        if not (mask & 8):
            assert S["bsq"] / out[0] <= p["sigma_max"] * (1 + 1e-8) and S["bsq"] / out[1] <= p["b2_over_u_max"] * (1 + 1e-8)
        assert np.array_equal(out[5:], q[5:])
        out2, mask2 = oracle.apply_floors(p, r, gcov, gcon, sg, out)
        assert np.allclose(out2, out, rtol=1e-9, atol=0) and not (mask2 & 3)
    # a healthy state is untouched
    gcov, gcon, sg, al = oracle.metric_at(p, 2.0, 0.1)
    q = np.array([1.0, 0.1, 0.1, 0.0, 0.01, 0.01, 0.0, 0.01])
    out, mask = oracle.apply_floors(p, 7.0, gcov, gcon, sg, q)
    assert mask == 0 and np.array_equal(out, q)
