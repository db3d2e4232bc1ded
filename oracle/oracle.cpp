// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, obviously-correct CPU statement of the HARM conservative update of ideal
// GR-MHD that the cuHARM paper (arXiv 2205.02484) describes.  It exists to CHECK the CUDA
// library; it is not a product path.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may build, load or call it.  It shares no code, header,
// table or helper with paper_2205_02484_b200/ (the CUDA path) and neither includes the other.
//
// Citations: "P:L<n>" = /root/reference/PAPER.md line n (with the equation it falls in);
// "A<n>" = a reading of the paper listed in DESIGN.md (where the text is silent or garbled).
//
// Arithmetic: IEEE fp64, built with -O2 -ffp-contract=off (no FMA contraction), no blocking,
// no fusion, no reordering beyond what the equations state.  OpenMP `parallel for` over the
// outermost zone index is used only so that the timed CPU baseline can use all host cores; every
// zone's arithmetic is independent of the thread count.
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): see the table in DESIGN.md.  Parts whose
// conventions are fixed by DESIGN.md rather than by the paper or by mathematics are marked
// "parity unpinned" at the function that implements them.

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

// Same field order as the library's parameter block, declared independently (no shared header).
struct oracle_params {
  int32_t struct_bytes;
  int32_t n1, n2, n3, ng;
  int32_t coords;  // 0 = MKS (eq. 39), 1 = Minkowski-Cartesian (A39)
  double a, gam;
  double r_in, r_out, R0, hslope;
  double xmin[3], xmax[3];
  int32_t recon;    // 0 = PLM+MC (eqs. 15-16), 1 = PPM (A20)
  int32_t riemann;  // 0 = LLF (eq. 17), 1 = HLL (eq. 20)
  int32_t bc_x1, bc_x2, bc_x3;  // 0 outflow(+inflow check in MKS X1), 1 periodic, 2 polar-reflect, 3 fixed
  double rho_fl_coef, rho_fl_pow, rho_fl_abs;
  double u_fl_coef, u_fl_pow, u_fl_abs;
  double sigma_max, b2_over_u_max, gamma_max;
  double newton_tol;
  int32_t newton_maxit, newton_extra;
  int32_t fixup_max_passes;
  int32_t n_x;      // hyper-exponential radial branch of eq. 39: exponent n_X; < 2 = plain exponential
  double r_break;   // radius of the transition X = x_b (the paper: 400 M); used when n_x >= 2 and r_break > R0
  int32_t inv_chain;    // 1: inversion fallback chain: 2D Newton -> 1D-W Brent -> entropy; 0: straight to eq. 34
  int32_t brent_maxit;  // iteration cap of the Brent solver
  double beta_min;      // eq. 33: p_g / (p_g + b^2/2) of P^n below this -> entropy inversion first and only; <= 0 disables
  double brent_tol;     // relative tolerance of the Brent solver (A40)
  int32_t polar_damp;   // 1: the polar velocity of the two zones nearest each pole is interpolated to zero at the pole (A16)
  // this grid is a slab of a larger one, split along X1 (P:L271-273 splits along theta; the
  // choice of direction is free).  n1_global > 0: the full grid has n1_global zones in X1 and this slab holds zones
  // i_offset .. i_offset + n1 - 1 of it (coordinates, spacing and geometry are those of the full grid); slab_lo /
  // slab_hi = 1: the lower / upper X1 side is an internal boundary whose ghost zones are filled by the neighbouring
  // slab (halo exchange), never by the X1 boundary rule.
  int32_t n1_global, i_offset, slab_lo, slab_hi;
  int32_t reserved;     // keeps the block a multiple of 8 bytes; must be 0
};

}  // extern "C"

namespace {

const double PI = 3.14159265358979323846;

// ------------------------------------------------------------------------------------------
// C-1  Coordinates (eq. 39; A14: the sine argument is pi(1+Y), not pi(1+Y)/2).
// ------------------------------------------------------------------------------------------
struct Coord {
  double r, th, drdX, dthdY, d2thdY2, d2rdX2;
};

// eq. 39, radial part: r = R0 + exp(X) for X < x_b, R0 + exp(X + (X - x_b)^{n_X}) for X >= x_b, x_b = ln(r_break - R0).
bool hyper_on(const oracle_params& p) { return p.coords == 0 && p.n_x >= 2 && p.r_break > p.R0; }

void radial_map(const oracle_params& p, double X, double& r, double& d1, double& d2) {
  double E = X, E1 = 1.0, E2 = 0.0;  // exponent and its first two derivatives
  if (hyper_on(p)) {
    double xb = std::log(p.r_break - p.R0);
    if (X >= xb) {
      double y = X - xb;
      E = X + std::pow(y, p.n_x);
      E1 = 1.0 + p.n_x * std::pow(y, p.n_x - 1);
      E2 = p.n_x * (p.n_x - 1) * std::pow(y, p.n_x - 2);
    }
  }
  double e = std::exp(E);
  r = p.R0 + e;
  d1 = e * E1;                 // dr/dX
  d2 = e * (E1 * E1 + E2);     // d2r/dX2
}

// X at which the map reaches the radius r (inverse of radial_map; bisection on the monotone exponent)
double radial_inverse(const oracle_params& p, double r) {
  double target = std::log(r - p.R0);
  if (!hyper_on(p)) return target;
  double xb = std::log(p.r_break - p.R0);
  if (target <= xb) return target;
  double lo = xb, hi = target;   // X + (X-xb)^n >= X, so the solution lies in [xb, target]
  for (int it = 0; it < 200; it++) {
    double mid = 0.5 * (lo + hi);
    double E = mid + std::pow(mid - xb, p.n_x);
    if (E < target) lo = mid; else hi = mid;
  }
  return 0.5 * (lo + hi);
}

Coord coord_map(const oracle_params& p, double X1, double X2) {
  Coord c;
  if (p.coords == 1) {  // Minkowski: unused
    c.r = 1.0; c.th = 0.5 * PI; c.drdX = 1.0; c.dthdY = 1.0; c.d2thdY2 = 0.0; c.d2rdX2 = 0.0;
    return c;
  }
  radial_map(p, X1, c.r, c.drdX, c.d2rdX2);
  double arg = PI * (1.0 + X2);
  c.th = 0.5 * PI * (1.0 + X2) + 0.5 * (1.0 - p.hslope) * std::sin(arg);
  c.dthdY = 0.5 * PI * (1.0 + (1.0 - p.hslope) * std::cos(arg));
  c.d2thdY2 = -0.5 * PI * PI * (1.0 - p.hslope) * std::sin(arg);
  return c;
}

struct Geom {
  double gcov[4][4], gcon[4][4], sqrtg, alpha;
};

// ------------------------------------------------------------------------------------------
// C-2  Metric (eq. 38), MKS components by the diagonal Jacobian J=(1,r',th',1).
// Inverse from the KS closed form; sqrt(-g) = Sigma |sin th| |r'| |th'|.
// polar_face != 0: A32 — the 2-face lies exactly on the axis: sqrt(-g) := 0; sin^2 floored.
// ------------------------------------------------------------------------------------------
void ks_cov(double a, double r, double th, double g[4][4]) {
  double s = std::sin(th), c = std::cos(th);
  double s2 = s * s;
  double Sig = r * r + a * a * c * c;  // the paper's rho^2
  double f = 2.0 * r / Sig;
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) g[m][n] = 0.0;
  g[0][0] = -1.0 + f;
  g[0][1] = g[1][0] = f;
  g[0][3] = g[3][0] = -a * s2 * f;
  g[1][1] = 1.0 + f;
  g[1][3] = g[3][1] = -a * s2 * (1.0 + f);
  g[2][2] = Sig;
  g[3][3] = s2 * (Sig + a * a * s2 * (1.0 + f));
}

void metric_at(const oracle_params& p, double X1, double X2, int polar_face, Geom& G) {
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) { G.gcov[m][n] = 0.0; G.gcon[m][n] = 0.0; }
  if (p.coords == 1) {
    G.gcov[0][0] = -1.0; G.gcon[0][0] = -1.0;
    for (int i = 1; i < 4; i++) { G.gcov[i][i] = 1.0; G.gcon[i][i] = 1.0; }
    G.sqrtg = 1.0; G.alpha = 1.0;
    return;
  }
  Coord c = coord_map(p, X1, X2);
  double a = p.a;
  double gks[4][4];
  ks_cov(a, c.r, c.th, gks);
  double J[4] = {1.0, c.drdX, c.dthdY, 1.0};
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) G.gcov[m][n] = J[m] * J[n] * gks[m][n];
  double s = std::sin(c.th), co = std::cos(c.th);
  double s2 = s * s;
  if (s2 < 1e-30) s2 = 1e-30;  // A32
  double Sig = c.r * c.r + a * a * co * co;
  double f = 2.0 * c.r / Sig;
  double Del = c.r * c.r - 2.0 * c.r + a * a;
  double ik[4][4];
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) ik[m][n] = 0.0;
  ik[0][0] = -(1.0 + f);
  ik[0][1] = ik[1][0] = f;
  ik[1][1] = Del / Sig;
  ik[1][3] = ik[3][1] = a / Sig;
  ik[2][2] = 1.0 / Sig;
  ik[3][3] = 1.0 / (Sig * s2);
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) G.gcon[m][n] = ik[m][n] / (J[m] * J[n]);
  G.sqrtg = Sig * std::fabs(s) * std::fabs(c.drdX) * std::fabs(c.dthdY);
  if (polar_face) G.sqrtg = 0.0;  // A32: every 2-flux through the axis is exactly zero
  G.alpha = 1.0 / std::sqrt(-G.gcon[0][0]);
}

// ------------------------------------------------------------------------------------------
// Connection coefficients (A19: closed-form derivatives of eq. 38 pushed through the
// Jacobian).  conn[l][n][k] = Gamma^l_{n k} = 1/2 g^{l s} (d_n g_{s k} + d_k g_{s n} - d_s g_{n k}).
// ------------------------------------------------------------------------------------------
void conn_at(const oracle_params& p, double X1, double X2, double conn[4][4][4]) {
  for (int l = 0; l < 4; l++) for (int n = 0; n < 4; n++) for (int k = 0; k < 4; k++) conn[l][n][k] = 0.0;
  if (p.coords == 1) return;
  Coord c = coord_map(p, X1, X2);
  double a = p.a, r = c.r, th = c.th;
  double s = std::sin(th), co = std::cos(th);
  double s2 = s * s;
  double Sig = r * r + a * a * co * co;
  double f = 2.0 * r / Sig;
  // derivatives of Sigma and f = 2r/Sigma
  double dSig_r = 2.0 * r, dSig_t = -2.0 * a * a * s * co;
  double df_r = 2.0 / Sig - 2.0 * r * dSig_r / (Sig * Sig);
  double df_t = -2.0 * r * dSig_t / (Sig * Sig);
  double ds2_t = 2.0 * s * co;
  // KS metric and its r- and theta-derivatives
  double g[4][4], dgr[4][4], dgt[4][4];
  ks_cov(a, r, th, g);
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) { dgr[m][n] = 0.0; dgt[m][n] = 0.0; }
  dgr[0][0] = df_r;                      dgt[0][0] = df_t;
  dgr[0][1] = dgr[1][0] = df_r;          dgt[0][1] = dgt[1][0] = df_t;
  dgr[0][3] = dgr[3][0] = -a * s2 * df_r;
  dgt[0][3] = dgt[3][0] = -a * (ds2_t * f + s2 * df_t);
  dgr[1][1] = df_r;                      dgt[1][1] = df_t;
  dgr[1][3] = dgr[3][1] = -a * s2 * df_r;
  dgt[1][3] = dgt[3][1] = -a * (ds2_t * (1.0 + f) + s2 * df_t);
  dgr[2][2] = dSig_r;                    dgt[2][2] = dSig_t;
  // g_phiphi = s2 * (Sig + a^2 s2 (1+f))
  dgr[3][3] = s2 * (dSig_r + a * a * s2 * df_r);
  dgt[3][3] = ds2_t * (Sig + a * a * s2 * (1.0 + f)) + s2 * (dSig_t + a * a * (ds2_t * (1.0 + f) + s2 * df_t));
  // MKS: gM_{mn} = J_m J_n g_{mn};  dJ_1/dX = r'',  dJ_2/dY = th''
  double J[4] = {1.0, c.drdX, c.dthdY, 1.0};
  double dJ1[4] = {0.0, c.d2rdX2, 0.0, 0.0};   // d J_m / dX  (= r' on the plain exponential branch)
  double dJ2[4] = {0.0, 0.0, c.d2thdY2, 0.0};  // d J_m / dY
  double dg[4][4][4];                          // dg[s][k][n] = d_n gM_{s k}
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) {
    dg[m][n][0] = 0.0;
    dg[m][n][3] = 0.0;
    dg[m][n][1] = (dJ1[m] * J[n] + J[m] * dJ1[n]) * g[m][n] + J[m] * J[n] * dgr[m][n] * c.drdX;
    dg[m][n][2] = (dJ2[m] * J[n] + J[m] * dJ2[n]) * g[m][n] + J[m] * J[n] * dgt[m][n] * c.dthdY;
  }
  Geom G;
  metric_at(p, X1, X2, 0, G);
  for (int l = 0; l < 4; l++)
    for (int n = 0; n < 4; n++)
      for (int k = 0; k < 4; k++) {
        double sum = 0.0;
        for (int sg = 0; sg < 4; sg++) sum += G.gcon[l][sg] * (dg[sg][k][n] + dg[sg][n][k] - dg[n][k][sg]);
        conn[l][n][k] = 0.5 * sum;
      }
}

// ------------------------------------------------------------------------------------------
// C-3  Primitive -> fluid state at one metric location (eq. 10).
// prim = (rho, u, ut1, ut2, ut3, B1, B2, B3).
// ------------------------------------------------------------------------------------------
struct State {
  double ucon[4], ucov[4], bcon[4], bcov[4], bsq, lorentz;
};

void fluid_state(const double prim[8], const Geom& G, State& S) {
  double qsq = 0.0;
  for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) qsq += G.gcov[i][j] * prim[1 + i] * prim[1 + j];
  double lor = std::sqrt(1.0 + qsq);
  S.lorentz = lor;
  double alpha = G.alpha;
  S.ucon[0] = lor / alpha;
  for (int i = 1; i < 4; i++) {
    double beta_i = G.gcon[0][i] * alpha * alpha;
    S.ucon[i] = prim[1 + i] - lor * beta_i / alpha;  // eq. 10
  }
  for (int m = 0; m < 4; m++) {
    double v = 0.0;
    for (int n = 0; n < 4; n++) v += G.gcov[m][n] * S.ucon[n];
    S.ucov[m] = v;
  }
  double bt = 0.0;
  for (int i = 1; i < 4; i++) bt += prim[4 + i] * S.ucov[i];  // b^t = B^i u^mu g_{i mu}
  S.bcon[0] = bt;
  for (int i = 1; i < 4; i++) S.bcon[i] = (prim[4 + i] + bt * S.ucon[i]) / S.ucon[0];
  for (int m = 0; m < 4; m++) {
    double v = 0.0;
    for (int n = 0; n < 4; n++) v += G.gcov[m][n] * S.bcon[n];
    S.bcov[m] = v;
  }
  double b2 = 0.0;
  for (int m = 0; m < 4; m++) b2 += S.bcon[m] * S.bcov[m];
  S.bsq = b2;
}

// mixed stress tensor T^m_n (eq. 5 with one index lowered)
void stress_mixed(const double prim[8], const State& S, double gam, double T[4][4]) {
  double rho = prim[0], u = prim[1];
  double p = (gam - 1.0) * u;
  double w = rho + u + p;
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < 4; n++) {
      double delta = (m == n) ? 1.0 : 0.0;
      T[m][n] = (w + S.bsq) * S.ucon[m] * S.ucov[n] + (p + 0.5 * S.bsq) * delta - S.bcon[m] * S.bcov[n];
    }
}

// ------------------------------------------------------------------------------------------
// C-4  Conserved variables (dir = 0) and fluxes (dir = 1,2,3)  (eqs. 6-8, P:L78-88;
// A1: induction flux sqrt(-g)(b^i u^d - b^d u^i); A18: energy variable is sqrt(-g) T^t_t).
// ------------------------------------------------------------------------------------------
void flux_vector(const double prim[8], const State& S, const Geom& G, double gam, int dir, double out[8]) {
  double T[4][4];
  stress_mixed(prim, S, gam, T);
  out[0] = G.sqrtg * prim[0] * S.ucon[dir];
  for (int n = 0; n < 4; n++) out[1 + n] = G.sqrtg * T[dir][n];
  for (int i = 1; i < 4; i++) out[4 + i] = G.sqrtg * (S.bcon[i] * S.ucon[dir] - S.bcon[dir] * S.ucon[i]);
}

// ------------------------------------------------------------------------------------------
// C-6  Wave speeds from the quadratic dispersion relation (eqs. 18-19).
// Roots of A v^2 + B v + C = 0, c1 >= c2.  A29: negative discriminant clamped to 0.
// ------------------------------------------------------------------------------------------
void wave_speeds(const double prim[8], const State& S, const Geom& G, double gam, int dir, double* c1, double* c2) {
  double rho = prim[0], u = prim[1];
  double p = (gam - 1.0) * u;
  double w = rho + u + p;
  double cs2 = gam * p / w;               // eq. 19
  double va2 = S.bsq / (S.bsq + w);
  double cms2 = va2 + cs2 * (1.0 - va2);  // eq. 18
  double ut = S.ucon[0], ud = S.ucon[dir];
  double A = ut * ut - cms2 * (G.gcon[0][0] + ut * ut);
  double B = -2.0 * (ut * ud - cms2 * (G.gcon[0][dir] + ut * ud));
  double C = ud * ud - cms2 * (G.gcon[dir][dir] + ud * ud);
  double disc = B * B - 4.0 * A * C;
  if (disc < 0.0) disc = 0.0;
  double sq = std::sqrt(disc);
  double ra = (-B + sq) / (2.0 * A);
  double rb = (-B - sq) / (2.0 * A);
  *c1 = (ra > rb) ? ra : rb;
  *c2 = (ra > rb) ? rb : ra;
}

// ------------------------------------------------------------------------------------------
// C-5  Reconstruction.  MC-limited slope (eq. 15; A2: signed last branch).
// ------------------------------------------------------------------------------------------
double slope_mc(double qm, double q0, double qp) {
  double dm = q0 - qm, dp = qp - q0;
  if (dm * dp < 0.0) return 0.0;
  double dc = 0.5 * (qp - qm);
  if (std::fabs(dm) < std::fabs(dp) && 2.0 * std::fabs(dm) < std::fabs(dc)) return 2.0 * dm;
  if (2.0 * std::fabs(dp) < std::fabs(dc)) return 2.0 * dp;
  return dc;
}

// Values of one variable at the lower (l) and upper (r) faces of the cell y[2], seen from inside
// that cell, from the 5 cell values y[0..4] centred on it.
// recon 0: PLM, eq. 16.  recon 1: PPM, A20 = basic Colella-Woodward (1984):
// MC-limited slopes, 4th-order interface values, monotonisation; no steepening / flattening.
void recon_cell(int recon, const double y[5], double* l, double* r) {
  if (recon == 0) {
    double dq = slope_mc(y[1], y[2], y[3]);
    *l = y[2] - 0.5 * dq;
    *r = y[2] + 0.5 * dq;
    return;
  }
  double dm = slope_mc(y[0], y[1], y[2]);
  double d0 = slope_mc(y[1], y[2], y[3]);
  double dp = slope_mc(y[2], y[3], y[4]);
  double ql = 0.5 * (y[1] + y[2]) - (d0 - dm) / 6.0;
  double qr = 0.5 * (y[2] + y[3]) - (dp - d0) / 6.0;
  double yc = y[2];
  if ((qr - yc) * (yc - ql) <= 0.0) {
    ql = yc; qr = yc;
  } else {
    double d = qr - ql;
    double m6 = d * (yc - 0.5 * (ql + qr));
    double lim = d * d / 6.0;
    if (m6 > lim) ql = 3.0 * yc - 2.0 * qr;
    else if (m6 < -lim) qr = 3.0 * yc - 2.0 * ql;
  }
  *l = ql; *r = qr;
}

// ------------------------------------------------------------------------------------------
// C-6  Riemann flux at one face from the two reconstructed states and the FACE metric
// (P:L139-161).  LLF eq. 17; HLL eq. 20 (A30: denominator guarded).
// ------------------------------------------------------------------------------------------
// entropy density S = p_g / rho^(gam-1), the quantity advected by eq. 11
double entropy_of(double rho, double u, double gam) { return (gam - 1.0) * u / std::pow(rho, gam - 1.0); }

// FS_out (may be null): the same Riemann flux for the entropy equation (eq. 11): conserved sqrt(-g) S u^t, flux
// sqrt(-g) S u^d, from the same two states and the same wave speeds.
void face_flux(const double pl[8], const double pr[8], const Geom& G, double gam, int dir, int riemann,
               double Fbar[8], double* cw_out, double* FS_out = nullptr) {
  State Sl, Sr;
  fluid_state(pl, G, Sl);
  fluid_state(pr, G, Sr);
  double Ul[8], Ur[8], Fl[8], Fr[8];
  flux_vector(pl, Sl, G, gam, 0, Ul);
  flux_vector(pr, Sr, G, gam, 0, Ur);
  flux_vector(pl, Sl, G, gam, dir, Fl);
  flux_vector(pr, Sr, G, gam, dir, Fr);
  double c1l, c2l, c1r, c2r;
  wave_speeds(pl, Sl, G, gam, dir, &c1l, &c2l);
  wave_speeds(pr, Sr, G, gam, dir, &c1r, &c2r);
  double cmax = std::max(0.0, std::max(c1r, c1l));
  double cmin = std::max(0.0, std::max(-c2r, -c2l));
  double cw = std::max(cmax, cmin);
  *cw_out = cw;
  for (int v = 0; v < 8; v++) {
    if (riemann == 0) {
      Fbar[v] = 0.5 * (Fl[v] + Fr[v] - cw * (Ur[v] - Ul[v]));  // eq. 17
    } else {
      double den = std::max(cmax + cmin, 1e-300);
      Fbar[v] = (cmax * Fl[v] + cmin * Fr[v] - cmax * cmin * (Ur[v] - Ul[v])) / den;  // eq. 20
    }
  }
  if (FS_out) {
    double sl = entropy_of(pl[0], pl[1], gam), sr = entropy_of(pr[0], pr[1], gam);
    double ul = G.sqrtg * sl * Sl.ucon[0], ur = G.sqrtg * sr * Sr.ucon[0];
    double fl = G.sqrtg * sl * Sl.ucon[dir], fr = G.sqrtg * sr * Sr.ucon[dir];
    if (riemann == 0) {
      *FS_out = 0.5 * (fl + fr - cw * (ur - ul));
    } else {
      double den = std::max(cmax + cmin, 1e-300);
      *FS_out = (cmax * fl + cmin * fr - cmax * cmin * (ur - ul)) / den;
    }
  }
}

// ------------------------------------------------------------------------------------------
// C-8  Source S_nu = sqrt(-g) T^k_l Gamma^l_{nu k} at the centre (eq. 7, eq. 14).
// ------------------------------------------------------------------------------------------
void source_term(const double prim[8], const Geom& G, const double conn[4][4][4], double gam, double S[4]) {
  State st;
  fluid_state(prim, G, st);
  double T[4][4];
  stress_mixed(prim, st, gam, T);
  for (int nu = 0; nu < 4; nu++) {
    double sum = 0.0;
    for (int k = 0; k < 4; k++) for (int l = 0; l < 4; l++) sum += T[k][l] * conn[l][nu][k];
    S[nu] = G.sqrtg * sum;
  }
}

// ------------------------------------------------------------------------------------------
// C-10  Noble 2D inversion (eqs. 27-31; A6 sign of eq. 30; A7 D = alpha rho u^t;
// A8 Newton policy).  Returns 0 = ok or a failure code; on failure the fluid primitives are the
// guess.  B^i = U_B / sqrt(-g) always.
//   1: D <= 0 or non-finite input   2: no convergence in maxit   3: W <= 0 or non-finite
//   4: v^2 outside [0,1)            5: rho <= 0                  6: u < 0
// ------------------------------------------------------------------------------------------
int invert_2d(const double U[8], const Geom& G, double gam, double prim[8], double tol, int maxit, int extra,
              int* iters_out) {
  double guess[8];
  for (int v = 0; v < 8; v++) guess[v] = prim[v];
  *iters_out = 0;
  double alpha = G.alpha, sg = G.sqrtg;
  for (int i = 1; i < 4; i++) prim[4 + i] = U[4 + i] / sg;
  double D = alpha * U[0] / sg;
  double Qcov[4], Bc[4];
  for (int m = 0; m < 4; m++) Qcov[m] = alpha * U[1 + m] / sg;
  Bc[0] = 0.0;
  for (int i = 1; i < 4; i++) Bc[i] = alpha * U[4 + i] / sg;
  bool finite_in = std::isfinite(D);
  for (int m = 0; m < 4; m++) finite_in = finite_in && std::isfinite(Qcov[m]) && std::isfinite(Bc[m]);
  if (!finite_in || !(D > 0.0)) return 1;
  double Qcon[4];
  for (int m = 0; m < 4; m++) {
    double v = 0.0;
    for (int n = 0; n < 4; n++) v += G.gcon[m][n] * Qcov[n];
    Qcon[m] = v;
  }
  double Bsq = 0.0;
  for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) Bsq += G.gcov[i][j] * Bc[i] * Bc[j];
  double QdotB = 0.0;
  for (int i = 1; i < 4; i++) QdotB += Qcov[i] * Bc[i];
  double ncon[4];
  ncon[0] = 1.0 / alpha;
  for (int i = 1; i < 4; i++) ncon[i] = -alpha * G.gcon[0][i];
  double Qdotn = 0.0;
  for (int m = 0; m < 4; m++) Qdotn += Qcov[m] * ncon[m];
  double Qsq = 0.0;
  for (int m = 0; m < 4; m++) Qsq += Qcon[m] * Qcov[m];
  double Qtsq = Qsq + Qdotn * Qdotn;
  double QdB2 = QdotB * QdotB;
  double gfac = (gam - 1.0) / gam;
  // initial guess (A8, A35)
  double qsq = 0.0;
  for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) qsq += G.gcov[i][j] * guess[1 + i] * guess[1 + j];
  double W = (1.0 + qsq) * (guess[0] + gam * guess[1]);
  double v2 = 0.0;
  for (int tries = 0; tries < 400; tries++) {
    v2 = (Qtsq + QdB2 * (Bsq + 2.0 * W) / (W * W)) / ((Bsq + W) * (Bsq + W));
    if (v2 < 1.0) break;
    W *= 10.0;
  }
  if (!(v2 < 1.0) || !(W > 0.0)) return 3;
  if (v2 < 0.0) v2 = 0.0;
  bool converged = false;
  int extra_left = -1;
  int it = 0;
  for (it = 1; it <= maxit; it++) {
    double W2 = W * W, W3 = W2 * W;
    double omv = 1.0 - v2;
    double sq = std::sqrt(omv);
    double pg = gfac * (W * omv - D * sq);  // eq. 31
    double f1 = Qtsq - v2 * (Bsq + W) * (Bsq + W) + QdB2 * (Bsq + 2.0 * W) / W2;  // eq. 29
    double f2 = -Qdotn - 0.5 * Bsq * (1.0 + v2) + QdB2 / (2.0 * W2) - W + pg;      // eq. 30 (A6)
    double j11 = -2.0 * (Bsq + W) * (v2 + QdB2 / W3);
    double j12 = -(Bsq + W) * (Bsq + W);
    double j21 = -1.0 - QdB2 / W3 + gfac * omv;
    double j22 = -0.5 * Bsq + gfac * (-W + D / (2.0 * sq));
    double det = j11 * j22 - j12 * j21;
    double dW = (-f1 * j22 + f2 * j12) / det;
    double dv = (-f2 * j11 + f1 * j21) / det;
    double Wn = std::fabs(W + dW);
    double vn = v2 + dv;
    if (vn < 0.0) vn = 0.0;
    if (vn > 1.0 - 1e-15) vn = 1.0 - 1e-15;
    double err = (Wn == 0.0) ? std::fabs(dW) : std::fabs(dW / Wn);
    W = Wn; v2 = vn;
    if (!std::isfinite(W) || !std::isfinite(v2)) { *iters_out = it; return 3; }
    if (extra_left < 0) {
      if (err <= tol) { extra_left = extra; }
    } else {
      extra_left--;
    }
    if (extra_left == 0) { converged = true; break; }
  }
  *iters_out = (it > maxit) ? maxit : it;
  if (!converged) return 2;
  if (!(W > 0.0)) return 3;
  if (!(v2 >= 0.0 && v2 < 1.0)) return 4;
  double lor = 1.0 / std::sqrt(1.0 - v2);
  double rho = D / lor;
  double w = W * (1.0 - v2);
  double u = (w - rho) / gam;
  if (!(rho > 0.0)) return 5;
  if (!(u >= 0.0)) return 6;
  prim[0] = rho;
  prim[1] = u;
  for (int i = 1; i < 4; i++) {
    double Qt = Qcon[i] + ncon[i] * Qdotn;
    prim[1 + i] = lor * (Qt + QdotB * Bc[i] / W) / (W + Bsq);
  }
  return 0;
}

// ------------------------------------------------------------------------------------------
// the fallback inversions of P:L229-239.  Common set-up: the Noble variables of eqs. 27-28.
// ------------------------------------------------------------------------------------------
struct Noble {
  double D, Qtsq, Bsq, QdB, Qdn, Qcon[4], ncon[4], Bc[4];
  double Qt[4];   // Qtilde^i, i = 1..3
  bool finite;
};

// energy_free: Qtilde^2 and Qtilde^i from the momentum components alone, through the spatial inverse metric
// gamma^{ij} = g^{ij} - g^{ti} g^{tj} / g^{tt}: "(Qtilde)^2 is independent on Qtilde^0, and therefore computing its value
// does not require the use of the energy conservation equation" -- the form the entropy method needs, since
// it is called exactly when the energy variable cannot be trusted.  Otherwise the 4-vector forms of invert_2d.
void noble_vars(const double U[8], const Geom& G, Noble& N, bool energy_free = false) {
  double alpha = G.alpha, sg = G.sqrtg;
  N.D = alpha * U[0] / sg;
  double Qcov[4];
  for (int m = 0; m < 4; m++) Qcov[m] = alpha * U[1 + m] / sg;
  N.Bc[0] = 0.0;
  for (int i = 1; i < 4; i++) N.Bc[i] = alpha * U[4 + i] / sg;
  N.finite = std::isfinite(N.D);
  for (int m = 0; m < 4; m++) N.finite = N.finite && std::isfinite(Qcov[m]) && std::isfinite(N.Bc[m]);
  for (int m = 0; m < 4; m++) {
    double v = 0.0;
    for (int n = 0; n < 4; n++) v += G.gcon[m][n] * Qcov[n];
    N.Qcon[m] = v;
  }
  N.Bsq = 0.0;
  for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) N.Bsq += G.gcov[i][j] * N.Bc[i] * N.Bc[j];
  N.QdB = 0.0;
  for (int i = 1; i < 4; i++) N.QdB += Qcov[i] * N.Bc[i];
  N.ncon[0] = 1.0 / alpha;
  for (int i = 1; i < 4; i++) N.ncon[i] = -alpha * G.gcon[0][i];
  N.Qdn = 0.0;
  for (int m = 0; m < 4; m++) N.Qdn += Qcov[m] * N.ncon[m];
  double Qsq = 0.0;
  for (int m = 0; m < 4; m++) Qsq += N.Qcon[m] * Qcov[m];
  N.Qtsq = Qsq + N.Qdn * N.Qdn;
  for (int i = 1; i < 4; i++) N.Qt[i] = N.Qcon[i] + N.ncon[i] * N.Qdn;
  if (energy_free) {
    N.finite = std::isfinite(N.D);
    for (int i = 1; i < 4; i++) N.finite = N.finite && std::isfinite(Qcov[i]) && std::isfinite(N.Bc[i]);
    N.Qtsq = 0.0;
    for (int i = 1; i < 4; i++) {
      double v = 0.0;
      for (int j = 1; j < 4; j++) v += (G.gcon[i][j] - G.gcon[0][i] * G.gcon[0][j] / G.gcon[0][0]) * Qcov[j];
      N.Qt[i] = v;
      N.Qtsq += v * Qcov[i];
    }
  }
}

// residual of eq. 29 at (W, v^2)
double eq29(const Noble& N, double W, double v2) {
  return N.Qtsq - v2 * (N.Bsq + W) * (N.Bsq + W) + N.QdB * N.QdB * (N.Bsq + 2.0 * W) / (W * W);
}

// Brent's method (Brent 1973, "zeroin") for f on [a, b] with f(a) f(b) <= 0.  Stops when the bracket is shorter
// than |b| (4 eps + tol) or f(b) = 0.  A40: the paper names the method only; the relative tolerance
// is a parameter, 1e-14 in the workloads -- far below the 1e-10 the paper quotes for Newton, so that two
// implementations land on the same root to round-off whatever path their bisection / interpolation choices take.
template <class F>
bool brent(F f, double a, double b, double fa, double fb, double tol, int maxit, double* root) {
  if (!(fa * fb <= 0.0)) return false;
  double c = a, fc = fa, d = b - a, e = d;
  for (int it = 0; it < maxit; it++) {
    if ((fb > 0.0 && fc > 0.0) || (fb < 0.0 && fc < 0.0)) { c = a; fc = fa; d = b - a; e = d; }
    if (std::fabs(fc) < std::fabs(fb)) { a = b; b = c; c = a; fa = fb; fb = fc; fc = fa; }
    double tol1 = std::fabs(b) * (2.0 * 2.220446049250313e-16 + 0.5 * tol);
    double xm = 0.5 * (c - b);
    if (std::fabs(xm) <= tol1 || fb == 0.0) { *root = b; return true; }
    if (std::fabs(e) >= tol1 && std::fabs(fa) > std::fabs(fb)) {
      double sfrac = fb / fa, p, q;
      if (a == c) {
        p = 2.0 * xm * sfrac;
        q = 1.0 - sfrac;
      } else {
        double qq = fa / fc, r = fb / fc;
        p = sfrac * (2.0 * xm * qq * (qq - r) - (b - a) * (r - 1.0));
        q = (qq - 1.0) * (r - 1.0) * (sfrac - 1.0);
      }
      if (p > 0.0) q = -q;
      p = std::fabs(p);
      double min1 = 3.0 * xm * q - std::fabs(tol1 * q), min2 = std::fabs(e * q);
      if (2.0 * p < (min1 < min2 ? min1 : min2)) { e = d; d = p / q; }
      else { d = xm; e = d; }
    } else {
      d = xm; e = d;
    }
    a = b; fa = fb;
    if (std::fabs(d) > tol1) b += d;
    else b += (xm >= 0.0 ? tol1 : -tol1);
    fb = f(b);
    if (!std::isfinite(fb)) return false;
  }
  return false;
}

// recover rho, u, utilde^i from (W, v^2) as in the 2D method; returns a failure code of invert_2d
int recover_prims(const Noble& N, double gam, double W, double v2, double u_given, bool use_u_given, double prim[8]) {
  if (!(W > 0.0) || !std::isfinite(W)) return 3;
  if (!(v2 >= 0.0 && v2 < 1.0)) return 4;
  double lor = 1.0 / std::sqrt(1.0 - v2);
  double rho = N.D / lor;
  double w = W * (1.0 - v2);
  double u = use_u_given ? u_given : (w - rho) / gam;
  if (!(rho > 0.0)) return 5;
  if (!(u >= 0.0)) return 6;
  prim[0] = rho;
  prim[1] = u;
  for (int i = 1; i < 4; i++) prim[1 + i] = lor * (N.Qt[i] + N.QdB * N.Bc[i] / W) / (W + N.Bsq);
  return 0;
}

// (ii) the 1D method: "analytically expressing v^2 from Equation (30), use its expression in Equation
// (29) which is then numerically solved using the Brent method".  With s = sqrt(1 - v^2) and eq. 31, eq. 30 (A6 sign)
// is the quadratic  (B^2/2 + g W) s^2 - g D s + [-Q.n - B^2 + (Q.B)^2/(2 W^2) - W] = 0,  g = (gam-1)/gam,
// whose constant term is negative wherever a physical state exists, so the root with the plus sign is the positive
// one.  The quadratic has real roots only above some W_d (its discriminant turns negative below), the eq. 29
// residual r(W) is negative in a thin band above W_d, crosses zero at the physical root and stays positive beyond
// (v^2 of eq. 30 decreases, eventually below zero).  A41 (bracket; the paper is silent): from W0 = Gamma^2 w of the
// guess, double W until r is defined and positive (upper end); halve W from there until r is negative or undefined
// (lower end); Brent then runs on r extended below W_d by the constant -r(upper end), so that the bracket always
// carries a sign change and the root, if one exists, is the only sign change of a continuous stretch.
// Returns 0 or a failure code (2: no bracket / no convergence / root at the edge of validity; 3..6 as invert_2d).
// "parity unpinned": A41.
bool v2_from_eq30(const Noble& N, double gam, double W, double* v2) {
  double g = (gam - 1.0) / gam;
  double qa = 0.5 * N.Bsq + g * W;
  double qb = -g * N.D;
  double qc = -N.Qdn - N.Bsq + N.QdB * N.QdB / (2.0 * W * W) - W;
  double disc = qb * qb - 4.0 * qa * qc;
  if (!(disc >= 0.0) || !(qa > 0.0)) return false;
  double sroot = (-qb + std::sqrt(disc)) / (2.0 * qa);
  *v2 = 1.0 - sroot * sroot;
  return std::isfinite(*v2);
}

int invert_1dw(const double U[8], const Geom& G, double gam, double prim[8], double tol, int maxit) {
  double guess[8];
  for (int v = 0; v < 8; v++) guess[v] = prim[v];
  for (int i = 1; i < 4; i++) prim[4 + i] = U[4 + i] / G.sqrtg;
  Noble N;
  noble_vars(U, G, N);
  if (!N.finite || !(N.D > 0.0)) return 1;
  double qsq = 0.0;
  for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) qsq += G.gcov[i][j] * guess[1 + i] * guess[1 + j];
  double W0 = (1.0 + qsq) * (guess[0] + gam * guess[1]);
  if (!(W0 > 0.0) || !std::isfinite(W0)) return 3;
  auto resid = [&](double W) {
    double v2;
    if (!v2_from_eq30(N, gam, W, &v2)) return std::nan("");
    return eq29(N, W, v2);
  };
  // bracket search (A41)
  double wb = W0, fb = resid(wb);
  for (int k = 0; k < 60 && !(std::isfinite(fb) && fb > 0.0); k++) { wb *= 2.0; fb = resid(wb); }
  if (!(std::isfinite(fb) && fb > 0.0)) return 2;
  const double below = -fb;
  auto rext = [&](double W) { double r = resid(W); return std::isfinite(r) ? r : below; };
  double wa = 0.5 * wb, fa = rext(wa);
  for (int k = 0; k < 60 && fa > 0.0; k++) { wa *= 0.5; fa = rext(wa); }
  if (fa > 0.0) return 2;
  double W;
  if (!brent(rext, wa, wb, fa, fb, tol, maxit, &W)) return 2;
  double v2;
  if (!v2_from_eq30(N, gam, W, &v2)) return 2;
  return recover_prims(N, gam, W, v2, 0.0, false, prim);
}

// (iii) the entropy method (eq. 32): W(v^2) = Gamma D + Gamma gam/(gam-1) (D/Gamma)^(gam-1) calS put
// into eq. 29, solved for v^2 in [0, 1) by Brent.  A36: eq. 32 holds as printed when its S is the CONSERVED
// entropy calS = Gamma S = alpha U_S / sqrt(-g) (as D = Gamma rho), S = p_g / rho^(gam-1).
// The residual is >= 0 at v^2 = 0 and -> -infinity as v^2 -> 1, so [0, 1 - 1e-15] always brackets a root.
// Returns 0 or: 1 (D <= 0, calS <= 0 or non-finite input), 2 (Brent failed), 3..6 as invert_2d.
int invert_entropy(const double U[8], double US, const Geom& G, double gam, double prim[8], double tol, int maxit) {
  for (int i = 1; i < 4; i++) prim[4 + i] = U[4 + i] / G.sqrtg;
  Noble N;
  noble_vars(U, G, N, true);
  double calS = G.alpha * US / G.sqrtg;
  if (!N.finite || !std::isfinite(calS) || !(N.D > 0.0) || !(calS > 0.0)) return 1;
  auto Wof = [&](double v2) {
    double lor = 1.0 / std::sqrt(1.0 - v2);
    return lor * N.D + lor * (gam / (gam - 1.0)) * std::pow(N.D / lor, gam - 1.0) * calS;  // eq. 32
  };
  auto resid = [&](double v2) { return eq29(N, Wof(v2), v2); };
  double a = 0.0, b = 1.0 - 1e-15;
  double fa = resid(a), fb = resid(b);
  if (!std::isfinite(fa) || !std::isfinite(fb)) return 2;
  double v2;
  if (fa == 0.0) v2 = 0.0;
  else if (!brent(resid, a, b, fa, fb, tol, maxit, &v2)) return 2;
  double lor = 1.0 / std::sqrt(1.0 - v2);
  double rho = N.D / lor;
  double pg = (calS / lor) * std::pow(rho, gam - 1.0);   // S rho^(gam-1), S = calS / Gamma
  return recover_prims(N, gam, Wof(v2), v2, pg / (gam - 1.0), true, prim);
}

// ------------------------------------------------------------------------------------------
// C-12  Floors (eqs. 35-37; A9-A12).  "parity unpinned" for the ceiling mechanism
// (A11) — the paper gives no formula; post-conditions and idempotence are pinned.
// Returns a bit mask: 1 rho floor, 2 u floor, 4 ceiling applied, 8 Lorentz cap, 16 ceiling
// re-inversion failed (additive fallback used).
// ------------------------------------------------------------------------------------------
int apply_floors(const oracle_params& p, double r, const Geom& G, double prim[8]) {
  int mask = 0;
  double rfl = std::max(p.rho_fl_abs, p.rho_fl_coef * std::pow(r, p.rho_fl_pow));
  double ufl = std::max(p.u_fl_abs, p.u_fl_coef * std::pow(r, p.u_fl_pow));
  if (prim[0] < rfl) { prim[0] = rfl; mask |= 1; }
  if (prim[1] < ufl) { prim[1] = ufl; mask |= 2; }
  if (p.sigma_max > 0.0 || p.b2_over_u_max > 0.0) {
    State S;
    fluid_state(prim, G, S);
    double drho = 0.0, du = 0.0;
    if (p.sigma_max > 0.0) drho = std::max(0.0, S.bsq / p.sigma_max - prim[0]);
    if (p.b2_over_u_max > 0.0) du = std::max(0.0, S.bsq / p.b2_over_u_max - prim[1]);
    if (drho > 0.0 || du > 0.0) {
      mask |= 4;
      double U[8], Uadd[8];
      flux_vector(prim, S, G, p.gam, 0, U);
      double padd[8] = {drho, du, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};  // at rest in the normal-observer frame
      State Sa;
      fluid_state(padd, G, Sa);
      flux_vector(padd, Sa, G, p.gam, 0, Uadd);
      for (int v = 0; v < 8; v++) U[v] += Uadd[v];
      double trial[8];
      for (int v = 0; v < 8; v++) trial[v] = prim[v];
      int iters;
      int flag = invert_2d(U, G, p.gam, trial, p.newton_tol, p.newton_maxit, p.newton_extra, &iters);
      if (flag == 0) {
        for (int v = 0; v < 5; v++) prim[v] = trial[v];
      } else {
        prim[0] += drho; prim[1] += du; mask |= 16;
      }
      // the injection slows the fluid, which raises b^2 a little: enforce eqs. 36-37 exactly with a final
      // clamp at fixed velocity (b^2 does not depend on rho, u at fixed utilde^i, B^i)
      State S2;
      fluid_state(prim, G, S2);
      if (p.sigma_max > 0.0) prim[0] = std::max(prim[0], S2.bsq / p.sigma_max);
      if (p.b2_over_u_max > 0.0) prim[1] = std::max(prim[1], S2.bsq / p.b2_over_u_max);
    }
  }
  if (p.gamma_max > 0.0) {
    double qsq = 0.0;
    for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) qsq += G.gcov[i][j] * prim[1 + i] * prim[1 + j];
    double lor = std::sqrt(1.0 + qsq);
    if (lor > p.gamma_max) {
      double fac = std::sqrt((p.gamma_max * p.gamma_max - 1.0) / (lor * lor - 1.0));  // A12
      for (int i = 1; i < 4; i++) prim[1 + i] *= fac;
      mask |= 8;
    }
  }
  return mask;
}

// ------------------------------------------------------------------------------------------
// Grid context
// ------------------------------------------------------------------------------------------
struct Ctx {
  oracle_params p;
  int n1g, n2g, n3g, ng;
  size_t nz;  // zones per variable, extended grid
  double dx[3], x0[3];
  std::vector<Geom> gc, gf1, gf2;   // centre, 1-face (i-1/2,j), 2-face (i,j-1/2); index i*n2g+j
  std::vector<double> conn;         // [i*n2g+j][4][4][4]
  std::vector<double> rc;           // r at centre
  double* prim;                     // bound, caller-owned
  std::vector<double> F[3], E[3], Phalf, Pnew, cw[3];
  std::vector<double> FS[3];        // entropy fluxes of eq. 11 (filled only when the fallback chain is on)
  std::vector<int32_t> flag;
  int64_t stats[8];
  int64_t chain[4];                 // 0 zones sent down the chain, 1 recovered by 1D-W, 2 by the entropy method, 3 entropy-first zones (eq. 33)
  double cwmax[3];

  size_t idx(int i, int j, int k) const { return ((size_t)i * n2g + j) * n3g + k; }
  size_t vidx(int v, int i, int j, int k) const { return (size_t)v * nz + idx(i, j, k); }
};

void get_prim(const Ctx& c, const double* P, int i, int j, int k, double out[8]) {
  for (int v = 0; v < 8; v++) out[v] = P[c.vidx(v, i, j, k)];
}

const Geom& geom_face(const Ctx& c, int dir, int i, int j) {
  if (dir == 1) return c.gf1[(size_t)i * c.n2g + j];
  if (dir == 2) return c.gf2[(size_t)i * c.n2g + j];
  return c.gc[(size_t)i * c.n2g + j];  // the metric is phi-independent: 3-faces == centres
}

void build_geometry(Ctx& c) {
  const oracle_params& p = c.p;
  size_t n = (size_t)c.n1g * c.n2g;
  c.gc.resize(n); c.gf1.resize(n); c.gf2.resize(n);
  c.conn.assign(n * 64, 0.0);
  c.rc.assign(n, 1.0);
  for (int i = 0; i < c.n1g; i++)
    for (int j = 0; j < c.n2g; j++) {
      int I = i - c.ng + (p.n1_global > 0 ? p.i_offset : 0), J = j - c.ng;   // global zone index in X1
      double X1c = c.x0[0] + (I + 0.5) * c.dx[0], X2c = c.x0[1] + (J + 0.5) * c.dx[1];
      double X1f = c.x0[0] + I * c.dx[0], X2f = c.x0[1] + J * c.dx[1];
      size_t q = (size_t)i * c.n2g + j;
      metric_at(p, X1c, X2c, 0, c.gc[q]);
      metric_at(p, X1f, X2c, 0, c.gf1[q]);
      int polar = (p.coords == 0 && p.bc_x2 == 2 && (J == 0 || J == p.n2)) ? 1 : 0;
      metric_at(p, X1c, X2f, polar, c.gf2[q]);
      double cn[4][4][4];
      conn_at(p, X1c, X2c, cn);
      std::memcpy(&c.conn[q * 64], cn, sizeof(cn));
      c.rc[q] = coord_map(p, X1c, X2c).r;
    }
}

// ------------------------------------------------------------------------------------------
// C-13  Boundary conditions (A15 outflow + inflow check; "parity unpinned" for the
// inflow check and the sqrt(-g) B rescale, which the paper does not spell out).
// Order: X1, then X2, then X3, each over the full extended range of the other two.
// ------------------------------------------------------------------------------------------
void inflow_check(const Ctx& c, double prim[8], const Geom& G, int inner) {
  State S;
  fluid_state(prim, G, S);
  bool bad = inner ? (S.ucon[1] > 0.0) : (S.ucon[1] < 0.0);
  if (!bad) return;
  double lor = S.lorentz;
  double alpha = G.alpha;
  double vt[4];
  for (int i = 1; i < 4; i++) vt[i] = prim[1 + i] / lor;
  vt[1] = (G.gcon[0][1] * alpha * alpha) / alpha;  // beta^1 / alpha  => u^1 = 0
  double vsq = 0.0;
  for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) vsq += G.gcov[i][j] * vt[i] * vt[j];
  double gmax = (c.p.gamma_max > 0.0) ? c.p.gamma_max : 50.0;
  double vmax = 1.0 - 1.0 / (gmax * gmax);
  if (vsq > vmax) vsq = vmax;
  double ln = 1.0 / std::sqrt(1.0 - vsq);
  for (int i = 1; i < 4; i++) prim[1 + i] = ln * vt[i];
}

void apply_bc(const Ctx& c, double* P) {
  const int ng = c.ng, n1 = c.p.n1, n2 = c.p.n2, n3 = c.p.n3;
  // X1
  if (c.p.bc_x1 != 3) {
    for (int g = 0; g < ng; g++)
      for (int side = 0; side < 2; side++) {
        if (c.p.n1_global > 0 && (side ? c.p.slab_hi : c.p.slab_lo)) continue;  // internal side: the halo exchange fills it
        int ig = side ? (ng + n1 + g) : (ng - 1 - g);
        int is;
        if (c.p.bc_x1 == 1) is = side ? (ng + g) : (ng + n1 - 1 - g);
        else is = side ? (ng + n1 - 1) : ng;  // outflow: adjacent interior zone
        for (int j = 0; j < c.n2g; j++)
          for (int k = 0; k < c.n3g; k++) {
            double q[8];
            get_prim(c, P, is, j, k, q);
            if (c.p.bc_x1 == 0) {
              const Geom& Gs = c.gc[(size_t)is * c.n2g + j];
              const Geom& Gg = c.gc[(size_t)ig * c.n2g + j];
              double ratio = Gs.sqrtg / Gg.sqrtg;
              for (int b = 5; b < 8; b++) q[b] *= ratio;
              if (c.p.coords == 0) inflow_check(c, q, Gg, side == 0);
            }
            for (int v = 0; v < 8; v++) P[c.vidx(v, ig, j, k)] = q[v];
          }
      }
  }
  // X2
  if (c.p.bc_x2 != 3) {
    for (int g = 0; g < ng; g++)
      for (int side = 0; side < 2; side++) {
        int jg = side ? (ng + n2 + g) : (ng - 1 - g);
        int js;
        if (c.p.bc_x2 == 1) js = side ? (ng + g) : (ng + n2 - 1 - g);
        else if (c.p.bc_x2 == 2) js = side ? (ng + n2 - 1 - g) : (ng + g);  // mirror
        else js = side ? (ng + n2 - 1) : ng;
        for (int i = 0; i < c.n1g; i++)
          for (int k = 0; k < c.n3g; k++) {
            double q[8];
            get_prim(c, P, i, js, k, q);
            if (c.p.bc_x2 == 2) { q[3] = -q[3]; q[6] = -q[6]; }  // u^2 -> -u^2, B^2 -> -B^2
            if (c.p.bc_x2 == 0) {
              double ratio = c.gc[(size_t)i * c.n2g + js].sqrtg / c.gc[(size_t)i * c.n2g + jg].sqrtg;
              for (int b = 5; b < 8; b++) q[b] *= ratio;
            }
            for (int v = 0; v < 8; v++) P[c.vidx(v, i, jg, k)] = q[v];
          }
      }
  }
  // X3
  if (c.p.bc_x3 != 3) {
    for (int g = 0; g < ng; g++)
      for (int side = 0; side < 2; side++) {
        int kg = side ? (ng + n3 + g) : (ng - 1 - g);
        int ks;
        if (c.p.bc_x3 == 1) {
          // periodic; for n3 < ng wrap repeatedly
          int K = side ? (n3 + g) : (-1 - g);
          int Kw = ((K % n3) + n3) % n3;
          ks = ng + Kw;
        } else {
          ks = side ? (ng + n3 - 1) : ng;
        }
        for (int i = 0; i < c.n1g; i++)
          for (int j = 0; j < c.n2g; j++)
            for (int v = 0; v < 8; v++) P[c.vidx(v, i, j, kg)] = P[c.vidx(v, i, j, ks)];
      }
  }
}

// ------------------------------------------------------------------------------------------
// Face fluxes in one direction over the range the flux-CT average needs (C-6):
// d-face index 0..N_d, transverse zones -1..N.  F[v] stored at the index of the zone whose
// LOWER d-face it is.  cw stored likewise (0 elsewhere).
// ------------------------------------------------------------------------------------------
void flux_dir(Ctx& c, const double* P, int dir, std::vector<double>& F, std::vector<double>& CW, double* cwmax,
              std::vector<double>* FS = nullptr) {
  const int ng = c.ng;
  int n[3] = {c.p.n1, c.p.n2, c.p.n3};
  int lo[3], hi[3];
  for (int d = 0; d < 3; d++) {
    if (d == dir - 1) { lo[d] = ng; hi[d] = ng + n[d]; }
    else { lo[d] = ng - 1; hi[d] = ng + n[d]; }
  }
  int e[3] = {0, 0, 0};
  e[dir - 1] = 1;
  F.assign(8 * c.nz, 0.0);
  CW.assign(c.nz, 0.0);
  if (FS) FS->assign(c.nz, 0.0);
  double cmax_all = 0.0;
#pragma omp parallel for reduction(max : cmax_all) schedule(static)
  for (int i = lo[0]; i <= hi[0]; i++)
    for (int j = lo[1]; j <= hi[1]; j++)
      for (int k = lo[2]; k <= hi[2]; k++) {
        // cell "m" = (i,j,k)-e is on the left of the face, cell "p" = (i,j,k) on the right
        double pl[8], pr[8];
        for (int v = 0; v < 8; v++) {
          double ym[5], yp[5];
          for (int s = 0; s < 5; s++) {
            int o = s - 2;
            ym[s] = P[c.vidx(v, i - e[0] + o * e[0], j - e[1] + o * e[1], k - e[2] + o * e[2])];
            yp[s] = P[c.vidx(v, i + o * e[0], j + o * e[1], k + o * e[2])];
          }
          double l, r;
          recon_cell(c.p.recon, ym, &l, &r);
          pl[v] = r;  // q^l at the face = upper-face value of the left cell
          recon_cell(c.p.recon, yp, &l, &r);
          pr[v] = l;  // q^r at the face = lower-face value of the right cell
        }
        const Geom& G = geom_face(c, dir, i, j);
        double Fb[8], cw, fs = 0.0;
        face_flux(pl, pr, G, c.p.gam, dir, c.p.riemann, Fb, &cw, FS ? &fs : nullptr);
        if (FS) (*FS)[c.idx(i, j, k)] = fs;
        for (int v = 0; v < 8; v++) F[c.vidx(v, i, j, k)] = Fb[v];
        CW[c.idx(i, j, k)] = cw;
        if (cw > cmax_all) cmax_all = cw;
      }
  *cwmax = cmax_all;
}

// ------------------------------------------------------------------------------------------
// C-7  Flux-CT (eqs. 21-22; A3: the two edges bounding the face).
// E^1_{i,j,k} lives on the edge (I, J-1/2, K-1/2), E^2 on (I-1/2, J, K-1/2), E^3 on (I-1/2, J-1/2, K).
// ------------------------------------------------------------------------------------------
void flux_ct(Ctx& c) {
  const int ng = c.ng, n1 = c.p.n1, n2 = c.p.n2, n3 = c.p.n3;
  std::vector<double>&F1 = c.F[0], &F2 = c.F[1], &F3 = c.F[2];
  for (int d = 0; d < 3; d++) c.E[d].assign(c.nz, 0.0);
  const int B1 = 5, B2 = 6, B3 = 7;
#pragma omp parallel for schedule(static)
  for (int i = ng; i <= ng + n1; i++)
    for (int j = ng; j <= ng + n2; j++)
      for (int k = ng; k <= ng + n3; k++) {
        c.E[0][c.idx(i, j, k)] = 0.25 * (F2[c.vidx(B3, i, j, k)] + F2[c.vidx(B3, i, j, k - 1)] -
                                         F3[c.vidx(B2, i, j, k)] - F3[c.vidx(B2, i, j - 1, k)]);
        c.E[1][c.idx(i, j, k)] = 0.25 * (F3[c.vidx(B1, i, j, k)] + F3[c.vidx(B1, i - 1, j, k)] -
                                         F1[c.vidx(B3, i, j, k)] - F1[c.vidx(B3, i, j, k - 1)]);
        c.E[2][c.idx(i, j, k)] = 0.25 * (F1[c.vidx(B2, i, j, k)] + F1[c.vidx(B2, i, j - 1, k)] -
                                         F2[c.vidx(B1, i, j, k)] - F2[c.vidx(B1, i - 1, j, k)]);
      }
  const std::vector<double>&E1 = c.E[0], &E2 = c.E[1], &E3 = c.E[2];
#pragma omp parallel for schedule(static)
  for (int i = ng; i <= ng + n1; i++)
    for (int j = ng; j <= ng + n2; j++)
      for (int k = ng; k <= ng + n3; k++) {
        bool in1 = i < ng + n1, in2 = j < ng + n2, in3 = k < ng + n3;
        if (in2 && in3) {  // 1-face (I-1/2, J, K)
          F1[c.vidx(B1, i, j, k)] = 0.0;
          F1[c.vidx(B2, i, j, k)] = 0.5 * (E3[c.idx(i, j, k)] + E3[c.idx(i, j + 1, k)]);
          F1[c.vidx(B3, i, j, k)] = -0.5 * (E2[c.idx(i, j, k)] + E2[c.idx(i, j, k + 1)]);
        }
        if (in1 && in3) {  // 2-face (I, J-1/2, K)
          F2[c.vidx(B2, i, j, k)] = 0.0;
          F2[c.vidx(B3, i, j, k)] = 0.5 * (E1[c.idx(i, j, k)] + E1[c.idx(i, j, k + 1)]);
          F2[c.vidx(B1, i, j, k)] = -0.5 * (E3[c.idx(i, j, k)] + E3[c.idx(i + 1, j, k)]);
        }
        if (in1 && in2) {  // 3-face (I, J, K-1/2)
          F3[c.vidx(B3, i, j, k)] = 0.0;
          F3[c.vidx(B1, i, j, k)] = 0.5 * (E2[c.idx(i, j, k)] + E2[c.idx(i + 1, j, k)]);
          F3[c.vidx(B2, i, j, k)] = -0.5 * (E1[c.idx(i, j, k)] + E1[c.idx(i, j + 1, k)]);
        }
      }
}

// ------------------------------------------------------------------------------------------
// C-11  Fix-up of failed zones (eq. 34; A13 deterministic Jacobi passes).
// "parity unpinned": stencil choice / pass order are DESIGN.md conventions.
// ------------------------------------------------------------------------------------------
// One Jacobi pass over the zones flagged in `fl` (> 0 or any non-zero: failed); donors are read from a snapshot of P
// taken at the start of the pass and must be good at the start of the pass; zones repaired in this pass are cleared in
// `fl` at its end.  Returns the number of zones left waiting.
int64_t fixup_pass(Ctx& c, double* P, std::vector<int32_t>& fl, int pass) {
  const int ng = c.ng, n1 = c.p.n1, n2 = c.p.n2, n3 = c.p.n3;
  const int fo[4][2] = {{1, 0}, {-1, 0}, {0, 1}, {0, -1}};
  const int dg[4][2] = {{1, 1}, {1, -1}, {-1, 1}, {-1, -1}};
  bool last = (pass == c.p.fixup_max_passes);
  std::vector<int32_t> flnew(fl);
  std::vector<double> snap(P, P + 5 * c.nz);
  int64_t left = 0;
  for (int i = ng; i < ng + n1; i++)
    for (int j = ng; j < ng + n2; j++)
      for (int k = ng; k < ng + n3; k++) {
        size_t q = c.idx(i, j, k);
        if (!fl[q]) continue;
        bool facegood = true, diaggood = true;
        for (int m = 0; m < 4; m++) {
          if (fl[c.idx(i + fo[m][0], j + fo[m][1], k)]) facegood = false;
          if (fl[c.idx(i + dg[m][0], j + dg[m][1], k)]) diaggood = false;
        }
        const int(*st)[2] = nullptr;
        if (facegood) st = fo; else if (diaggood) st = dg;
        if (st) {
          for (int v = 0; v < 5; v++) {
            double sum = 0.0;
            for (int m = 0; m < 4; m++) sum += snap[c.vidx(v, i + st[m][0], j + st[m][1], k)];
            P[c.vidx(v, i, j, k)] = 0.25 * sum;
          }
        } else if (last) {
          int cnt = 0;
          double sum[5] = {0, 0, 0, 0, 0};
          for (int di = -1; di <= 1; di++)
            for (int dj = -1; dj <= 1; dj++) {
              if (!di && !dj) continue;
              if (fl[c.idx(i + di, j + dj, k)]) continue;
              cnt++;
              for (int v = 0; v < 5; v++) sum[v] += snap[c.vidx(v, i + di, j + dj, k)];
            }
          if (cnt > 0) for (int v = 0; v < 5; v++) P[c.vidx(v, i, j, k)] = sum[v] / cnt;
          c.stats[7]++;
        } else {
          left++;
          continue;
        }
        flnew[q] = 0;
        c.stats[1]++;
        // floors on the repaired zone (A34)
        double q8[8];
        get_prim(c, P, i, j, k, q8);
        size_t g2 = (size_t)i * c.n2g + j;
        apply_floors(c.p, c.rc[g2], c.gc[g2], q8);
        for (int v = 0; v < 5; v++) P[c.vidx(v, i, j, k)] = q8[v];
      }
  fl.swap(flnew);
  return left;
}

int64_t interior_failed(const Ctx& c) {
  int64_t n = 0;
  for (int i = c.ng; i < c.ng + c.p.n1; i++)
    for (int j = c.ng; j < c.ng + c.p.n2; j++)
      for (int k = c.ng; k < c.ng + c.p.n3; k++) if (c.flag[c.idx(i, j, k)]) n++;
  return n;
}

void fixup(Ctx& c, double* P) {
  int64_t nbad = interior_failed(c);
  c.stats[0] += nbad;
  if (!nbad) return;
  std::vector<int32_t> fl(c.flag);
  for (int pass = 0; pass <= c.p.fixup_max_passes; pass++)
    if (!fixup_pass(c, P, fl, pass)) break;
}

// ------------------------------------------------------------------------------------------
// SURVEY 8(f)3, second half -- "to increase the numerical stability in the polar region, the polar component of the
// 4-velocity in the two cells closest to the pole is modified, by an interpolation to zero at the pole".
// A16 (the paper gives no formula): in the two zones nearest each pole, J = 0, 1 and J = N2-1, N2-2, the primitive
// utilde^2 is replaced by the straight line in X^2 through zero at the pole (X^2 = -1 or +1) and the value of the
// third zone (J = 2 or N2-3) of the same (I, K).  Applied to the result of inversion + floors of every substep, before
// the ghost fill (whose reflection continues the same line across the pole); only with the polar reflection in X^2
// and at least 6 zones.  "parity unpinned" for the choice of variable and anchor zone; the linearity is pinned.
// ------------------------------------------------------------------------------------------
void polar_damp(Ctx& c, double* P) {
  const int ng = c.ng, n1 = c.p.n1, n2 = c.p.n2, n3 = c.p.n3;
  if (c.p.bc_x2 != 2 || n2 < 6) return;
  auto X2 = [&](int J) { return c.x0[1] + (J + 0.5) * c.dx[1]; };   // centre of zone J (interior numbering)
  const double north = c.x0[1], south = c.x0[1] + n2 * c.dx[1];
  for (int i = ng; i < ng + n1; i++)
    for (int k = ng; k < ng + n3; k++)
      for (int m = 0; m < 2; m++) {
        double a = P[c.vidx(3, i, ng + 2, k)];
        P[c.vidx(3, i, ng + m, k)] = a * (X2(m) - north) / (X2(2) - north);
        double b = P[c.vidx(3, i, ng + n2 - 3, k)];
        P[c.vidx(3, i, ng + n2 - 1 - m, k)] = b * (south - X2(n2 - 1 - m)) / (south - X2(n2 - 3));
      }
}

// ------------------------------------------------------------------------------------------
// C-9  One RK2 substep (eq. 25; A5 source added; A34 order; A35 guess).
// ------------------------------------------------------------------------------------------
void substep(Ctx& c, const double* Pflux, const double* Pbase, double dtau, double* Pout, bool record_cw, bool with_repair = true) {
  double cwm[3];
  const bool chain = c.p.inv_chain != 0;
  for (int d = 1; d <= 3; d++) flux_dir(c, Pflux, d, c.F[d - 1], c.cw[d - 1], &cwm[d - 1], chain ? &c.FS[d - 1] : nullptr);
  if (record_cw) for (int d = 0; d < 3; d++) c.cwmax[d] = cwm[d];
  flux_ct(c);
  const int ng = c.ng, n1 = c.p.n1, n2 = c.p.n2, n3 = c.p.n3;
  std::memcpy(Pout, Pbase, 8 * c.nz * sizeof(double));
  for (int i = ng; i < ng + n1; i++)   // (flags outside the interior are never set by this loop: with slabs they hold
    for (int j = ng; j < ng + n2; j++)  //  the neighbour's flags, refreshed by the halo exchange)
      for (int k = ng; k < ng + n3; k++) c.flag[c.idx(i, j, k)] = 0;
  int64_t nfl_rho = 0, nfl_u = 0, nceil = 0, ncap = 0, nits = 0;
  int64_t nchain = 0, n1dw = 0, nent = 0, nbeta = 0;
#pragma omp parallel for reduction(+ : nfl_rho, nfl_u, nceil, ncap, nits, nchain, n1dw, nent, nbeta) schedule(static)
  for (int i = ng; i < ng + n1; i++)
    for (int j = ng; j < ng + n2; j++)
      for (int k = ng; k < ng + n3; k++) {
        size_t g2 = (size_t)i * c.n2g + j;
        const Geom& G = c.gc[g2];
        double pb[8], pf[8];
        get_prim(c, Pbase, i, j, k, pb);
        get_prim(c, Pflux, i, j, k, pf);
        State Sb;
        fluid_state(pb, G, Sb);
        double U[8];
        flux_vector(pb, Sb, G, c.p.gam, 0, U);
        double S[4];
        const double(*cn)[4][4] = reinterpret_cast<const double(*)[4][4]>(&c.conn[g2 * 64]);
        source_term(pf, G, cn, c.p.gam, S);
        for (int v = 0; v < 8; v++) {
          double div = (c.F[0][c.vidx(v, i + 1, j, k)] - c.F[0][c.vidx(v, i, j, k)]) / c.dx[0] +
                       (c.F[1][c.vidx(v, i, j + 1, k)] - c.F[1][c.vidx(v, i, j, k)]) / c.dx[1] +
                       (c.F[2][c.vidx(v, i, j, k + 1)] - c.F[2][c.vidx(v, i, j, k)]) / c.dx[2];
          double src = (v >= 1 && v <= 4) ? S[v - 1] : 0.0;
          U[v] = U[v] + dtau * (-div + src);
        }
        double pn[8];
        for (int v = 0; v < 8; v++) pn[v] = pb[v];  // A35
        int iters = 0;
        int flag;
        if (!chain) {
          flag = invert_2d(U, G, c.p.gam, pn, c.p.newton_tol, c.p.newton_maxit, c.p.newton_extra, &iters);
        } else {
          // the chain of P:L233-239.  The entropy equation (eq. 11) is advanced like the others:
          // U_S* = sqrt(-g) S u^t (P^n) - dtau div F_S, no source.
          double US = G.sqrtg * entropy_of(pb[0], pb[1], c.p.gam) * Sb.ucon[0];
          double divS = (c.FS[0][c.idx(i + 1, j, k)] - c.FS[0][c.idx(i, j, k)]) / c.dx[0] +
                        (c.FS[1][c.idx(i, j + 1, k)] - c.FS[1][c.idx(i, j, k)]) / c.dx[1] +
                        (c.FS[2][c.idx(i, j, k + 1)] - c.FS[2][c.idx(i, j, k)]) / c.dx[2];
          US = US + dtau * (-divS);
          // eq. 33 (A37): beta = p_g / (p_g + b^2/2) of the primitives at the previous time step
          double pg = (c.p.gam - 1.0) * pb[1];
          bool beta_small = c.p.beta_min > 0.0 && pg / (pg + 0.5 * Sb.bsq) < c.p.beta_min;
          if (beta_small) {
            nbeta++;
            flag = invert_entropy(U, US, G, c.p.gam, pn, c.p.brent_tol, c.p.brent_maxit);   // first and only choice
            if (flag == 0) nent++;
          } else {
            flag = invert_2d(U, G, c.p.gam, pn, c.p.newton_tol, c.p.newton_maxit, c.p.newton_extra, &iters);
            if (flag != 0 && flag != 1) {      // 1: D <= 0 or non-finite input: no method applies
              nchain++;
              int f2 = flag;
              if (flag == 2 || flag == 3) {    // "fails to produce results" -> 1D-W by Brent
                for (int v = 0; v < 8; v++) pn[v] = pb[v];
                f2 = invert_1dw(U, G, c.p.gam, pn, c.p.brent_tol, c.p.brent_maxit);
                if (f2 == 0) n1dw++;
              }
              if (f2 != 0) {                   // non-physical values, or 1D-W failed too -> the entropy fix
                for (int v = 0; v < 8; v++) pn[v] = pb[v];
                f2 = invert_entropy(U, US, G, c.p.gam, pn, c.p.brent_tol, c.p.brent_maxit);
                if (f2 == 0) nent++;
              }
              if (f2 != 0) { for (int v = 0; v < 5; v++) pn[v] = pb[v]; }   // still failed: the guess stays, eq. 34 repairs
              flag = f2;
            }
          }
        }
        nits += iters;
        if (flag == 0) {
          int m = apply_floors(c.p, c.rc[g2], G, pn);
          nfl_rho += (m & 1) ? 1 : 0; nfl_u += (m & 2) ? 1 : 0; nceil += (m & 4) ? 1 : 0; ncap += (m & 8) ? 1 : 0;
        }
        c.flag[c.idx(i, j, k)] = flag;
        for (int v = 0; v < 8; v++) Pout[c.vidx(v, i, j, k)] = pn[v];
      }
  c.stats[2] += nfl_rho; c.stats[3] += nfl_u; c.stats[4] += nceil; c.stats[5] += ncap; c.stats[6] += nits;
  c.chain[0] += nchain; c.chain[1] += n1dw; c.chain[2] += nent; c.chain[3] += nbeta;
  if (c.p.polar_damp) polar_damp(c, Pout);   // P:L311; A16
  // A34: ghosts are refreshed before the repair (so that ghost donors belong to the same state) and after it
  apply_bc(c, Pout);
  if (!with_repair) return;
  fixup(c, Pout);
  apply_bc(c, Pout);
}

}  // namespace

// ==========================================================================================
// C interface (host pointers everywhere).
// ==========================================================================================
extern "C" {

typedef struct OracleCtx* oracle_handle;
struct OracleCtx { Ctx c; };

void oracle_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

int oracle_get_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// ---- point-level entry points (for the pins) ----
void oracle_radial_map(const oracle_params* p, double X1, double out[4]) {   // r, r', r'', and X of r_out
  radial_map(*p, X1, out[0], out[1], out[2]);
  out[3] = radial_inverse(*p, p->r_out);
}

void oracle_coord_map(const oracle_params* p, double X1, double X2, double out[5]) {
  Coord c = coord_map(*p, X1, X2);
  out[0] = c.r; out[1] = c.th; out[2] = c.drdX; out[3] = c.dthdY; out[4] = c.d2thdY2;
}

void oracle_metric_at(const oracle_params* p, double X1, double X2, int polar_face, double gcov[16], double gcon[16],
                      double* sqrtg, double* alpha) {
  Geom G;
  metric_at(*p, X1, X2, polar_face, G);
  std::memcpy(gcov, G.gcov, sizeof(G.gcov));
  std::memcpy(gcon, G.gcon, sizeof(G.gcon));
  *sqrtg = G.sqrtg; *alpha = G.alpha;
}

void oracle_conn_at(const oracle_params* p, double X1, double X2, double conn[64]) {
  double cn[4][4][4];
  conn_at(*p, X1, X2, cn);
  std::memcpy(conn, cn, sizeof(cn));
}

static void geom_from_arrays(const double gcov[16], const double gcon[16], double sqrtg, Geom& G) {
  std::memcpy(G.gcov, gcov, sizeof(G.gcov));
  std::memcpy(G.gcon, gcon, sizeof(G.gcon));
  G.sqrtg = sqrtg;
  G.alpha = 1.0 / std::sqrt(-G.gcon[0][0]);
}

void oracle_fluid_state(const double prim[8], const double gcov[16], const double gcon[16], double ucon[4],
                        double ucov[4], double bcon[4], double bcov[4], double* bsq) {
  Geom G; geom_from_arrays(gcov, gcon, 1.0, G);
  State S; fluid_state(prim, G, S);
  for (int m = 0; m < 4; m++) { ucon[m] = S.ucon[m]; ucov[m] = S.ucov[m]; bcon[m] = S.bcon[m]; bcov[m] = S.bcov[m]; }
  *bsq = S.bsq;
}

void oracle_flux_vector(const double prim[8], const double gcov[16], const double gcon[16], double sqrtg, double gam,
                        int dir, double out[8]) {
  Geom G; geom_from_arrays(gcov, gcon, sqrtg, G);
  State S; fluid_state(prim, G, S);
  flux_vector(prim, S, G, gam, dir, out);
}

void oracle_wave_speeds(const double prim[8], const double gcov[16], const double gcon[16], double gam, int dir,
                        double* c1, double* c2) {
  Geom G; geom_from_arrays(gcov, gcon, 1.0, G);
  State S; fluid_state(prim, G, S);
  wave_speeds(prim, S, G, gam, dir, c1, c2);
}

double oracle_slope_mc(double qm, double q0, double qp) { return slope_mc(qm, q0, qp); }

void oracle_recon_cell(int recon, const double y[5], double* l, double* r) { recon_cell(recon, y, l, r); }

void oracle_face_flux(const double pl[8], const double pr[8], const double gcov[16], const double gcon[16],
                      double sqrtg, double gam, int dir, int riemann, double Fbar[8], double* cw) {
  Geom G; geom_from_arrays(gcov, gcon, sqrtg, G);
  face_flux(pl, pr, G, gam, dir, riemann, Fbar, cw);
}

void oracle_source_term(const double prim[8], const double gcov[16], const double gcon[16], double sqrtg,
                        const double conn[64], double gam, double S[4]) {
  Geom G; geom_from_arrays(gcov, gcon, sqrtg, G);
  source_term(prim, G, reinterpret_cast<const double(*)[4][4]>(conn), gam, S);
}

int oracle_invert_2d(const double U[8], const double gcov[16], const double gcon[16], double sqrtg, double gam,
                     double prim_inout[8], double tol, int maxit, int extra, int* iters) {
  Geom G; geom_from_arrays(gcov, gcon, sqrtg, G);
  return invert_2d(U, G, gam, prim_inout, tol, maxit, extra, iters);
}

int oracle_apply_floors(const oracle_params* p, double r, const double gcov[16], const double gcon[16], double sqrtg,
                        double prim_inout[8]) {
  Geom G; geom_from_arrays(gcov, gcon, sqrtg, G);
  return apply_floors(*p, r, G, prim_inout);
}

// ---- grid-level entry points (mirror the library's calls, host pointers) ----
int oracle_grid_init(oracle_handle* out, const oracle_params* p) {
  if (!out || !p) return -1;
  if (p->struct_bytes != (int32_t)sizeof(oracle_params)) return -1;
  if (p->n1 < 1 || p->n2 < 1 || p->n3 < 1 || p->ng < 3) return -1;
  OracleCtx* h = new OracleCtx();
  Ctx& c = h->c;
  c.p = *p;
  c.ng = p->ng;
  c.n1g = p->n1 + 2 * p->ng; c.n2g = p->n2 + 2 * p->ng; c.n3g = p->n3 + 2 * p->ng;
  c.nz = (size_t)c.n1g * c.n2g * c.n3g;
  if (p->coords == 0) {
    c.x0[0] = std::log(p->r_in - p->R0);
    c.dx[0] = (radial_inverse(*p, p->r_out) - c.x0[0]) / (p->n1_global > 0 ? p->n1_global : p->n1);   // uniform in X up to the X of r_out
    c.x0[1] = -1.0; c.dx[1] = 2.0 / p->n2;
    c.x0[2] = 0.0;  c.dx[2] = 2.0 * PI / p->n3;
  } else {
    int n[3] = {p->n1_global > 0 ? p->n1_global : p->n1, p->n2, p->n3};
    for (int d = 0; d < 3; d++) { c.x0[d] = p->xmin[d]; c.dx[d] = (p->xmax[d] - p->xmin[d]) / n[d]; }
  }
  build_geometry(c);
  c.prim = nullptr;
  c.flag.assign(c.nz, 0);
  c.Phalf.assign(8 * c.nz, 0.0);
  c.Pnew.assign(8 * c.nz, 0.0);
  for (int s = 0; s < 8; s++) c.stats[s] = 0;
  for (int s = 0; s < 4; s++) c.chain[s] = 0;
  for (int d = 0; d < 3; d++) c.cwmax[d] = 0.0;
  *out = h;
  return 0;
}

int oracle_destroy(oracle_handle h) { delete h; return 0; }

// loc 0 centre, 1 = 1-face, 2 = 2-face: 22 comps (gcov 00 01 02 03 11 12 13 22 23 33, gcon same, sqrtg, alpha)
// loc 3: 40 comps Gamma^l_{nk}, l-major, (n,k) in the same 10-pair order.  out[comp][n1g][n2g].
int oracle_get_geom(oracle_handle h, int loc, double* out) {
  Ctx& c = h->c;
  static const int pm[10] = {0, 0, 0, 0, 1, 1, 1, 2, 2, 3}, pn[10] = {0, 1, 2, 3, 1, 2, 3, 2, 3, 3};
  size_t n = (size_t)c.n1g * c.n2g;
  if (loc >= 0 && loc <= 2) {
    const std::vector<Geom>& g = (loc == 0) ? c.gc : (loc == 1) ? c.gf1 : c.gf2;
    for (size_t q = 0; q < n; q++) {
      for (int s = 0; s < 10; s++) { out[s * n + q] = g[q].gcov[pm[s]][pn[s]]; out[(10 + s) * n + q] = g[q].gcon[pm[s]][pn[s]]; }
      out[20 * n + q] = g[q].sqrtg;
      out[21 * n + q] = g[q].alpha;
    }
    return 0;
  }
  if (loc == 3) {
    for (size_t q = 0; q < n; q++)
      for (int l = 0; l < 4; l++)
        for (int s = 0; s < 10; s++) out[(size_t)(l * 10 + s) * n + q] = c.conn[q * 64 + l * 16 + pm[s] * 4 + pn[s]];
    return 0;
  }
  return -1;
}

int oracle_bind(oracle_handle h, double* prim) {
  h->c.prim = prim;
  apply_bc(h->c, prim);
  return 0;
}

int oracle_apply_bc(oracle_handle h, double* prim) { apply_bc(h->c, prim); return 0; }

// stage-level: the polar-velocity interpolation of P:L311 (A16) on a caller-provided primitive array, in place
int oracle_polar_damp(oracle_handle h, double* prim) { polar_damp(h->c, prim); return 0; }

// one full RK2 step in place (eq. 25)
int oracle_step(oracle_handle h, double dt) {
  Ctx& c = h->c;
  if (!c.prim) return -2;
  substep(c, c.prim, c.prim, 0.5 * dt, c.Phalf.data(), true);
  substep(c, c.Phalf.data(), c.prim, dt, c.Pnew.data(), false);
  std::memcpy(c.prim, c.Pnew.data(), 8 * c.nz * sizeof(double));
  return 0;
}

// Slab decomposition: the two substeps of eq. 25 as calls of their own, so that the caller can exchange
// the halo planes of the half-step array between them and of the primitive array after them.
//   which = 0: predictor, P^n -> the half-step array (oracle_half);  which = 1: corrector, in place into the bound array.
int oracle_substep(oracle_handle h, int which, double dt) {
  Ctx& c = h->c;
  if (!c.prim) return -2;
  if (which == 0) {
    substep(c, c.prim, c.prim, 0.5 * dt, c.Phalf.data(), true);
  } else {
    substep(c, c.Phalf.data(), c.prim, dt, c.Pnew.data(), false);
    std::memcpy(c.prim, c.Pnew.data(), 8 * c.nz * sizeof(double));
  }
  return 0;
}
// ... and the substep itself in pieces, for slabs whose failed zones may lie next to an internal boundary: the repair's
// Jacobi passes one by one, with a halo exchange of the array and of the flags (oracle_flags) between them.
int oracle_substep_update(oracle_handle h, int which, double dt) {
  Ctx& c = h->c;
  if (!c.prim) return -2;
  if (which == 0) substep(c, c.prim, c.prim, 0.5 * dt, c.Phalf.data(), true, false);
  else substep(c, c.Phalf.data(), c.prim, dt, c.Pnew.data(), false, false);
  return 0;
}
// out[0] = failed zones of this slab (interior) at the start of pass 0 (0 in later passes), out[1] = zones left waiting
int oracle_repair_pass(oracle_handle h, int which, int pass, int64_t out[2]) {
  Ctx& c = h->c;
  double* P = which == 0 ? c.Phalf.data() : c.Pnew.data();
  out[0] = 0;
  if (pass == 0) { out[0] = interior_failed(c); c.stats[0] += out[0]; }
  out[1] = fixup_pass(c, P, c.flag, pass);
  return 0;
}
int oracle_substep_finish(oracle_handle h, int which) {
  Ctx& c = h->c;
  apply_bc(c, which == 0 ? c.Phalf.data() : c.Pnew.data());
  return 0;
}
// the corrector works into a scratch array; this copies it over the bound primitives (end of the step)
int oracle_commit(oracle_handle h) { std::memcpy(h->c.prim, h->c.Pnew.data(), 8 * h->c.nz * sizeof(double)); return 0; }
double* oracle_new(oracle_handle h) { return h->c.Pnew.data(); }
int32_t* oracle_flags(oracle_handle h) { return h->c.flag.data(); }
double* oracle_half(oracle_handle h) { return h->c.Phalf.data(); }
// the three face-speed maxima the predictor of the last step saw, and eq. 26 from a given triple (after a max over slabs)
int oracle_last_cw(oracle_handle h, double cw[3]) { for (int d = 0; d < 3; d++) cw[d] = h->c.cwmax[d]; return 0; }
int oracle_dt_of_cw(oracle_handle h, double xi, const double cw[3], double* dt_out) {
  double inv = 0.0;
  for (int d = 0; d < 3; d++) inv += cw[d] / (xi * h->c.dx[d]);
  *dt_out = 1.0 / inv;
  return 0;
}
// face-speed maxima of the bound primitives (what oracle_cfl_dt reduces)
int oracle_cfl_cw(oracle_handle h, double cw[3]) {
  Ctx& c = h->c;
  if (!c.prim) return -2;
  for (int d = 1; d <= 3; d++) flux_dir(c, c.prim, d, c.F[d - 1], c.cw[d - 1], &cw[d - 1]);
  return 0;
}

// stage-level: fluxes of one direction from an arbitrary primitive array (before flux-CT)
int oracle_flux_dir(oracle_handle h, const double* prim, int dir, double* F_out, double* cw_out, double* cwmax) {
  Ctx& c = h->c;
  std::vector<double> F, CW;
  double m;
  flux_dir(c, prim, dir, F, CW, &m);
  if (F_out) std::memcpy(F_out, F.data(), 8 * c.nz * sizeof(double));
  if (cw_out) std::memcpy(cw_out, CW.data(), c.nz * sizeof(double));
  if (cwmax) *cwmax = m;
  return 0;
}

// stage-level: flux-CT on caller-provided flux arrays [8][nz] each (in place) -> EMFs [3][nz]
int oracle_flux_ct(oracle_handle h, double* F1, double* F2, double* F3, double* E_out) {
  Ctx& c = h->c;
  double* Fs[3] = {F1, F2, F3};
  for (int d = 0; d < 3; d++) c.F[d].assign(Fs[d], Fs[d] + 8 * c.nz);
  flux_ct(c);
  for (int d = 0; d < 3; d++) {
    std::memcpy(Fs[d], c.F[d].data(), 8 * c.nz * sizeof(double));
    if (E_out) std::memcpy(E_out + d * c.nz, c.E[d].data(), c.nz * sizeof(double));
  }
  return 0;
}

// stage-level: conserved update with caller-provided (already CT-replaced) fluxes; for the flux-CT pin
// "arbitrary fluxes leave eq. 23 unchanged" only the B components are updated here:
// prim B^i <- (sqrt(-g) B^i - dtau * div F(B^i)) / sqrt(-g)
int oracle_update_B_only(oracle_handle h, double* prim, const double* F1, const double* F2, const double* F3,
                         double dtau) {
  Ctx& c = h->c;
  const int ng = c.ng;
  const double* Fs[3] = {F1, F2, F3};
  std::vector<double> out(3 * c.nz);
  for (int i = ng; i < ng + c.p.n1; i++)
    for (int j = ng; j < ng + c.p.n2; j++)
      for (int k = ng; k < ng + c.p.n3; k++) {
        double sg = c.gc[(size_t)i * c.n2g + j].sqrtg;
        for (int v = 5; v < 8; v++) {
          double div = (Fs[0][c.vidx(v, i + 1, j, k)] - Fs[0][c.vidx(v, i, j, k)]) / c.dx[0] +
                       (Fs[1][c.vidx(v, i, j + 1, k)] - Fs[1][c.vidx(v, i, j, k)]) / c.dx[1] +
                       (Fs[2][c.vidx(v, i, j, k + 1)] - Fs[2][c.vidx(v, i, j, k)]) / c.dx[2];
          double U = sg * prim[c.vidx(v, i, j, k)] + dtau * (-div);
          out[(size_t)(v - 5) * c.nz + c.idx(i, j, k)] = U / sg;
        }
      }
  for (int i = ng; i < ng + c.p.n1; i++)
    for (int j = ng; j < ng + c.p.n2; j++)
      for (int k = ng; k < ng + c.p.n3; k++)
        for (int v = 5; v < 8; v++) prim[c.vidx(v, i, j, k)] = out[(size_t)(v - 5) * c.nz + c.idx(i, j, k)];
  return 0;
}

int oracle_prim_to_cons(oracle_handle h, const double* prim, double* U) {
  Ctx& c = h->c;
#pragma omp parallel for schedule(static)
  for (int i = 0; i < c.n1g; i++)
    for (int j = 0; j < c.n2g; j++)
      for (int k = 0; k < c.n3g; k++) {
        const Geom& G = c.gc[(size_t)i * c.n2g + j];
        double q[8], out[8];
        get_prim(c, prim, i, j, k, q);
        State S;
        fluid_state(q, G, S);
        flux_vector(q, S, G, c.p.gam, 0, out);
        for (int v = 0; v < 8; v++) U[c.vidx(v, i, j, k)] = out[v];
      }
  return 0;
}

// pure inversion on full-grid arrays: no floors, no fix-ups
int oracle_cons_to_prim(oracle_handle h, const double* U, double* prim_inout, int32_t* flag) {
  Ctx& c = h->c;
#pragma omp parallel for schedule(static)
  for (int i = 0; i < c.n1g; i++)
    for (int j = 0; j < c.n2g; j++)
      for (int k = 0; k < c.n3g; k++) {
        const Geom& G = c.gc[(size_t)i * c.n2g + j];
        double u8[8], q[8];
        for (int v = 0; v < 8; v++) { u8[v] = U[c.vidx(v, i, j, k)]; q[v] = prim_inout[c.vidx(v, i, j, k)]; }
        int iters;
        int f = invert_2d(u8, G, c.p.gam, q, c.p.newton_tol, c.p.newton_maxit, c.p.newton_extra, &iters);
        for (int v = 0; v < 8; v++) prim_inout[c.vidx(v, i, j, k)] = q[v];
        if (flag) flag[c.idx(i, j, k)] = f;
      }
  return 0;
}

// C-14 (eq. 26; A17): dt^l = xi dx^l / max over faces of c_w^l ; 1/dt = sum_l 1/dt^l
int oracle_cfl_dt(oracle_handle h, double xi, double* dt_out) {
  Ctx& c = h->c;
  if (!c.prim) return -2;
  double inv = 0.0;
  for (int d = 1; d <= 3; d++) {
    double m;
    flux_dir(c, c.prim, d, c.F[d - 1], c.cw[d - 1], &m);
    double dtl = xi * c.dx[d - 1] / m;
    inv += 1.0 / dtl;
  }
  *dt_out = 1.0 / inv;
  return 0;
}

// dt from the predictor's face speeds of the last oracle_step (the paper's "next time step")
int oracle_last_cfl_dt(oracle_handle h, double xi, double* dt_out) {
  Ctx& c = h->c;
  double inv = 0.0;
  for (int d = 0; d < 3; d++) inv += c.cwmax[d] / (xi * c.dx[d]);
  *dt_out = 1.0 / inv;
  return 0;
}

// C-15 (eq. 23; A4): corner-centred divergence of sqrt(-g) B over corners whose 8 (4 in
// 2D) cells are interior (periodic X3 copies count as interior).
int oracle_divb(oracle_handle h, double* max_abs, double* max_norm) {
  Ctx& c = h->c;
  if (!c.prim) return -2;
  const int ng = c.ng, n1 = c.p.n1, n2 = c.p.n2, n3 = c.p.n3;
  double mabs = 0.0, mnorm = 0.0;
  bool two_d = (n3 == 1);
  int khi = two_d ? ng : ((c.p.bc_x3 == 1) ? ng + n3 - 1 : ng + n3 - 2);
  for (int i = ng; i <= ng + n1 - 2; i++)
    for (int j = ng; j <= ng + n2 - 2; j++)
      for (int k = ng; k <= khi; k++) {
        double D = 0.0, A = 0.0;
        int nl3 = two_d ? 1 : 2;
        for (int l1 = 0; l1 < 2; l1++)
          for (int l2 = 0; l2 < 2; l2++)
            for (int l3 = 0; l3 < nl3; l3++) {
              int ii = i + l1, jj = j + l2, kk = k + l3;
              double sg = c.gc[(size_t)ii * c.n2g + jj].sqrtg;
              double w = two_d ? 0.5 : 0.25;
              double t1 = (l1 ? 1.0 : -1.0) * sg * c.prim[c.vidx(5, ii, jj, kk)] * w / c.dx[0];
              double t2 = (l2 ? 1.0 : -1.0) * sg * c.prim[c.vidx(6, ii, jj, kk)] * w / c.dx[1];
              D += t1 + t2; A += std::fabs(t1) + std::fabs(t2);
              if (!two_d) {
                double t3 = (l3 ? 1.0 : -1.0) * sg * c.prim[c.vidx(7, ii, jj, kk)] * w / c.dx[2];
                D += t3; A += std::fabs(t3);
              }
            }
        if (std::fabs(D) > mabs) mabs = std::fabs(D);
        // A4 (addition): a corner whose terms sum to less than 1e-290 in magnitude is skipped in the normalised
        // measure: there the terms sit within 2^53 of the subnormal range, where rounding is absolute, not relative,
        // and |D| / sum|terms| says nothing (the far edge of the numerical diffusion front of B decays into that
        // range after a few dozen steps).  max |D| itself still covers every corner.
        if (A > 1e-290 && std::fabs(D) / A > mnorm) mnorm = std::fabs(D) / A;
      }
  *max_abs = mabs; *max_norm = mnorm;
  return 0;
}

// fluxes through the coordinate shell of zone centres X1 = X1_i (eqs. 43-46),
// "at the horizon" when i is the shell nearest r_h.  In the code's coordinates the integrand of each surface
// integral is sqrt(-g) x (the X1 component of the current) dX2 dX3, which is coordinate invariant:
//   out[0] = Mdot  = sum sqrt(-g) rho u^1            dX2 dX3   (eq. 43; negative for inflow, as printed)
//   out[1] = phi_B = 1/2 sum sqrt(-g) |B^1|          dX2 dX3   (eq. 44; *F^{rt} = B^r)
//   out[2] = Ldot  = sum sqrt(-g) T^1_phi            dX2 dX3   (eq. 45)
//   out[3] = Edot  = sum -sqrt(-g) T^1_t             dX2 dX3   (eq. 46)
// i: interior numbering 0..n1-1.  Plain sums in (j, k) order.
int oracle_shell_fluxes(oracle_handle h, int32_t i, double out[4]) {
  Ctx& c = h->c;
  if (!c.prim) return -2;
  if (i < 0 || i >= c.p.n1) return -1;
  const int ng = c.ng, n2 = c.p.n2, n3 = c.p.n3;
  const int ii = ng + i;
  const double dA = c.dx[1] * c.dx[2];
  double mdot = 0.0, phib = 0.0, ldot = 0.0, edot = 0.0;
  for (int j = ng; j < ng + n2; j++) {
    const Geom& G = c.gc[(size_t)ii * c.n2g + j];
    for (int k = ng; k < ng + n3; k++) {
      double q[8];
      for (int v = 0; v < 8; v++) q[v] = c.prim[c.vidx(v, ii, j, k)];
      State S;
      fluid_state(q, G, S);
      double F[8];
      flux_vector(q, S, G, c.p.gam, 1, F);   // sqrt(-g) x (rho u^1, T^1_t, T^1_1, T^1_2, T^1_3, ...)
      mdot += F[0] * dA;
      phib += 0.5 * G.sqrtg * std::fabs(q[5]) * dA;
      ldot += F[4] * dA;
      edot += -F[1] * dA;
    }
  }
  out[0] = mdot; out[1] = phib; out[2] = ldot; out[3] = edot;
  return 0;
}

// 0 failed inversions, 1 zones repaired, 2 rho-floor hits, 3 u-floor hits, 4 ceilings, 5 Lorentz caps,
// 6 Newton iterations, 7 zones repaired by the last-resort rule
int oracle_get_stats(oracle_handle h, int64_t out[8]) {
  for (int s = 0; s < 8; s++) out[s] = h->c.stats[s];
  return 0;
}

// 0 zones sent down the fallback chain, 1 recovered by 1D-W, 2 recovered by the entropy method, 3 entropy-first zones
int oracle_get_chain_stats(oracle_handle h, int64_t out[4]) {
  for (int s = 0; s < 4; s++) out[s] = h->c.chain[s];
  return 0;
}

// point-level entry points of the fallback inversions (for the pins)
int oracle_invert_1dw(const double U[8], const double gcov[16], const double gcon[16], double sqrtg, double gam,
                      double prim_inout[8], double tol, int maxit) {
  Geom G; geom_from_arrays(gcov, gcon, sqrtg, G);
  return invert_1dw(U, G, gam, prim_inout, tol, maxit);
}

int oracle_invert_entropy(const double U[8], double US, const double gcov[16], const double gcon[16], double sqrtg,
                          double gam, double prim_inout[8], double tol, int maxit) {
  Geom G; geom_from_arrays(gcov, gcon, sqrtg, G);
  return invert_entropy(U, US, G, gam, prim_inout, tol, maxit);
}

// conserved entropy sqrt(-g) S u^t of a primitive state (eq. 11)
double oracle_entropy_cons(const double prim[8], const double gcov[16], const double gcon[16], double sqrtg, double gam) {
  Geom G; geom_from_arrays(gcov, gcon, sqrtg, G);
  State S; fluid_state(prim, G, S);
  return G.sqrtg * entropy_of(prim[0], prim[1], gam) * S.ucon[0];
}

// entropy flux of one direction over the faces flux_dir covers (eq. 11), out[nz]
int oracle_entropy_flux_dir(oracle_handle h, const double* prim, int dir, double* FS_out) {
  Ctx& c = h->c;
  std::vector<double> F, CW, FS;
  double m;
  flux_dir(c, prim, dir, F, CW, &m, &FS);
  std::memcpy(FS_out, FS.data(), c.nz * sizeof(double));
  return 0;
}

int oracle_get_flags(oracle_handle h, int32_t* out) {
  std::memcpy(out, h->c.flag.data(), h->c.nz * sizeof(int32_t));
  return 0;
}

// stage-level: floors / ceilings / Lorentz cap (C-12) on every interior zone of a caller-provided primitive array,
// in place; mask[zone] = apply_floors' bit mask (may be null)
int oracle_apply_floors_grid(oracle_handle h, double* prim, int32_t* mask) {
  Ctx& c = h->c;
  const int ng = c.ng;
  for (int i = ng; i < ng + c.p.n1; i++)
    for (int j = ng; j < ng + c.p.n2; j++)
      for (int k = ng; k < ng + c.p.n3; k++) {
        size_t g2 = (size_t)i * c.n2g + j;
        double q[8];
        get_prim(c, prim, i, j, k, q);
        int m = apply_floors(c.p, c.rc[g2], c.gc[g2], q);
        for (int v = 0; v < 8; v++) prim[c.vidx(v, i, j, k)] = q[v];
        if (mask) mask[c.idx(i, j, k)] = m;
      }
  return 0;
}

// stage-level: fix-up on a caller-provided primitive array with caller-provided flags
int oracle_fixup(oracle_handle h, double* prim, const int32_t* flag) {
  Ctx& c = h->c;
  c.flag.assign(flag, flag + c.nz);
  fixup(c, prim);
  return 0;
}

}  // extern "C"
