// cuharm_phys.cuh — per-zone / per-face device arithmetic of the HARM update (fp64, sm_100a).
//
// Written from the paper (arXiv 2205.02484): "P:L<n>" = PAPER.md line n; "A<n>" = a DESIGN.md reading.
// Shares nothing with oracle/ (the CPU checker): no header, table, constant generator or helper.
//
// Metric storage.  In Kerr-Schild coordinates and under the diagonal MKS Jacobian (eqs. 38-39) the covariant and
// the contravariant metric have the same zero pattern: the (0,2), (1,2), (2,3) entries vanish.  Only the seven
// entries 00 01 03 11 13 22 33 of each are stored and every contraction below skips the structural zeros (adding
// an exact zero never changes a sum, so this is the same arithmetic as the full 4x4 contraction).
#pragma once
#include <cstdint>

namespace cuharm {

// one geometry record: 16 doubles = one 128-byte line, read as a warp-wide broadcast
struct Geom {
  double g00, g01, g03, g11, g13, g22, g33;  // g_{mu nu}
  double c00, c01, c03, c11, c13, c22, c33;  // g^{mu nu}
  double sg, alpha;                          // sqrt(-g), lapse 1/sqrt(-g^tt)
};
static_assert(sizeof(Geom) == 128, "Geom must be one cache line");

__device__ __forceinline__ Geom load_geom(const Geom* __restrict__ tab, int q) {
  const double2* s = reinterpret_cast<const double2*>(tab + q);
  Geom G;
  double2 v;
  v = __ldg(s + 0); G.g00 = v.x; G.g01 = v.y;
  v = __ldg(s + 1); G.g03 = v.x; G.g11 = v.y;
  v = __ldg(s + 2); G.g13 = v.x; G.g22 = v.y;
  v = __ldg(s + 3); G.g33 = v.x; G.c00 = v.y;
  v = __ldg(s + 4); G.c01 = v.x; G.c03 = v.y;
  v = __ldg(s + 5); G.c11 = v.x; G.c13 = v.y;
  v = __ldg(s + 6); G.c22 = v.x; G.c33 = v.y;
  v = __ldg(s + 7); G.sg = v.x; G.alpha = v.y;
  return G;
}

// ---------------------------------------------------------------------------------------------------------
// Primitive -> four-velocity and magnetic four-vector (eq. 10).
// q = (rho, u, ut1, ut2, ut3, B1, B2, B3).
// ---------------------------------------------------------------------------------------------------------
struct State {
  double u0, u1, u2, u3;      // u^mu
  double l0, l1, l2, l3;      // u_mu
  double b0, b1, b2, b3;      // b^mu
  double m0, m1, m2, m3;      // b_mu
  double bsq, lor;
};

__device__ __forceinline__ double gamma_sq_minus_one(const double q[8], const Geom& G) {
  // g_ij ut^i ut^j
  return G.g11 * q[2] * q[2] + G.g22 * q[3] * q[3] + G.g33 * q[4] * q[4] + 2.0 * (G.g13 * q[2] * q[4]);
}

__device__ __forceinline__ void lower(const Geom& G, double v0, double v1, double v2, double v3, double& w0, double& w1,
                                      double& w2, double& w3) {
  w0 = G.g00 * v0 + G.g01 * v1 + G.g03 * v3;
  w1 = G.g01 * v0 + G.g11 * v1 + G.g13 * v3;
  w2 = G.g22 * v2;
  w3 = G.g03 * v0 + G.g13 * v1 + G.g33 * v3;
}

__device__ __forceinline__ void fluid_state(const double q[8], const Geom& G, State& S) {
  const double lor = sqrt(1.0 + gamma_sq_minus_one(q, G));  // Gamma
  S.lor = lor;
  const double a = G.alpha;
  S.u0 = lor / a;
  // beta^i / alpha = alpha g^{ti};  u^i = ut^i - Gamma beta^i / alpha  (eq. 10)
  const double la = lor * a;
  S.u1 = q[2] - la * G.c01;
  S.u2 = q[3];
  S.u3 = q[4] - la * G.c03;
  lower(G, S.u0, S.u1, S.u2, S.u3, S.l0, S.l1, S.l2, S.l3);
  const double bt = q[5] * S.l1 + q[6] * S.l2 + q[7] * S.l3;  // b^t = B^i u_i
  const double iu0 = 1.0 / S.u0;
  S.b0 = bt;
  S.b1 = (q[5] + bt * S.u1) * iu0;  // b^i = (B^i + b^t u^i) / u^t
  S.b2 = (q[6] + bt * S.u2) * iu0;
  S.b3 = (q[7] + bt * S.u3) * iu0;
  lower(G, S.b0, S.b1, S.b2, S.b3, S.m0, S.m1, S.m2, S.m3);
  S.bsq = S.b0 * S.m0 + S.b1 * S.m1 + S.b2 * S.m2 + S.b3 * S.m3;
}

__device__ __forceinline__ double pick(int d, double a0, double a1, double a2, double a3) {
  return d == 0 ? a0 : (d == 1 ? a1 : (d == 2 ? a2 : a3));
}

// ---------------------------------------------------------------------------------------------------------
// Conserved variables (DIR = 0) and fluxes (DIR = 1,2,3): eqs. 5-8.
//   [0] sqrt(-g) rho u^d   [1..4] sqrt(-g) T^d_nu   [5..7] sqrt(-g)(b^i u^d - b^d u^i)   (A1: sign; A18)
// ---------------------------------------------------------------------------------------------------------
template <int DIR>
__device__ __forceinline__ void flux_vector(const double q[8], const State& S, const Geom& G, double gam, double out[8]) {
  const double pg = (gam - 1.0) * q[1];
  const double w = q[0] + q[1] + pg;        // enthalpy density
  const double ud = pick(DIR, S.u0, S.u1, S.u2, S.u3);
  const double bd = pick(DIR, S.b0, S.b1, S.b2, S.b3);
  const double eta = (w + S.bsq) * ud;
  const double ptot = pg + 0.5 * S.bsq;
  const double sg = G.sg;
  out[0] = sg * (q[0] * ud);
  double t0 = eta * S.l0 - bd * S.m0;
  double t1 = eta * S.l1 - bd * S.m1;
  double t2 = eta * S.l2 - bd * S.m2;
  double t3 = eta * S.l3 - bd * S.m3;
  if (DIR == 0) t0 += ptot;
  if (DIR == 1) t1 += ptot;
  if (DIR == 2) t2 += ptot;
  if (DIR == 3) t3 += ptot;
  out[1] = sg * t0;
  out[2] = sg * t1;
  out[3] = sg * t2;
  out[4] = sg * t3;
  out[5] = sg * (S.b1 * ud - bd * S.u1);
  out[6] = sg * (S.b2 * ud - bd * S.u2);
  out[7] = sg * (S.b3 * ud - bd * S.u3);
}

// ---------------------------------------------------------------------------------------------------------
// Fast-magnetosonic bounds from the quadratic dispersion relation (eqs. 18-19): roots of
// A v^2 + B v + C = 0, c1 >= c2.  A29: a negative discriminant is clamped to zero.
// ---------------------------------------------------------------------------------------------------------
template <int DIR>
__device__ __forceinline__ void wave_speeds(const double q[8], const State& S, const Geom& G, double gam, double& c1,
                                            double& c2) {
  const double pg = (gam - 1.0) * q[1];
  const double w = q[0] + q[1] + pg;
  const double cs2 = gam * pg / w;               // eq. 19
  const double va2 = S.bsq / (S.bsq + w);
  const double cms2 = va2 + cs2 * (1.0 - va2);   // eq. 18
  const double ut = S.u0;
  const double ud = pick(DIR, S.u0, S.u1, S.u2, S.u3);
  const double gtd = DIR == 1 ? G.c01 : (DIR == 3 ? G.c03 : 0.0);
  const double gdd = DIR == 1 ? G.c11 : (DIR == 2 ? G.c22 : G.c33);
  const double A = ut * ut - cms2 * (G.c00 + ut * ut);
  const double B = -2.0 * (ut * ud - cms2 * (gtd + ut * ud));
  const double C = ud * ud - cms2 * (gdd + ud * ud);
  double disc = B * B - 4.0 * A * C;
  disc = disc < 0.0 ? 0.0 : disc;
  const double sq = sqrt(disc);
  const double i2A = 1.0 / (2.0 * A);
  const double ra = (-B + sq) * i2A;
  const double rb = (-B - sq) * i2A;
  c1 = ra > rb ? ra : rb;
  c2 = ra > rb ? rb : ra;
}

// ---------------------------------------------------------------------------------------------------------
// Reconstruction.  MC-limited slope, eq. 15 (A2: the last branch is signed).
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double slope_mc(double qm, double q0, double qp) {
  const double dm = q0 - qm, dp = qp - q0;
  const double dc = 0.5 * (qp - qm);
  const double am = 2.0 * fabs(dm), ap = 2.0 * fabs(dp), ac = fabs(dc);
  // for dm, dp of one sign |dc| is the mean of |dm|, |dp|: at most one of the one-sided tests can hold
  double s = dc;
  s = (ap < ac) ? 2.0 * dp : s;
  s = (am < ac && fabs(dm) < fabs(dp)) ? 2.0 * dm : s;
  return (dm * dp < 0.0) ? 0.0 : s;
}

// Values at the lower (ql) and upper (qr) face of the cell y2 from the cell values y0..y4 around it.
// RECON 0: piecewise linear, eq. 16.  RECON 1: piecewise parabolic (A20): MC-limited
// slopes, 4th-order interface values, monotonisation; no steepening, no flattening.
template <int RECON>
__device__ __forceinline__ void recon_cell(double y0, double y1, double y2, double y3, double y4, double& ql, double& qr) {
  if (RECON == 0) {
    const double dq = slope_mc(y1, y2, y3);
    ql = y2 - 0.5 * dq;
    qr = y2 + 0.5 * dq;
  } else {
    const double dm = slope_mc(y0, y1, y2);
    const double d0 = slope_mc(y1, y2, y3);
    const double dp = slope_mc(y2, y3, y4);
    double l = 0.5 * (y1 + y2) - (d0 - dm) / 6.0;
    double r = 0.5 * (y2 + y3) - (dp - d0) / 6.0;
    if ((r - y2) * (y2 - l) <= 0.0) {
      l = y2;
      r = y2;
    } else {
      const double d = r - l;
      const double m6 = d * (y2 - 0.5 * (l + r));
      const double lim = d * d / 6.0;
      if (m6 > lim) l = 3.0 * y2 - 2.0 * r;
      else if (m6 < -lim) r = 3.0 * y2 - 2.0 * l;
    }
    ql = l;
    qr = r;
  }
}

// ---------------------------------------------------------------------------------------------------------
// Riemann flux at one face from the two reconstructed states and the FACE metric.
// RIEMANN 0: local Lax-Friedrichs, eq. 17.  RIEMANN 1: HLL, eq. 20 (A30: guarded denominator).
// ---------------------------------------------------------------------------------------------------------
template <int DIR, int RIEMANN>
__device__ __forceinline__ void face_flux(const double pl[8], const double pr[8], const Geom& G, double gam, double F[8],
                                          double& cw) {
  State S;
  double Ul[8], Fl[8], c1l, c2l;
  fluid_state(pl, G, S);
  flux_vector<0>(pl, S, G, gam, Ul);
  flux_vector<DIR>(pl, S, G, gam, Fl);
  wave_speeds<DIR>(pl, S, G, gam, c1l, c2l);
  double Ur[8], Fr[8], c1r, c2r;
  fluid_state(pr, G, S);
  flux_vector<0>(pr, S, G, gam, Ur);
  flux_vector<DIR>(pr, S, G, gam, Fr);
  wave_speeds<DIR>(pr, S, G, gam, c1r, c2r);
  const double cmax = fmax(0.0, fmax(c1r, c1l));
  const double cmin = fmax(0.0, fmax(-c2r, -c2l));
  cw = fmax(cmax, cmin);
  if (RIEMANN == 0) {
#pragma unroll
    for (int v = 0; v < 8; v++) F[v] = 0.5 * (Fl[v] + Fr[v] - cw * (Ur[v] - Ul[v]));
  } else {
    const double iden = 1.0 / fmax(cmax + cmin, 1e-300);
    const double cc = cmax * cmin;
#pragma unroll
    for (int v = 0; v < 8; v++) F[v] = (cmax * Fl[v] + cmin * Fr[v] - cc * (Ur[v] - Ul[v])) * iden;
  }
}

// ---------------------------------------------------------------------------------------------------------
// Geometric source S_nu = sqrt(-g) T^kappa_lambda Gamma^lambda_{nu kappa} (eq. 7; eq. 14).
// conn: 40 doubles, Gamma^l_{nk} with l-major and the (n,k) pair order 00 01 02 03 11 12 13 22 23 33.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ int pair_index(int n, int k) {
  // index of the unordered pair (n,k) in 00 01 02 03 11 12 13 22 23 33
  const int lo = n < k ? n : k, hi = n < k ? k : n;
  return lo * 4 - (lo * (lo - 1)) / 2 + (hi - lo);
}

__device__ __forceinline__ void source_term(const double q[8], const State& S, const Geom& G, const double* __restrict__ conn,
                                            double gam, double src[4]) {
  const double pg = (gam - 1.0) * q[1];
  const double w = q[0] + q[1] + pg;
  const double eta = w + S.bsq;
  const double ptot = pg + 0.5 * S.bsq;
  const double uc[4] = {S.u0, S.u1, S.u2, S.u3}, ul[4] = {S.l0, S.l1, S.l2, S.l3};
  const double bc[4] = {S.b0, S.b1, S.b2, S.b3}, bl[4] = {S.m0, S.m1, S.m2, S.m3};
  double T[4][4];  // T^k_l
#pragma unroll
  for (int k = 0; k < 4; k++)
#pragma unroll
    for (int l = 0; l < 4; l++) T[k][l] = eta * uc[k] * ul[l] + (k == l ? ptot : 0.0) - bc[k] * bl[l];
#pragma unroll
  for (int nu = 0; nu < 4; nu++) {
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 4; k++)
#pragma unroll
      for (int l = 0; l < 4; l++) s += T[k][l] * __ldg(conn + l * 10 + pair_index(nu, k));
    src[nu] = G.sg * s;
  }
}

// ---------------------------------------------------------------------------------------------------------
// Noble 2D Newton-Raphson inversion (eqs. 27-31; A6: minus sign in eq. 30; A7: D = alpha rho u^t;
// A8: guess, |dW/W| criterion, `extra` more iterations, iteration cap).  Returns 0 or a failure code
// (include/cuharm.h); on failure the fluid primitives keep the guess.  B^i = U_B / sqrt(-g) always.
// ---------------------------------------------------------------------------------------------------------
struct NewtonCfg {
  double tol;
  int maxit, extra;
};

__device__ __noinline__ int invert_2d(const double U[8], const Geom& G, double gam, double q[8], NewtonCfg nc, int& iters) {
  iters = 0;
  const double a = G.alpha;
  const double isg = 1.0 / G.sg;
  const double B1 = U[5] * isg, B2 = U[6] * isg, B3 = U[7] * isg;
  const double g1 = q[2], g2 = q[3], g3 = q[4];  // guess velocity
  const double grho = q[0], gu = q[1];
  q[5] = B1; q[6] = B2; q[7] = B3;
  const double aisg = a * isg;
  const double D = aisg * U[0];
  const double Q0 = aisg * U[1], Q1 = aisg * U[2], Q2 = aisg * U[3], Q3 = aisg * U[4];  // Q_mu
  const double Bc1 = a * B1, Bc2 = a * B2, Bc3 = a * B3;                                  // script-B^i
  const bool fin = isfinite(D) && isfinite(Q0) && isfinite(Q1) && isfinite(Q2) && isfinite(Q3) && isfinite(Bc1) &&
                   isfinite(Bc2) && isfinite(Bc3);
  if (!fin || !(D > 0.0)) return 1;
  // Q^mu = g^{mu nu} Q_nu
  const double Qc0 = G.c00 * Q0 + G.c01 * Q1 + G.c03 * Q3;
  const double Qc1 = G.c01 * Q0 + G.c11 * Q1 + G.c13 * Q3;
  const double Qc2 = G.c22 * Q2;
  const double Qc3 = G.c03 * Q0 + G.c13 * Q1 + G.c33 * Q3;
  const double Bsq = G.g11 * Bc1 * Bc1 + G.g22 * Bc2 * Bc2 + G.g33 * Bc3 * Bc3 + 2.0 * (G.g13 * Bc1 * Bc3);
  const double QdB = Q1 * Bc1 + Q2 * Bc2 + Q3 * Bc3;
  // n_mu = (-alpha,0,0,0); n^mu = (1/alpha, -alpha g^{ti})
  const double n0 = 1.0 / a, n1 = -a * G.c01, n3 = -a * G.c03;
  const double Qdn = Q0 * n0 + Q1 * n1 + Q3 * n3;
  const double Qsq = Qc0 * Q0 + Qc1 * Q1 + Qc2 * Q2 + Qc3 * Q3;
  const double Qtsq = Qsq + Qdn * Qdn;
  const double QdB2 = QdB * QdB;
  const double gfac = (gam - 1.0) / gam;
  // initial guess: W = Gamma^2 w from the guess, v^2 from eq. 29 at that W
  const double qsq = G.g11 * g1 * g1 + G.g22 * g2 * g2 + G.g33 * g3 * g3 + 2.0 * (G.g13 * g1 * g3);
  double W = (1.0 + qsq) * (grho + gam * gu);
  double v2 = 0.0;
  for (int t = 0; t < 400; t++) {
    v2 = (Qtsq + QdB2 * (Bsq + 2.0 * W) / (W * W)) / ((Bsq + W) * (Bsq + W));
    if (v2 < 1.0) break;
    W *= 10.0;
  }
  if (!(v2 < 1.0) || !(W > 0.0)) return 3;
  v2 = v2 < 0.0 ? 0.0 : v2;
  bool converged = false;
  int extra_left = -1;
  int it;
  for (it = 1; it <= nc.maxit; it++) {
    const double iW = 1.0 / W;
    const double iW2 = iW * iW, iW3 = iW2 * iW;
    const double omv = 1.0 - v2;
    const double sq = sqrt(omv);
    const double BW = Bsq + W;
    const double pg = gfac * (W * omv - D * sq);                                   // eq. 31
    const double f1 = Qtsq - v2 * BW * BW + QdB2 * (Bsq + 2.0 * W) * iW2;          // eq. 29
    const double f2 = -Qdn - 0.5 * Bsq * (1.0 + v2) + 0.5 * QdB2 * iW2 - W + pg;   // eq. 30 (A6)
    const double j11 = -2.0 * BW * (v2 + QdB2 * iW3);
    const double j12 = -BW * BW;
    const double j21 = -1.0 - QdB2 * iW3 + gfac * omv;
    const double j22 = -0.5 * Bsq + gfac * (-W + D / (2.0 * sq));
    const double idet = 1.0 / (j11 * j22 - j12 * j21);
    const double dW = (-f1 * j22 + f2 * j12) * idet;
    const double dv = (-f2 * j11 + f1 * j21) * idet;
    const double Wn = fabs(W + dW);
    double vn = v2 + dv;
    vn = vn < 0.0 ? 0.0 : vn;
    vn = vn > 1.0 - 1e-15 ? 1.0 - 1e-15 : vn;
    const double err = (Wn == 0.0) ? fabs(dW) : fabs(dW / Wn);
    W = Wn;
    v2 = vn;
    if (!isfinite(W) || !isfinite(v2)) { iters = it; return 3; }
    if (extra_left < 0) {
      if (err <= nc.tol) extra_left = nc.extra;
    } else {
      extra_left--;
    }
    if (extra_left == 0) { converged = true; break; }
  }
  iters = it > nc.maxit ? nc.maxit : it;
  if (!converged) return 2;
  if (!(W > 0.0)) return 3;
  if (!(v2 >= 0.0 && v2 < 1.0)) return 4;
  const double lor = 1.0 / sqrt(1.0 - v2);
  const double rho = D / lor;
  const double w = W * (1.0 - v2);
  const double u = (w - rho) / gam;
  if (!(rho > 0.0)) return 5;
  if (!(u >= 0.0)) return 6;
  q[0] = rho;
  q[1] = u;
  const double f = lor / (W + Bsq);
  const double QdBW = QdB / W;
  q[2] = f * (Qc1 + n1 * Qdn + QdBW * Bc1);  // ut^i = Gamma [Qt^i + (Q.B) B^i / W] / (W + B^2)
  q[3] = f * (Qc2 + QdBW * Bc2);
  q[4] = f * (Qc3 + n3 * Qdn + QdBW * Bc3);
  return 0;
}

// ---------------------------------------------------------------------------------------------------------
// Floors and ceilings (eqs. 35-37; A9-A12).  rfl, ufl: the eq. 35 profiles of this (i,j).
// Bit mask returned: 1 rho floor, 2 u floor, 4 ceiling applied, 8 Lorentz cap, 16 ceiling re-inversion failed.
// ---------------------------------------------------------------------------------------------------------
struct FloorCfg {
  double sigma_max, b2_over_u_max, gamma_max;
};

__device__ __forceinline__ int apply_floors(double q[8], const Geom& G, double rfl, double ufl, FloorCfg fc, double gam,
                                            NewtonCfg nc) {
  int mask = 0;
  if (q[0] < rfl) { q[0] = rfl; mask |= 1; }
  if (q[1] < ufl) { q[1] = ufl; mask |= 2; }
  if (fc.sigma_max > 0.0 || fc.b2_over_u_max > 0.0) {
    // b^2 by the identity b^2 = (B^2 + (B.u)^2) / Gamma^2 would be cheaper, but the state is needed below anyway
    State S;
    fluid_state(q, G, S);
    double drho = 0.0, du = 0.0;
    if (fc.sigma_max > 0.0) drho = fmax(0.0, S.bsq / fc.sigma_max - q[0]);
    if (fc.b2_over_u_max > 0.0) du = fmax(0.0, S.bsq / fc.b2_over_u_max - q[1]);
    if (drho > 0.0 || du > 0.0) {  // rare: mass/energy injected at rest in the normal-observer frame (A11)
      mask |= 4;
      double U[8], Ua[8];
      flux_vector<0>(q, S, G, gam, U);
      double qa[8] = {drho, du, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
      State Sa;
      fluid_state(qa, G, Sa);
      flux_vector<0>(qa, Sa, G, gam, Ua);
#pragma unroll
      for (int v = 0; v < 8; v++) U[v] += Ua[v];
      double t[8];
#pragma unroll
      for (int v = 0; v < 8; v++) t[v] = q[v];
      int its;
      const int flag = invert_2d(U, G, gam, t, nc, its);
      if (flag == 0) {
#pragma unroll
        for (int v = 0; v < 5; v++) q[v] = t[v];
      } else {
        q[0] += drho;
        q[1] += du;
        mask |= 16;
      }
      State S2;
      fluid_state(q, G, S2);
      if (fc.sigma_max > 0.0) q[0] = fmax(q[0], S2.bsq / fc.sigma_max);
      if (fc.b2_over_u_max > 0.0) q[1] = fmax(q[1], S2.bsq / fc.b2_over_u_max);
    }
  }
  if (fc.gamma_max > 0.0) {
    const double qsq = gamma_sq_minus_one(q, G);
    const double lor = sqrt(1.0 + qsq);
    if (lor > fc.gamma_max) {
      const double f = sqrt((fc.gamma_max * fc.gamma_max - 1.0) / (lor * lor - 1.0));  // A12
      q[2] *= f; q[3] *= f; q[4] *= f;
      mask |= 8;
    }
  }
  return mask;
}

}  // namespace cuharm
