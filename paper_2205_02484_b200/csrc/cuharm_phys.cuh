// cuharm_phys.cuh — per-zone / per-face device arithmetic of the HARM update (fp64, sm_100a).
//
// Written from the paper (arXiv 2205.02484): "P:L<n>" = PAPER.md line n; "A<n>" = a DESIGN.md reading.
// Shares nothing with oracle/ (the CPU checker): no header, table, constant generator or helper.
//
// Metric storage.  In Kerr-Schild coordinates and under the diagonal MKS Jacobian (eqs. 38-39) the covariant and
// the contravariant metric have the same zero pattern: the (0,2), (1,2), (2,3) entries vanish, and g^{t phi} = 0 as
// well.  Only the seven entries 00 01 03 11 13 22 33 of each are stored and every contraction below skips the
// structural zeros (adding an exact zero never changes a sum: the same arithmetic as the full 4x4 contraction).
#pragma once
#include <cstdint>

namespace cuharm {

// one geometry record: 20 doubles = 160 bytes, read as a warp-wide broadcast.  g^{t phi} vanishes identically in
// Kerr-Schild coordinates (and in Minkowski), so c03 is kept only for the export helper; the arithmetic skips it.
struct Geom {
  double g00, g01, g03, g11, g13, g22, g33;  // g_{mu nu}
  double c00, c01, c03, c11, c13, c22, c33;  // g^{mu nu}
  double sg, alpha;                          // sqrt(-g), lapse 1/sqrt(-g^tt)
  double ialpha, ac01;                       // 1/alpha, alpha g^{t1} = -beta^1/alpha
  double isg, pad;                           // 1/sqrt(-g) (0 where sqrt(-g) = 0: the polar faces, A32)
};
static_assert(sizeof(Geom) == 160, "Geom is 20 doubles");

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
  v = __ldg(s + 8); G.ialpha = v.x; G.ac01 = v.y;
  v = __ldg(s + 9); G.isg = v.x; G.pad = 0.0;
  return G;
}

// the same record from shared memory (or any generic pointer): plain loads
__device__ __forceinline__ Geom load_geom_shared(const double* t) {
  const double2* s = reinterpret_cast<const double2*>(t);
  Geom G;
  double2 v;
  v = s[0]; G.g00 = v.x; G.g01 = v.y;
  v = s[1]; G.g03 = v.x; G.g11 = v.y;
  v = s[2]; G.g13 = v.x; G.g22 = v.y;
  v = s[3]; G.g33 = v.x; G.c00 = v.y;
  v = s[4]; G.c01 = v.x; G.c03 = v.y;
  v = s[5]; G.c11 = v.x; G.c13 = v.y;
  v = s[6]; G.c22 = v.x; G.c33 = v.y;
  v = s[7]; G.sg = v.x; G.alpha = v.y;
  v = s[8]; G.ialpha = v.x; G.ac01 = v.y;
  v = s[9]; G.isg = v.x; G.pad = 0.0;
  return G;
}

// ---------------------------------------------------------------------------------------------------------
// Reciprocal and reciprocal square root for the hot path: the hardware seed (MUFU.RCP64H / MUFU.RSQ64H, about 20
// good bits) plus ONE third-order Newton step, no special-case path.  Result within 2 ulp for normal, finite
// arguments; callers guarantee that (x > 0 where a root is taken, |x| far from the subnormal range).  The IEEE
// division sequence nvcc emits costs three times the fp64 instructions and enters a ~100-instruction slow path
// whenever the NUMERATOR is zero — which it is (B = 0) in 90 % of the zones of a torus workload.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double frcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x, r, 1.0);     // 1 - x r, |e| <~ 2^-20
  return fma(r, fma(e, e, e), r);       // r (1 + e + e^2): error e^3
}

__device__ __forceinline__ double frsqrt(double x) {
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x * r, r, 1.0);               // 1 - x r^2
  return fma(r, e * fma(0.375, e, 0.5), r);           // r (1 + e/2 + 3 e^2/8): error 5 e^3/16
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
  // covariant spatial components: u_i = g_ij utilde^j exactly, because g_ij beta^j = g_ti (the shift lowered by the
  // spatial metric) cancels the u^t term of u_i = g_it u^t + g_ij u^j; likewise u_t = -alpha Gamma + beta^i u_i with
  // beta^1 = alpha (alpha g^{t1}) the only non-zero shift component in Kerr-Schild coordinates.
  S.l1 = fma(G.g11, q[2], G.g13 * q[4]);
  S.l2 = G.g22 * q[3];
  S.l3 = fma(G.g13, q[2], G.g33 * q[4]);
  const double x = 1.0 + fma(S.l1, q[2], fma(S.l2, q[3], S.l3 * q[4]));  // Gamma^2 = 1 + g_ij ut^i ut^j
  const double ilor = frsqrt(x);
  const double lor = x * ilor;  // Gamma = sqrt(1 + q^2)
  S.lor = lor;
  S.u0 = lor * G.ialpha;
  // beta^i / alpha = alpha g^{ti};  u^i = ut^i - Gamma beta^i / alpha  (eq. 10);  g^{t2} = g^{t3} = 0
  S.u1 = fma(-lor, G.ac01, q[2]);
  S.u2 = q[3];
  S.u3 = q[4];
  S.l0 = G.alpha * fma(G.ac01, S.l1, -lor);
  const double bt = fma(q[5], S.l1, fma(q[6], S.l2, q[7] * S.l3));  // b^t = B^i u_i
  const double iu0 = G.alpha * ilor;
  S.b0 = bt;
  S.b1 = fma(bt, S.u1, q[5]) * iu0;  // b^i = (B^i + b^t u^i) / u^t
  S.b2 = fma(bt, S.u2, q[6]) * iu0;
  S.b3 = fma(bt, S.u3, q[7]) * iu0;
  lower(G, S.b0, S.b1, S.b2, S.b3, S.m0, S.m1, S.m2, S.m3);
  S.bsq = fma(S.b0, S.m0, fma(S.b1, S.m1, fma(S.b2, S.m2, S.b3 * S.m3)));
}

__device__ __forceinline__ double pick(int d, double a0, double a1, double a2, double a3) {
  return d == 0 ? a0 : (d == 1 ? a1 : (d == 2 ? a2 : a3));
}

// ---------------------------------------------------------------------------------------------------------
// Conserved variables (DIR = 0) and fluxes (DIR = 1,2,3) DIVIDED BY sqrt(-g): eqs. 5-8.
//   [0] rho u^d   [1..4] T^d_nu   [5..7] b^i u^d - b^d u^i   (A1: sign; A18)
// For DIR = 0 the last three are B^i themselves: b^i u^t - b^t u^i = B^i by the definition of b^i.
// ---------------------------------------------------------------------------------------------------------
template <int DIR>
__device__ __forceinline__ void flux_hat(const double q[8], const State& S, double gam, double out[8]) {
  const double pg = (gam - 1.0) * q[1];
  const double w = q[0] + q[1] + pg;        // enthalpy density
  const double ud = pick(DIR, S.u0, S.u1, S.u2, S.u3);
  const double bd = pick(DIR, S.b0, S.b1, S.b2, S.b3);
  const double eta = (w + S.bsq) * ud;
  const double ptot = fma(0.5, S.bsq, pg);
  out[0] = q[0] * ud;
  double t0 = eta * S.l0 - bd * S.m0;
  double t1 = eta * S.l1 - bd * S.m1;
  double t2 = eta * S.l2 - bd * S.m2;
  double t3 = eta * S.l3 - bd * S.m3;
  if (DIR == 0) t0 += ptot;
  if (DIR == 1) t1 += ptot;
  if (DIR == 2) t2 += ptot;
  if (DIR == 3) t3 += ptot;
  out[1] = t0;
  out[2] = t1;
  out[3] = t2;
  out[4] = t3;
  if (DIR == 0) {
    out[5] = q[5]; out[6] = q[6]; out[7] = q[7];
  } else {
    out[5] = DIR == 1 ? 0.0 : S.b1 * ud - bd * S.u1;
    out[6] = DIR == 2 ? 0.0 : S.b2 * ud - bd * S.u2;
    out[7] = DIR == 3 ? 0.0 : S.b3 * ud - bd * S.u3;
  }
}

template <int DIR>
__device__ __forceinline__ void flux_vector(const double q[8], const State& S, const Geom& G, double gam, double out[8]) {
  flux_hat<DIR>(q, S, gam, out);
#pragma unroll
  for (int v = 0; v < 8; v++) out[v] *= G.sg;
}

// ---------------------------------------------------------------------------------------------------------
// Fast-magnetosonic bounds from the quadratic dispersion relation (eqs. 18-19): the roots
// cp >= cm of A v^2 + B v + C = 0.  c_ms^2 = v_a^2 + c_s^2 (1 - v_a^2) = (b^2 + gam p) / (b^2 + w).
// A = (u^t)^2 (1 - c_ms^2) - c_ms^2 g^tt > 0 because g^tt < 0 everywhere in Kerr-Schild coordinates, so the
// "+" root is the larger one.  A29: a negative discriminant is clamped to zero.
// ---------------------------------------------------------------------------------------------------------
// ONLY_MAX: return in cp the larger of (cp, -cm, 0) = (|B/2| + sqrt(disc)) / A, which is all eq. 17 needs (the same
// floating-point value as taking the maximum of the two roots' magnitudes); cm is then not set.
template <int DIR, bool ONLY_MAX = false>
__device__ __forceinline__ void wave_speeds(const double q[8], const State& S, const Geom& G, double gam, double& cp,
                                            double& cm) {
  // c_ms^2 = N / D with N = b^2 + gam p, D = b^2 + w (eqs. 18-19).  The quadratic is homogeneous in its
  // coefficients, so it is scaled by D > 0 and c_ms^2 is never formed: A = (D - N) (u^t)^2 - N g^tt, ...
  const double pg = (gam - 1.0) * q[1];
  const double w = q[0] + q[1] + pg;
  const double N = fma(gam, pg, S.bsq);
  const double DmN = (S.bsq + w) - N;
  const double ut = S.u0;
  const double ud = pick(DIR, S.u0, S.u1, S.u2, S.u3);
  const double gdd = DIR == 1 ? G.c11 : (DIR == 2 ? G.c22 : G.c33);
  const double A = fma(DmN * ut, ut, -N * G.c00);
  const double hB = DIR == 1 ? fma(DmN * ut, ud, -N * G.c01) : (DmN * ut) * ud;  // = -B/2; g^{t2} = g^{t3} = 0
  const double C = fma(DmN * ud, ud, -N * gdd);
  double disc = fma(hB, hB, -A * C);             // (B^2 - 4AC)/4
  disc = disc > 1e-300 ? disc : 1e-300;
  const double sq = disc * frsqrt(disc);
  const double iA = frcp(A);
  if (ONLY_MAX) {
    cp = (fabs(hB) + sq) * iA;
  } else {
    cp = (hB + sq) * iA;
    cm = (hB - sq) * iA;
  }
}

// ---------------------------------------------------------------------------------------------------------
// Reconstruction.  The fp64 pipe and the issue slots bound the flux kernels, so the limiter
// is written for the fewest fp64 instructions; every form below equals the paper's in exact arithmetic and
// differs from the literal transcription by rounding only.
//
// MC-limited slope, eq. 15 (A2: the last branch is signed), from the two one-sided differences
// dm = q_I - q_{I-1}, dp = q_{I+1} - q_I.  Returned DOUBLED: 2 dq = minmod(4 dm, 4 dp, dm + dp)  (scaling by a
// power of two is exact).  "dm dp < 0" is read off the sign bits; when one of them is zero the minmod is zero anyway.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double same_sign_factor(double a, double b, int hi_one) {
  // the double whose high word is hi_one (low word 0) if a and b carry the same sign bit, else +0.0
  const int x = __double2hiint(a) ^ __double2hiint(b);
  return __hiloint2double(~(x >> 31) & hi_one, 0);
}

__device__ __forceinline__ double slope2_mc(double dm, double dp) {
  const double sum = dm + dp;
  const double one = fabs(dm) < fabs(dp) ? dm : dp;              // the smaller one-sided difference
  const double four = one * same_sign_factor(dm, dp, 0x40100000);  // 4 one, or 0 at an extremum
  return fabs(four) < fabs(sum) ? four : sum;
}

// PLM face values of a cell from its doubled slope (eq. 16): q -+ dq/2
__device__ __forceinline__ void plm_faces(double y, double s2, double& l, double& r) {
  l = fma(-0.25, s2, y);
  r = fma(0.25, s2, y);
}

// PPM (A20): 4th-order edge value between cells 0 and 1 from their values and DOUBLED MC slopes:
// (y0 + y1)/2 - (dq1 - dq0)/6 ...
__device__ __forceinline__ double ppm_edge(double y0, double y1, double s20, double s21) {
  return fma(-1.0 / 12.0, s21 - s20, 0.5 * (y0 + y1));
}
// the same with the difference d01 = y1 - y0 at hand: (y0 + y1)/2 = y0 + d01/2, one instruction less
__device__ __forceinline__ double ppm_edge_d(double y0, double d01, double s20, double s21) {
  return fma(-1.0 / 12.0, s21 - s20, fma(0.5, d01, y0));
}

// ... and the monotonisation of the parabola of a cell with value y and edge values l (lower), r (upper).
// With a = r - y, b = y - l the three cases of Colella-Woodward eq. 1.10 are: a b <= 0 -> l = r = y;
// |b| > 2|a| -> l = 3y - 2r = y - 2a;  |a| > 2|b| -> r = 3y - 2l = y + 2b.  Hence l = y - min(|b|, 2|a|) sgn(b),
// r = y + min(|a|, 2|b|) sgn(a) for a b > 0 (a zero a or b gives l = r = y through the min), else l = r = y.
__device__ __forceinline__ void ppm_mono(double y, double& l, double& r) {
  const double a = r - y, b = y - l;
  const double a2 = a + a, b2 = b + b;
  const double bp = fabs(b) < fabs(a2) ? b : a2;
  const double ap = fabs(a) < fabs(b2) ? a : b2;
  const double f = same_sign_factor(a, b, 0x3ff00000);  // 1 or 0
  l = fma(-f, bp, y);
  r = fma(f, ap, y);
}

// ---------------------------------------------------------------------------------------------------------
// Riemann flux at one face from the two reconstructed states and the FACE metric.
// RIEMANN 0: local Lax-Friedrichs, eq. 17.  RIEMANN 1: HLL, eq. 20 (A30: guarded denominator).
// sqrt(-g) multiplies the combination once (it is common to U^l, U^r, F^l, F^r at a face).
// ---------------------------------------------------------------------------------------------------------
// One side's contribution F^d + c U (both divided by sqrt(-g)) formed in one go: with uh = u^d + c u^t and
// bh = b^d + c b^t,  [0] rho uh;  [1..4] (w + b^2) uh u_nu + (p + b^2/2)(delta^d_nu + c delta^t_nu) - bh b_nu;
// [5..7] b^i uh - bh u^i  (= c B^d for i = d).  Algebraically the same as flux_hat<DIR> + c flux_hat<0>.
template <int DIR>
__device__ __forceinline__ void side_flux(const double q[8], const State& S, double gam, double c, double out[8]) {
  const double pg = (gam - 1.0) * q[1];
  const double w = q[0] + q[1] + pg;
  const double ptot = fma(0.5, S.bsq, pg);
  const double ud = pick(DIR, S.u0, S.u1, S.u2, S.u3);
  const double bd = pick(DIR, S.b0, S.b1, S.b2, S.b3);
  const double uh = fma(c, S.u0, ud), bh = fma(c, S.b0, bd);
  const double e = (w + S.bsq) * uh;
  out[0] = q[0] * uh;
  double t0 = fma(c, ptot, fma(e, S.l0, -bh * S.m0));
  double t1 = fma(e, S.l1, -bh * S.m1);
  double t2 = fma(e, S.l2, -bh * S.m2);
  double t3 = fma(e, S.l3, -bh * S.m3);
  if (DIR == 1) t1 += ptot;
  if (DIR == 2) t2 += ptot;
  if (DIR == 3) t3 += ptot;
  out[1] = t0;
  out[2] = t1;
  out[3] = t2;
  out[4] = t3;
  out[5] = DIR == 1 ? c * q[5] : fma(S.b1, uh, -bh * S.u1);
  out[6] = DIR == 2 ? c * q[6] : fma(S.b2, uh, -bh * S.u2);
  out[7] = DIR == 3 ? c * q[7] : fma(S.b3, uh, -bh * S.u3);
}

template <int DIR, int RIEMANN>
__device__ __forceinline__ void face_flux(const double pl[8], const double pr[8], const Geom& G, double gam, double F[8],
                                          double& cw) {
  State Sl, Sr;
  double Hl[8], Hr[8], cpl, cml = 0.0, cpr, cmr = 0.0;
  fluid_state(pl, G, Sl);
  fluid_state(pr, G, Sr);
  wave_speeds<DIR, RIEMANN == 0>(pl, Sl, G, gam, cpl, cml);
  wave_speeds<DIR, RIEMANN == 0>(pr, Sr, G, gam, cpr, cmr);
  double cmax = 0.0, cmin = 0.0;
  if (RIEMANN == 0) {
    cw = fmax(cpl, cpr);  // = max(c_max, c_min) of P:L154: each side's bound is already max(c_1, -c_2) >= 0
  } else {
    cmax = fmax(0.0, fmax(cpr, cpl));
    cmin = fmax(0.0, fmax(-cmr, -cml));
    cw = fmax(cmax, cmin);
  }
  if (RIEMANN == 0) {
    // eq. 17: (F^l + F^r - c_w (U^r - U^l))/2 = ((F^l + c_w U^l) + (F^r - c_w U^r))/2
    side_flux<DIR>(pl, Sl, gam, cw, Hl);
    side_flux<DIR>(pr, Sr, gam, -cw, Hr);
    const double hsg = 0.5 * G.sg;
#pragma unroll
    for (int v = 0; v < 8; v++) F[v] = hsg * (Hl[v] + Hr[v]);
  } else {
    // eq. 20: (c_max F^l + c_min F^r - c_max c_min (U^r - U^l)) / (c_max + c_min)
    //       = (c_max (F^l + c_min U^l) + c_min (F^r - c_max U^r)) / (c_max + c_min)
    side_flux<DIR>(pl, Sl, gam, cmin, Hl);
    side_flux<DIR>(pr, Sr, gam, -cmax, Hr);
    const double sc = G.sg * frcp(fmax(cmax + cmin, 1e-300));
    const double wl = sc * cmax, wr = sc * cmin;
#pragma unroll
    for (int v = 0; v < 8; v++) F[v] = fma(wl, Hl[v], wr * Hr[v]);
  }
}

// ---------------------------------------------------------------------------------------------------------
// Geometric source S_nu = sqrt(-g) T^kappa_lambda Gamma^lambda_{nu kappa} (eq. 7; eq. 14),
// evaluated as (1/2) sqrt(-g) T^{kl} d_nu g_{kl} (identical: T^{kl} is symmetric, see source_weights in
// cuharm_geom.cuh).  sw: the 14 precomputed weights of this (i, j): sqrt(-g) x (1/2 | 1) x d_nu g_e for nu = 1, 2 and
// e over the metric entries 00 01 03 11 13 22 33.  nu = t and nu = phi vanish identically (the metric depends on
// neither: energy and angular-momentum conservation) and are not formed.  src = (S_t, S_1, S_2, S_3).
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void source_term(const double q[8], const State& S, const Geom& G, const double* sw, double gam,
                                            double src[4]) {
  const double pg = (gam - 1.0) * q[1];
  const double w = q[0] + q[1] + pg;
  const double eta = w + S.bsq;
  const double ptot = fma(0.5, S.bsq, pg);
  const double e0 = eta * S.u0, e1 = eta * S.u1, e2 = eta * S.u2, e3 = eta * S.u3;
  // T^{kl} = (w + b^2) u^k u^l + (p + b^2/2) g^{kl} - b^k b^l  (eq. 5), the 7 entries that meet a non-zero d g_{kl}
  const double T00 = fma(e0, S.u0, fma(ptot, G.c00, -S.b0 * S.b0));
  const double T01 = fma(e0, S.u1, fma(ptot, G.c01, -S.b0 * S.b1));
  const double T03 = fma(e0, S.u3, -S.b0 * S.b3);  // g^{t phi} = 0
  const double T11 = fma(e1, S.u1, fma(ptot, G.c11, -S.b1 * S.b1));
  const double T13 = fma(e1, S.u3, fma(ptot, G.c13, -S.b1 * S.b3));
  const double T22 = fma(e2, S.u2, fma(ptot, G.c22, -S.b2 * S.b2));
  const double T33 = fma(e3, S.u3, fma(ptot, G.c33, -S.b3 * S.b3));
  src[0] = 0.0;
  src[1] = fma(T00, sw[0], fma(T01, sw[1], fma(T03, sw[2], fma(T11, sw[3], fma(T13, sw[4], fma(T22, sw[5], T33 * sw[6]))))));
  src[2] = fma(T00, sw[7], fma(T01, sw[8], fma(T03, sw[9], fma(T11, sw[10], fma(T13, sw[11], fma(T22, sw[12], T33 * sw[13]))))));
  src[3] = 0.0;
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

__device__ __forceinline__ int invert_2d(const double U[8], const Geom& G, double gam, double q[8], NewtonCfg nc, int& iters) {
  iters = 0;
  const double a = G.alpha;
  const double isg = G.isg;
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
  if (!fin || !(D > 0.0) || !(isg > 0.0)) return 1;
  // Q^mu = g^{mu nu} Q_nu  (g^{t phi} = 0)
  const double Qc0 = G.c00 * Q0 + G.c01 * Q1;
  const double Qc1 = G.c01 * Q0 + G.c11 * Q1 + G.c13 * Q3;
  const double Qc2 = G.c22 * Q2;
  const double Qc3 = G.c13 * Q1 + G.c33 * Q3;
  const double Bsq = G.g11 * Bc1 * Bc1 + G.g22 * Bc2 * Bc2 + G.g33 * Bc3 * Bc3 + 2.0 * (G.g13 * Bc1 * Bc3);
  const double QdB = Q1 * Bc1 + Q2 * Bc2 + Q3 * Bc3;
  // n_mu = (-alpha,0,0,0); n^mu = (1/alpha, -alpha g^{ti})
  const double n1 = -G.ac01;
  const double Qdn = fma(Q0, G.ialpha, Q1 * n1);
  const double Qsq = Qc0 * Q0 + Qc1 * Q1 + Qc2 * Q2 + Qc3 * Q3;
  const double Qtsq = fma(Qdn, Qdn, Qsq);
  const double QdB2 = QdB * QdB;
  const double igam = frcp(gam);
  const double gfac = (gam - 1.0) * igam;
  // initial guess: W = Gamma^2 w from the guess, v^2 from eq. 29 at that W
  const double qsq = G.g11 * g1 * g1 + G.g22 * g2 * g2 + G.g33 * g3 * g3 + 2.0 * (G.g13 * g1 * g3);
  double W = (1.0 + qsq) * fma(gam, gu, grho);
  if (!(W > 0.0) || !isfinite(W)) return 3;
  double v2 = 0.0;
  for (int t = 0; t < 400; t++) {
    const double iW = frcp(W), iBW = frcp(Bsq + W);
    v2 = fma(QdB2 * fma(2.0, W, Bsq), iW * iW, Qtsq) * (iBW * iBW);
    if (v2 < 1.0 || !(W < 1e300)) break;
    W *= 10.0;
  }
  if (!(v2 < 1.0)) return 3;
  v2 = v2 < 0.0 ? 0.0 : v2;
  // One Newton update of (W, v^2); returns whether |dW/W| <= tol held for this update.
  auto newton_step = [&]() {
    const double iW = frcp(W);
    const double iW2 = iW * iW, iW3 = iW2 * iW;
    const double omv = 1.0 - v2;
    const double isq = frsqrt(omv);
    const double sq = omv * isq;
    const double BW = Bsq + W;
    const double pg = gfac * fma(W, omv, -D * sq);                                  // eq. 31
    const double f1 = fma(QdB2 * fma(2.0, W, Bsq), iW2, fma(-v2 * BW, BW, Qtsq));    // eq. 29
    const double f2 = fma(0.5 * QdB2, iW2, fma(-0.5 * Bsq, 1.0 + v2, -Qdn)) - W + pg;  // eq. 30 (A6)
    const double j11 = -2.0 * BW * fma(QdB2, iW3, v2);
    const double j12 = -BW * BW;
    const double j21 = fma(gfac, omv, fma(-QdB2, iW3, -1.0));
    const double j22 = fma(gfac, fma(0.5 * D, isq, -W), -0.5 * Bsq);
    const double idet = frcp(fma(j11, j22, -j12 * j21));
    const double dW = fma(f2, j12, -f1 * j22) * idet;
    const double dv = fma(f1, j21, -f2 * j11) * idet;
    const double Wn = fabs(W + dW);
    double vn = v2 + dv;
    vn = vn < 0.0 ? 0.0 : vn;
    vn = vn > 1.0 - 1e-15 ? 1.0 - 1e-15 : vn;
    W = Wn;
    v2 = vn;
    return (Wn == 0.0) ? (fabs(dW) <= nc.tol) : (fabs(dW) <= nc.tol * Wn);  // |dW/W| <= tol
  };
  // iterate to the criterion (the only data-dependent branch), then `extra` more updates, all within maxit; a
  // non-finite iterate never meets the criterion, so finiteness is tested once, after the loops
  int it = 1;
  bool small = false;
  for (; it <= nc.maxit; it++) {
    small = newton_step();
    if (small) break;
  }
  int more = 0;
  if (small) {
    more = min(nc.extra, nc.maxit - it);
    for (int e = 0; e < more; e++) newton_step();
    it += more;
  }
  iters = it > nc.maxit ? nc.maxit : it;
  if (!isfinite(W) || !isfinite(v2) || W == 0.0) return 3;
  if (!small || more < nc.extra) return 2;
  if (!(W > 0.0)) return 3;
  if (!(v2 >= 0.0 && v2 < 1.0)) return 4;
  const double omv = 1.0 - v2;
  const double lor = frsqrt(omv);
  const double rho = D * (omv * lor);  // D / Gamma
  const double w = W * omv;
  const double u = (w - rho) * igam;
  if (!(rho > 0.0)) return 5;
  if (!(u >= 0.0)) return 6;
  q[0] = rho;
  q[1] = u;
  const double f = lor * frcp(W + Bsq);
  const double QdBW = QdB * frcp(W);
  q[2] = f * (fma(n1, Qdn, Qc1) + QdBW * Bc1);  // ut^i = Gamma [Qt^i + (Q.B) B^i / W] / (W + B^2)
  q[3] = f * fma(QdBW, Bc2, Qc2);
  q[4] = f * fma(QdBW, Bc3, Qc3);
  return 0;
}

// out-of-line copy for rare paths (the ceiling re-inversion)
__device__ __noinline__ int invert_2d_cold(const double* U, const Geom* Gp, double gam, double* q, NewtonCfg nc) {
  int its;
  const Geom G = load_geom(Gp, 0);
  return invert_2d(U, G, gam, q, nc, its);
}

// ---------------------------------------------------------------------------------------------------------
// Floors and ceilings (eqs. 35-37; A9-A12).  rfl, ufl: the eq. 35 profiles of this (i,j).
// Bit mask returned: 1 rho floor, 2 u floor, 4 ceiling applied, 8 Lorentz cap, 16 ceiling re-inversion failed.
// ---------------------------------------------------------------------------------------------------------
struct FloorCfg {
  double sigma_max, b2_over_u_max, gamma_max;
  double isigma, ib2u;  // reciprocals of the two ceilings (host-computed; 0 when the ceiling is disabled)
};

// rare path of the ceilings: mass / energy injected at rest in the normal-observer frame, re-inversion (A11)
__device__ __noinline__ int apply_ceilings_cold(double* q, const Geom* Gp, double drho, double du, FloorCfg fc, double gam,
                                                NewtonCfg nc) {
  const Geom G = load_geom(Gp, 0);
  int mask = 4;
  State S;
  fluid_state(q, G, S);
  double U[8], Ua[8];
  flux_vector<0>(q, S, G, gam, U);
  double qa[8] = {drho, du, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
  State Sa;
  fluid_state(qa, G, Sa);
  flux_vector<0>(qa, Sa, G, gam, Ua);
  for (int v = 0; v < 8; v++) U[v] += Ua[v];
  double t[8];
  for (int v = 0; v < 8; v++) t[v] = q[v];
  const int flag = invert_2d_cold(U, Gp, gam, t, nc);
  if (flag == 0) {
    for (int v = 0; v < 5; v++) q[v] = t[v];
  } else {
    q[0] += drho;
    q[1] += du;
    mask |= 16;
  }
  State S2;
  fluid_state(q, G, S2);
  if (fc.sigma_max > 0.0) q[0] = fmax(q[0], S2.bsq * fc.isigma);
  if (fc.b2_over_u_max > 0.0) q[1] = fmax(q[1], S2.bsq * fc.ib2u);
  return mask;
}

__device__ __forceinline__ int apply_floors(double q[8], const Geom& G, const Geom* Gp, double rfl, double ufl, FloorCfg fc,
                                            double gam, NewtonCfg nc) {
  int mask = 0;
  if (q[0] < rfl) { q[0] = rfl; mask |= 1; }
  if (q[1] < ufl) { q[1] = ufl; mask |= 2; }
  const double qsq = gamma_sq_minus_one(q, G);
  if (fc.sigma_max > 0.0 || fc.b2_over_u_max > 0.0) {
    // b^2 = (g_ij B^i B^j + (b^t)^2) / (u^t)^2 with b^t = B^i u_i  (from b^i = (B^i + b^t u^i)/u^t and b.u = 0)
    const double lor2 = 1.0 + qsq;
    const double lor = lor2 * frsqrt(lor2);
    const double u0 = lor * G.ialpha;
    const double u1 = fma(-lor, G.ac01, q[2]);
    const double l1 = G.g01 * u0 + G.g11 * u1 + G.g13 * q[4];
    const double l2 = G.g22 * q[3];
    const double l3 = G.g03 * u0 + G.g13 * u1 + G.g33 * q[4];
    const double bt = q[5] * l1 + q[6] * l2 + q[7] * l3;
    const double B2 = G.g11 * q[5] * q[5] + G.g22 * q[6] * q[6] + G.g33 * q[7] * q[7] + 2.0 * (G.g13 * q[5] * q[7]);
    const double bsq = fma(bt, bt, B2) * (G.alpha * G.alpha) * frcp(lor2);
    double drho = 0.0, du = 0.0;
    if (fc.sigma_max > 0.0) drho = fmax(0.0, fma(bsq, fc.isigma, -q[0]));
    if (fc.b2_over_u_max > 0.0) du = fmax(0.0, fma(bsq, fc.ib2u, -q[1]));
    if (drho > 0.0 || du > 0.0) {
      // the out-of-line rare path works on a copy, so that only the copy's address escapes and q stays in registers
      double t[8];
#pragma unroll
      for (int v = 0; v < 8; v++) t[v] = q[v];
      mask |= apply_ceilings_cold(t, Gp, drho, du, fc, gam, nc);
#pragma unroll
      for (int v = 0; v < 8; v++) q[v] = t[v];
    }
  }
  if (fc.gamma_max > 0.0) {
    const double q2 = (mask & 4) ? gamma_sq_minus_one(q, G) : qsq;
    if (q2 > fc.gamma_max * fc.gamma_max - 1.0) {
      const double f = sqrt((fc.gamma_max * fc.gamma_max - 1.0) / q2);  // A12
      q[2] *= f; q[3] *= f; q[4] *= f;
      mask |= 8;
    }
  }
  return mask;
}

}  // namespace cuharm
