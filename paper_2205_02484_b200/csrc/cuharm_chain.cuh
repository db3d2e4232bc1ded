// cuharm_chain.cuh — the inversion fallback chain of P:L229-239 as a sparse follow-up of the update kernel
// (SURVEY 8(f)1): for the zones the 2D Newton-Raphson method failed in, and for the strongly magnetised zones of
// eq. 33, the 1D method for W and the entropy method (eq. 32 put into eq. 29; eq. 11 advanced for
// those zones only), both solved by Brent's method.  Cold code: it runs over the (short) list the update kernel
// leaves behind, one thread per listed zone, so nothing here is written for speed.  fp64 throughout; pow() is the
// CUDA math library's.  Shares nothing with oracle/.
#pragma once
#include "cuharm_flux.cuh"

namespace cuharm {

struct ChainCfg {
  int on;          // inv_chain
  int brent_maxit;
  double beta_min, brent_tol;
};

// code the update kernel leaves in flag[] for a zone of eq. 33 (entropy method first and only)
constexpr int KIND_ENTROPY_FIRST = 100;

// The Noble variables of eqs. 27-28 at a zone centre.  `momentum_only`: Qtilde^i and Qtilde^2 through the spatial
// inverse metric gamma^{ij} = g^{ij} - g^{ti} g^{tj} / g^{tt} acting on Q_j alone -- "(Qtilde)^2 is independent on
// Qtilde^0" -- so the energy variable, which is what cannot be trusted when the entropy method is called,
// does not enter.
struct NobleVars {
  double D, Qtsq, Bsq, QdB, Qdn;
  double Qt1, Qt2, Qt3;  // Qtilde^i
  double Bc1, Bc2, Bc3;  // script-B^i
  bool finite;
};

__device__ inline void noble_setup(const double U[8], const Geom& G, bool momentum_only, NobleVars& N) {
  const double f = G.alpha / G.sg;
  N.D = f * U[0];
  const double Q0 = f * U[1], Q1 = f * U[2], Q2 = f * U[3], Q3 = f * U[4];
  N.Bc1 = f * U[5]; N.Bc2 = f * U[6]; N.Bc3 = f * U[7];
  N.Bsq = G.g11 * N.Bc1 * N.Bc1 + G.g22 * N.Bc2 * N.Bc2 + G.g33 * N.Bc3 * N.Bc3 + 2.0 * G.g13 * N.Bc1 * N.Bc3;
  N.QdB = Q1 * N.Bc1 + Q2 * N.Bc2 + Q3 * N.Bc3;
  const bool fin3 = isfinite(N.D) && isfinite(Q1) && isfinite(Q2) && isfinite(Q3) && isfinite(N.Bc1) && isfinite(N.Bc2) &&
                    isfinite(N.Bc3);
  if (momentum_only) {
    N.finite = fin3;
    N.Qdn = 0.0;
    N.Qt1 = (G.c11 - G.c01 * G.c01 / G.c00) * Q1 + G.c13 * Q3;   // g^{t2} = g^{t3} = 0 in Kerr-Schild coordinates
    N.Qt2 = G.c22 * Q2;
    N.Qt3 = G.c13 * Q1 + G.c33 * Q3;
    N.Qtsq = N.Qt1 * Q1 + N.Qt2 * Q2 + N.Qt3 * Q3;
  } else {
    N.finite = fin3 && isfinite(Q0);
    const double n0 = 1.0 / G.alpha, n1 = -G.alpha * G.c01;       // n^mu = (1/alpha, -alpha g^{ti})
    N.Qdn = Q0 * n0 + Q1 * n1;
    const double Qc0 = G.c00 * Q0 + G.c01 * Q1;
    const double Qc1 = G.c01 * Q0 + G.c11 * Q1 + G.c13 * Q3;
    const double Qc2 = G.c22 * Q2;
    const double Qc3 = G.c13 * Q1 + G.c33 * Q3;
    N.Qtsq = (Qc0 * Q0 + Qc1 * Q1 + Qc2 * Q2 + Qc3 * Q3) + N.Qdn * N.Qdn;
    N.Qt1 = Qc1 + n1 * N.Qdn;
    N.Qt2 = Qc2;
    N.Qt3 = Qc3;
  }
}

// residual of eq. 29 at (W, v^2)
__device__ inline double eq29_residual(const NobleVars& N, double W, double v2) {
  const double BW = N.Bsq + W;
  return N.Qtsq - v2 * BW * BW + N.QdB * N.QdB * (N.Bsq + 2.0 * W) / (W * W);
}

// rho, u, utilde^i from (W, v^2); u_fixed >= 0 replaces the energy-based u (entropy method).
// Returns 0 or a failure code of invert_2d (3 W, 4 v^2, 5 rho, 6 u).
__device__ inline int prims_from_Wv2(const NobleVars& N, double gam, double W, double v2, bool have_u, double u_fixed, double q[8]) {
  if (!(W > 0.0) || !isfinite(W)) return 3;
  if (!(v2 >= 0.0 && v2 < 1.0)) return 4;
  const double lor = 1.0 / sqrt(1.0 - v2);
  const double rho = N.D / lor;
  const double u = have_u ? u_fixed : (W * (1.0 - v2) - rho) / gam;
  if (!(rho > 0.0)) return 5;
  if (!(u >= 0.0)) return 6;
  q[0] = rho;
  q[1] = u;
  const double den = W + N.Bsq, k = N.QdB / W;
  q[2] = lor * (N.Qt1 + k * N.Bc1) / den;
  q[3] = lor * (N.Qt2 + k * N.Bc2) / den;
  q[4] = lor * (N.Qt3 + k * N.Bc3) / den;
  return 0;
}

// Brent's root finder (R. P. Brent 1973, ch. 4: inverse quadratic interpolation / secant with bisection safeguard) on
// a bracket [xa, xb] with f(xa) f(xb) <= 0.  Convergence: half the bracket <= |x| (2 eps + tol/2), or an exact zero.
// A40: the paper only names the method; tol is a parameter (1e-14 in the workloads).
template <class Fn>
__device__ inline bool brent_root(Fn f, double xa, double xb, double ya, double yb, double tol, int maxit, double& root) {
  if (!(ya * yb <= 0.0)) return false;
  const double eps = 2.220446049250313e-16;
  double xc = xa, yc = ya, step = xb - xa, prev = step;
  for (int it = 0; it < maxit; it++) {
    if ((yb > 0.0 && yc > 0.0) || (yb < 0.0 && yc < 0.0)) { xc = xa; yc = ya; step = xb - xa; prev = step; }
    if (fabs(yc) < fabs(yb)) { xa = xb; xb = xc; xc = xa; ya = yb; yb = yc; yc = ya; }
    const double t1 = fabs(xb) * (2.0 * eps + 0.5 * tol);
    const double half = 0.5 * (xc - xb);
    if (fabs(half) <= t1 || yb == 0.0) { root = xb; return true; }
    bool bisect = true;
    if (fabs(prev) >= t1 && fabs(ya) > fabs(yb)) {
      const double s = yb / ya;
      double p, q;
      if (xa == xc) {  // secant
        p = 2.0 * half * s;
        q = 1.0 - s;
      } else {         // inverse quadratic
        const double qa = ya / yc, r = yb / yc;
        p = s * (2.0 * half * qa * (qa - r) - (xb - xa) * (r - 1.0));
        q = (qa - 1.0) * (r - 1.0) * (s - 1.0);
      }
      if (p > 0.0) q = -q;
      p = fabs(p);
      const double lim1 = 3.0 * half * q - fabs(t1 * q), lim2 = fabs(prev * q);
      if (2.0 * p < fmin(lim1, lim2)) { prev = step; step = p / q; bisect = false; }
    }
    if (bisect) { step = half; prev = half; }
    xa = xb; ya = yb;
    xb += fabs(step) > t1 ? step : (half >= 0.0 ? t1 : -t1);
    yb = f(xb);
    if (!isfinite(yb)) return false;
  }
  return false;
}

// The 1D method: v^2 expressed from eq. 30 and put into eq. 29, which is solved for W by Brent.
// With s = sqrt(1 - v^2) and eq. 31, eq. 30 (A6) reads (B^2/2 + g W) s^2 - g D s + [-Q.n - B^2 + (Q.B)^2/(2 W^2) - W]
// = 0, g = (gam-1)/gam; the physical s is the root with the plus sign.  Bracket (A41): from W0 = Gamma^2 w
// of the guess double W until the residual is defined and positive; halve from there until it is negative or
// undefined; where the quadratic has no real root the residual is continued by minus its value at the upper end.
__device__ inline bool v2_of_W(const NobleVars& N, double gam, double W, double& v2) {
  const double g = (gam - 1.0) / gam;
  const double A = 0.5 * N.Bsq + g * W, B = -g * N.D;
  const double C = -N.Qdn - N.Bsq + N.QdB * N.QdB / (2.0 * W * W) - W;
  const double disc = B * B - 4.0 * A * C;
  if (!(disc >= 0.0) || !(A > 0.0)) return false;
  const double s = (-B + sqrt(disc)) / (2.0 * A);
  v2 = 1.0 - s * s;
  return isfinite(v2);
}

__device__ inline int invert_1dw_dev(const double U[8], const Geom& G, double gam, double q[8], double tol, int maxit) {
  const double qsq = gamma_sq_minus_one(q, G);
  const double W0 = (1.0 + qsq) * (q[0] + gam * q[1]);
  q[5] = U[5] / G.sg; q[6] = U[6] / G.sg; q[7] = U[7] / G.sg;
  NobleVars N;
  noble_setup(U, G, false, N);
  if (!N.finite || !(N.D > 0.0)) return 1;
  if (!(W0 > 0.0) || !isfinite(W0)) return 3;
  const double nan = __longlong_as_double(0x7ff8000000000000LL);
  auto res = [&](double W) { double v2; return v2_of_W(N, gam, W, v2) ? eq29_residual(N, W, v2) : nan; };
  double wb = W0, yb = res(wb);
  for (int k = 0; k < 60 && !(isfinite(yb) && yb > 0.0); k++) { wb *= 2.0; yb = res(wb); }
  if (!(isfinite(yb) && yb > 0.0)) return 2;
  const double below = -yb;
  auto rext = [&](double W) { const double r = res(W); return isfinite(r) ? r : below; };
  double wa = 0.5 * wb, ya = rext(wa);
  for (int k = 0; k < 60 && ya > 0.0; k++) { wa *= 0.5; ya = rext(wa); }
  if (ya > 0.0) return 2;
  double W, v2;
  if (!brent_root(rext, wa, wb, ya, yb, tol, maxit, W)) return 2;
  if (!v2_of_W(N, gam, W, v2)) return 2;
  return prims_from_Wv2(N, gam, W, v2, false, 0.0, q);
}

// The entropy method (eq. 32; A36: eq. 32's S is the conserved calS = Gamma S = alpha U_S / sqrt(-g),
// S = p_g / rho^(gam-1)): W(v^2) = Gamma D + Gamma gam/(gam-1) (D/Gamma)^(gam-1) calS in eq. 29, solved for
// v^2 on [0, 1 - 1e-15] by Brent.  Returns 0, 1 (D <= 0, calS <= 0, non-finite input), 2 (no root found), 3..6.
__device__ inline int invert_entropy_dev(const double U[8], double US, const Geom& G, double gam, double q[8], double tol,
                                         int maxit) {
  q[5] = U[5] / G.sg; q[6] = U[6] / G.sg; q[7] = U[7] / G.sg;
  NobleVars N;
  noble_setup(U, G, true, N);
  const double calS = G.alpha * US / G.sg;
  if (!N.finite || !isfinite(calS) || !(N.D > 0.0) || !(calS > 0.0)) return 1;
  const double gg = gam / (gam - 1.0);
  auto W_of = [&](double v2) {
    const double lor = 1.0 / sqrt(1.0 - v2);
    return lor * N.D + lor * gg * pow(N.D / lor, gam - 1.0) * calS;  // eq. 32
  };
  auto res = [&](double v2) { return eq29_residual(N, W_of(v2), v2); };
  const double xa = 0.0, xb = 1.0 - 1e-15;
  const double ya = res(xa), yb = res(xb);
  if (!isfinite(ya) || !isfinite(yb)) return 2;
  double v2 = 0.0;
  if (ya != 0.0 && !brent_root(res, xa, xb, ya, yb, tol, maxit, v2)) return 2;
  const double lor = 1.0 / sqrt(1.0 - v2);
  const double rho = N.D / lor;
  const double pg = (calS / lor) * pow(rho, gam - 1.0);
  return prims_from_Wv2(N, gam, W_of(v2), v2, true, pg / (gam - 1.0), q);
}

// ---------------------------------------------------------------------------------------------------------
// Entropy flux of eq. 11 through the lower DIR-face of zone (i, j, k): the same Riemann combination
// (eq. 17 / eq. 20) of the same two reconstructed states with the same wave speeds as the other eight fluxes, for
// the conserved variable sqrt(-g) S u^t with flux sqrt(-g) S u^DIR.  Recomputed here for the six faces of a listed
// zone instead of being stored for every face of the grid.
// ---------------------------------------------------------------------------------------------------------
template <int RECON>
__device__ inline void cell_edges(const double* y, long long sd, double& lo, double& hi) {
  // limited lower / upper edge values of the cell at y (eq. 16; PPM: A20)
  if (RECON == 0) {
    plm_faces(y[0], slope2_mc(y[0] - y[-sd], y[sd] - y[0]), lo, hi);
  } else {
    const double d21 = y[-sd] - y[-2 * sd], d10 = y[0] - y[-sd], d01 = y[sd] - y[0], d12 = y[2 * sd] - y[sd];
    const double sm = slope2_mc(d21, d10), s0 = slope2_mc(d10, d01), sp = slope2_mc(d01, d12);
    lo = ppm_edge(y[-sd], y[0], sm, s0);
    hi = ppm_edge(y[0], y[sd], s0, sp);
    ppm_mono(y[0], lo, hi);
  }
}

__device__ inline double entropy_density(double rho, double u, double gam) { return (gam - 1.0) * u / pow(rho, gam - 1.0); }

template <int DIR, int RECON, int RIEMANN>
__device__ inline double entropy_face_flux(const double* P, long long nz, long long idx, long long sd, const Geom& G, double gam) {
  double pl[8], pr[8];
#pragma unroll
  for (int v = 0; v < 8; v++) {
    double lo, hi;
    cell_edges<RECON>(P + v * nz + idx - sd, sd, lo, hi);
    pl[v] = hi;
    cell_edges<RECON>(P + v * nz + idx, sd, lo, hi);
    pr[v] = lo;
  }
  State Sl, Sr;
  fluid_state(pl, G, Sl);
  fluid_state(pr, G, Sr);
  double cpl, cml, cpr, cmr;
  wave_speeds<DIR, false>(pl, Sl, G, gam, cpl, cml);
  wave_speeds<DIR, false>(pr, Sr, G, gam, cpr, cmr);
  const double cmax = fmax(0.0, fmax(cpr, cpl)), cmin = fmax(0.0, fmax(-cmr, -cml));
  const double sl = entropy_density(pl[0], pl[1], gam), sr = entropy_density(pr[0], pr[1], gam);
  const double udl = pick(DIR, Sl.u0, Sl.u1, Sl.u2, Sl.u3), udr = pick(DIR, Sr.u0, Sr.u1, Sr.u2, Sr.u3);
  const double ul = G.sg * sl * Sl.u0, ur = G.sg * sr * Sr.u0;
  const double fl = G.sg * sl * udl, fr = G.sg * sr * udr;
  if (RIEMANN == 0) {
    const double cw = fmax(cmax, cmin);
    return 0.5 * (fl + fr - cw * (ur - ul));  // eq. 17
  }
  return (cmax * fl + cmin * fr - cmax * cmin * (ur - ul)) / fmax(cmax + cmin, 1e-300);  // eq. 20
}

struct ChainArgs {
  Dims d;
  const double* Pflux;  // state the fluxes of this substep were built from
  double* Pout;         // fluid primitives of a listed zone still hold P^n (the Newton guess); B is already updated
  const Geom *C, *F1g, *F2g;
  const double* floors;
  int* flag;             // in: the 2D method's failure code, or KIND_ENTROPY_FIRST; out: the chain's verdict
  const int* list;
  const double* ustar;   // [8][nz]: the updated conserved variables U* of the listed zones, as the update kernel formed them
  const unsigned long long* nfail;
  unsigned long long* nbad;   // zones still failed afterwards
  unsigned long long* stats;  // [8] of cuharm_get_stats
  unsigned long long* cstats; // [4] of cuharm_get_chain_stats
  const double* dt;
  double dtfac, idx1, idx2, idx3, gam;
  NewtonCfg nc;
  FloorCfg fc;
  ChainCfg cc;
};

template <int RECON, int RIEMANN>
__global__ void __launch_bounds__(128) chain_kernel(ChainArgs a) {
  const Dims& d = a.d;
  const unsigned long long nf = *a.nfail;
  unsigned long long c_chain = 0, c_1dw = 0, c_ent = 0, c_beta = 0, c_bad = 0;
  int fl_rho = 0, fl_u = 0, fl_ceil = 0, fl_cap = 0;
  for (unsigned long long e = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; e < nf;
       e += (unsigned long long)gridDim.x * blockDim.x) {
    const long long idx = a.list[e];
    const int kind = a.flag[idx];
    if (kind == 1) { c_bad++; continue; }  // D <= 0 or non-finite input: no method applies
    const int i = (int)(idx / d.s1), j = (int)((idx - i * d.s1) / d.s2);
    const int q2 = i * d.n2g + j;
    const Geom G = load_geom(a.C, q2);
    double U[8], pb[8], pn[8];
#pragma unroll
    for (int v = 0; v < 8; v++) U[v] = a.ustar[v * d.nz + idx];
#pragma unroll
    for (int v = 0; v < 8; v++) pb[v] = a.Pout[v * d.nz + idx];
    // eq. 11 for this zone: U_S* = sqrt(-g) S u^t (P^n) - dtau div F_S (no source)
    const double lor = sqrt(1.0 + gamma_sq_minus_one(pb, G));
    double US = G.sg * entropy_density(pb[0], pb[1], a.gam) * (lor / G.alpha);
    {
      const Geom G1a = load_geom(a.F1g, q2), G1b = load_geom(a.F1g, q2 + d.n2g);
      const Geom G2a = load_geom(a.F2g, q2), G2b = load_geom(a.F2g, q2 + 1);
      const double f1a = entropy_face_flux<1, RECON, RIEMANN>(a.Pflux, d.nz, idx, d.s1, G1a, a.gam);
      const double f1b = entropy_face_flux<1, RECON, RIEMANN>(a.Pflux, d.nz, idx + d.s1, d.s1, G1b, a.gam);
      const double f2a = entropy_face_flux<2, RECON, RIEMANN>(a.Pflux, d.nz, idx, d.s2, G2a, a.gam);
      const double f2b = entropy_face_flux<2, RECON, RIEMANN>(a.Pflux, d.nz, idx + d.s2, d.s2, G2b, a.gam);
      const double f3a = entropy_face_flux<3, RECON, RIEMANN>(a.Pflux, d.nz, idx, 1, G, a.gam);
      const double f3b = entropy_face_flux<3, RECON, RIEMANN>(a.Pflux, d.nz, idx + 1, 1, G, a.gam);
      const double divS = (f1b - f1a) * a.idx1 + (f2b - f2a) * a.idx2 + (f3b - f3a) * a.idx3;
      US = US + a.dtfac * __ldg(a.dt) * (-divS);
    }
    int f2;
#pragma unroll
    for (int v = 0; v < 8; v++) pn[v] = pb[v];
    if (kind == KIND_ENTROPY_FIRST) {  // eq. 33: the entropy method is the first and only choice
      c_beta++;
      f2 = invert_entropy_dev(U, US, G, a.gam, pn, a.cc.brent_tol, a.cc.brent_maxit);
      if (f2 == 0) c_ent++;
    } else {
      c_chain++;
      f2 = kind;
      if (kind == 2 || kind == 3) {    // "fails to produce results" -> the 1D method
        f2 = invert_1dw_dev(U, G, a.gam, pn, a.cc.brent_tol, a.cc.brent_maxit);
        if (f2 == 0) c_1dw++;
      }
      if (f2 != 0) {                   // non-physical values, or the 1D method failed too -> the entropy method
#pragma unroll
        for (int v = 0; v < 8; v++) pn[v] = pb[v];
        f2 = invert_entropy_dev(U, US, G, a.gam, pn, a.cc.brent_tol, a.cc.brent_maxit);
        if (f2 == 0) c_ent++;
      }
    }
    if (f2 != 0) {
#pragma unroll
      for (int v = 0; v < 5; v++) pn[v] = pb[v];  // the guess stays; eq. 34 repairs the zone
      c_bad++;
    } else {
      const int m = apply_floors(pn, G, a.C + q2, a.floors[2 * q2], a.floors[2 * q2 + 1], a.fc, a.gam, a.nc);
      fl_rho += m & 1; fl_u += (m >> 1) & 1; fl_ceil += (m >> 2) & 1; fl_cap += (m >> 3) & 1;
    }
    a.flag[idx] = f2;
#pragma unroll
    for (int v = 0; v < 8; v++) a.Pout[v * d.nz + idx] = pn[v];
  }
  if (c_bad) atomicAdd(a.nbad, c_bad);
  if (c_chain) atomicAdd(a.cstats + 0, c_chain);
  if (c_1dw) atomicAdd(a.cstats + 1, c_1dw);
  if (c_ent) atomicAdd(a.cstats + 2, c_ent);
  if (c_beta) atomicAdd(a.cstats + 3, c_beta);
  if (fl_rho) atomicAdd(a.stats + 2, (unsigned long long)fl_rho);
  if (fl_u) atomicAdd(a.stats + 3, (unsigned long long)fl_u);
  if (fl_ceil) atomicAdd(a.stats + 4, (unsigned long long)fl_ceil);
  if (fl_cap) atomicAdd(a.stats + 5, (unsigned long long)fl_cap);
}

// Stage-level test helper (cuharm_invert_fallback): one of the two fallback methods on full-grid arrays, like
// cons_to_prim_kernel.  method 1: the 1D method; 2: the entropy method (US[zone] = conserved entropy sqrt(-g) S u^t).
struct FallbackArgs {
  Dims d;
  const double* U;
  const double* US;
  double* prim;
  int* flag;
  const Geom* C;
  double gam;
  int method;
  ChainCfg cc;
};

__global__ void __launch_bounds__(128) fallback_kernel(FallbackArgs a) {
  const Dims& d = a.d;
  const int k = blockIdx.x * 128 + threadIdx.x;
  if (k >= d.n3g) return;
  const int j = blockIdx.y, i = blockIdx.z;
  const long long idx = i * d.s1 + j * d.s2 + k;
  const Geom G = load_geom(a.C, i * d.n2g + j);
  double q[8], U[8];
#pragma unroll
  for (int v = 0; v < 8; v++) { U[v] = a.U[v * d.nz + idx]; q[v] = a.prim[v * d.nz + idx]; }
  const int f = a.method == 1 ? invert_1dw_dev(U, G, a.gam, q, a.cc.brent_tol, a.cc.brent_maxit)
                              : invert_entropy_dev(U, a.US[idx], G, a.gam, q, a.cc.brent_tol, a.cc.brent_maxit);
#pragma unroll
  for (int v = 0; v < 8; v++) a.prim[v * d.nz + idx] = q[v];
  if (a.flag) a.flag[idx] = f;
}

}  // namespace cuharm
