// cuharm_geom.cuh — geometry precompute (S0): Kerr-Schild metric in modified Kerr-Schild coordinates
// (eqs. 38-39; A14), its inverse, sqrt(-g), lapse at centres / 1-faces / 2-faces, connection
// coefficients at centres from closed-form derivatives (A19), floor profiles (eq. 35).
// One thread per (i,j) column; runs once, cost irrelevant.  Shares nothing with oracle/.
#pragma once
#include "cuharm_phys.cuh"

namespace cuharm {

struct GeomArgs {
  int n1g, n2g, ng, n2;
  int i_off;       // global X1 index of this grid's first interior zone (slab decomposition; 0 for the whole grid)
  int coords, polar_bc;  // polar_bc: X2 boundary is the polar reflection -> the 2-faces J = 0, n2 lie on the axis (A32)
  double a, R0, hslope;
  double xb;       // X1 of the exponential -> hyper-exponential transition (eq. 39); used when nx >= 2
  int nx;          // exponent n_X of the hyper-exponential branch; < 2: plain exponential everywhere
  double x0_1, x0_2, dx1, dx2;
  double rho_fl_coef, rho_fl_pow, rho_fl_abs, u_fl_coef, u_fl_pow, u_fl_abs;
  Geom *C, *F1, *F2;
  double* conn;    // [n1g*n2g][40]  (export helper only)
  double* srcw;    // [n1g*n2g][14]  source weights (source_weights below)
  double* floors;  // [n1g*n2g][2]
  double* rec;     // [n1g*n2g][36]  centre geometry record (20) + source weights (14) + floors (2), one bulk copy per tile
};

struct MksPoint {
  double r, th, rp, thp, thpp;  // r, theta, dr/dX1, dtheta/dX2, d2theta/dX2^2
  double rpp;                   // d2r/dX1^2
};

__device__ inline double ipow(double y, int n) {  // y^n for small n >= 0 by repeated multiplication
  double v = 1.0;
  for (int q = 0; q < n; q++) v *= y;
  return v;
}

__device__ inline MksPoint mks_point(const GeomArgs& A, double X1, double X2) {
  const double PI = 3.14159265358979323846;
  MksPoint p;
  // eq. 39: r = R0 + exp(E), E = X for X < x_b, E = X + (X - x_b)^n_X beyond; r' = (r - R0) E', r'' = (r - R0)(E'^2 + E'')
  double E = X1, E1 = 1.0, E2 = 0.0;
  if (A.nx >= 2 && X1 >= A.xb) {
    const double y = X1 - A.xb;
    const double ym2 = ipow(y, A.nx - 2);
    E = X1 + ym2 * y * y;
    E1 = 1.0 + A.nx * ym2 * y;
    E2 = A.nx * (A.nx - 1) * ym2;
  }
  const double e = exp(E);
  p.r = A.R0 + e;
  p.rp = e * E1;
  p.rpp = e * (E1 * E1 + E2);
  const double arg = PI * (1.0 + X2);
  const double s = sin(arg), c = cos(arg);
  p.th = 0.5 * PI * (1.0 + X2) + 0.5 * (1.0 - A.hslope) * s;
  p.thp = 0.5 * PI * (1.0 + (1.0 - A.hslope) * c);
  p.thpp = -0.5 * PI * PI * (1.0 - A.hslope) * s;
  return p;
}

__device__ inline void flat_geom(Geom& G) {
  G.g00 = -1.0; G.g01 = 0.0; G.g03 = 0.0; G.g11 = 1.0; G.g13 = 0.0; G.g22 = 1.0; G.g33 = 1.0;
  G.c00 = -1.0; G.c01 = 0.0; G.c03 = 0.0; G.c11 = 1.0; G.c13 = 0.0; G.c22 = 1.0; G.c33 = 1.0;
  G.sg = 1.0; G.alpha = 1.0;
  G.ialpha = 1.0; G.ac01 = 0.0; G.isg = 1.0; G.pad = 0.0;
}

// eq. 38 with Sigma = r^2 + a^2 cos^2(theta), transformed by J = diag(1, r', theta', 1)
__device__ inline void mks_geom(const GeomArgs& A, double X1, double X2, bool on_axis, Geom& G) {
  const MksPoint p = mks_point(A, X1, X2);
  const double a = A.a, r = p.r;
  const double sn = sin(p.th), cs = cos(p.th);
  const double s2 = sn * sn;
  const double Sig = r * r + a * a * cs * cs;
  const double f = 2.0 * r / Sig;
  G.g00 = -1.0 + f;
  G.g01 = f * p.rp;
  G.g03 = -a * s2 * f;
  G.g11 = (1.0 + f) * p.rp * p.rp;
  G.g13 = -a * s2 * (1.0 + f) * p.rp;
  G.g22 = Sig * p.thp * p.thp;
  G.g33 = s2 * (Sig + a * a * s2 * (1.0 + f));
  const double s2f = s2 < 1e-30 ? 1e-30 : s2;  // A32
  const double Del = r * r - 2.0 * r + a * a;
  G.c00 = -(1.0 + f);
  G.c01 = f / p.rp;
  G.c03 = 0.0;
  G.c11 = Del / Sig / (p.rp * p.rp);
  G.c13 = a / Sig / p.rp;
  G.c22 = 1.0 / Sig / (p.thp * p.thp);
  G.c33 = 1.0 / (Sig * s2f);
  G.sg = on_axis ? 0.0 : Sig * fabs(sn) * fabs(p.rp) * fabs(p.thp);
  G.alpha = 1.0 / sqrt(-G.c00);
  G.ialpha = sqrt(-G.c00);
  G.ac01 = G.alpha * G.c01;
  G.isg = G.sg > 0.0 ? 1.0 / G.sg : 0.0;
  G.pad = 0.0;
}

// d_c g_{mn} (c = 1, 2; the metric depends on X1, X2 only) in closed form: eq. 38 differentiated in r and theta and
// pushed through the diagonal Jacobian J = diag(1, r', theta', 1), including the dJ/dX terms (A19).
__device__ inline void mks_dmetric(const GeomArgs& A, double X1, double X2, double dg[4][4][4]) {
  const MksPoint p = mks_point(A, X1, X2);
  const double a = A.a, r = p.r;
  const double sn = sin(p.th), cs = cos(p.th);
  const double s2 = sn * sn;
  const double Sig = r * r + a * a * cs * cs;
  const double f = 2.0 * r / Sig;
  // d/dr and d/dtheta of Sigma, f, sin^2
  const double Sr = 2.0 * r, St = -2.0 * a * a * sn * cs;
  const double fr = 2.0 / Sig - 2.0 * r * Sr / (Sig * Sig);
  const double ft = -2.0 * r * St / (Sig * Sig);
  const double s2t = 2.0 * sn * cs;
  double k[4][4] = {}, kr[4][4] = {}, kt[4][4] = {};  // KS metric and its r-, theta-derivatives
  k[0][0] = -1.0 + f;               kr[0][0] = fr;              kt[0][0] = ft;
  k[0][1] = f;                      kr[0][1] = fr;              kt[0][1] = ft;
  k[0][3] = -a * s2 * f;            kr[0][3] = -a * s2 * fr;    kt[0][3] = -a * (s2t * f + s2 * ft);
  k[1][1] = 1.0 + f;                kr[1][1] = fr;              kt[1][1] = ft;
  k[1][3] = -a * s2 * (1.0 + f);    kr[1][3] = -a * s2 * fr;    kt[1][3] = -a * (s2t * (1.0 + f) + s2 * ft);
  k[2][2] = Sig;                    kr[2][2] = Sr;              kt[2][2] = St;
  const double h = Sig + a * a * s2 * (1.0 + f);
  k[3][3] = s2 * h;
  kr[3][3] = s2 * (Sr + a * a * s2 * fr);
  kt[3][3] = s2t * h + s2 * (St + a * a * (s2t * (1.0 + f) + s2 * ft));
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < m; n++) { k[m][n] = k[n][m]; kr[m][n] = kr[n][m]; kt[m][n] = kt[n][m]; }
  const double J[4] = {1.0, p.rp, p.thp, 1.0};
  const double J1[4] = {0.0, p.rpp, 0.0, 0.0};   // dJ/dX1 = r'' (= r' on the plain exponential branch)
  const double J2[4] = {0.0, 0.0, p.thpp, 0.0};  // dJ/dX2
  for (int m = 0; m < 4; m++)
    for (int n = 0; n < 4; n++) {
      dg[m][n][0] = 0.0;
      dg[m][n][3] = 0.0;
      dg[m][n][1] = (J1[m] * J[n] + J[m] * J1[n]) * k[m][n] + J[m] * J[n] * kr[m][n] * p.rp;
      dg[m][n][2] = (J2[m] * J[n] + J[m] * J2[n]) * k[m][n] + J[m] * J[n] * kt[m][n] * p.thp;
    }
}

// Gamma^l_{nk} = 1/2 g^{ls} (d_n g_{sk} + d_k g_{sn} - d_s g_{nk})
__device__ inline void mks_conn(const double dg[4][4][4], const Geom& G, double* out40) {
  double gc[4][4] = {};
  gc[0][0] = G.c00; gc[0][1] = gc[1][0] = G.c01; gc[0][3] = gc[3][0] = G.c03; gc[1][1] = G.c11;
  gc[1][3] = gc[3][1] = G.c13; gc[2][2] = G.c22; gc[3][3] = G.c33;
  int s = 0;
  for (int l = 0; l < 4; l++) {
    for (int n = 0; n < 4; n++)
      for (int kk = n; kk < 4; kk++) {
        double sum = 0.0;
        for (int m = 0; m < 4; m++) sum += gc[l][m] * (dg[m][kk][n] + dg[m][n][kk] - dg[n][kk][m]);
        out40[s++] = 0.5 * sum;
      }
  }
}

// Source weights.  With T^{kl} symmetric, eq. 7's S_nu = sqrt(-g) T^k_l Gamma^l_{nu k} = sqrt(-g) T^{ks} Gamma_{s nu k}
// and the last two terms of Gamma_{s nu k} = (d_nu g_{sk} + d_k g_{s nu} - d_s g_{nu k})/2 are antisymmetric in (k, s):
// S_nu = (1/2) sqrt(-g) T^{kl} d_nu g_{kl}, a sum over the 7 metric entries that do not vanish identically (the
// off-diagonal ones counted twice), for nu = 1, 2 (nu = t, phi: zero, the metric depends on neither).
// w[7 (nu - 1) + e] = sqrt(-g) x (1/2 or 1) x d_nu g_e, e over 00 01 03 11 13 22 33.
__device__ inline void source_weights(const double dg[4][4][4], double sg, double* w14) {
  const int em[7] = {0, 0, 0, 1, 1, 2, 3}, en[7] = {0, 1, 3, 1, 3, 2, 3};
  for (int nu = 1; nu <= 2; nu++)
    for (int e = 0; e < 7; e++) w14[7 * (nu - 1) + e] = sg * (em[e] == en[e] ? 0.5 : 1.0) * dg[em[e]][en[e]][nu];
}

__global__ void geom_kernel(GeomArgs A) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= A.n1g * A.n2g) return;
  const int i = t / A.n2g, j = t % A.n2g;
  const int I = i - A.ng + A.i_off, Jz = j - A.ng;
  Geom C, F1, F2;
  double cn[40], sw[14];
  double rc = 1.0;
  if (A.coords == 1) {
    flat_geom(C); flat_geom(F1); flat_geom(F2);
    for (int s = 0; s < 40; s++) cn[s] = 0.0;
    for (int s = 0; s < 14; s++) sw[s] = 0.0;
  } else {
    // the same rounding as a plain product-then-sum: keeps the face coordinate of the polar faces exact
    const double X1c = __dadd_rn(A.x0_1, __dmul_rn(I + 0.5, A.dx1)), X2c = __dadd_rn(A.x0_2, __dmul_rn(Jz + 0.5, A.dx2));
    const double X1f = __dadd_rn(A.x0_1, __dmul_rn((double)I, A.dx1)), X2f = __dadd_rn(A.x0_2, __dmul_rn((double)Jz, A.dx2));
    mks_geom(A, X1c, X2c, false, C);
    mks_geom(A, X1f, X2c, false, F1);
    const bool axis = A.polar_bc && (Jz == 0 || Jz == A.n2);
    mks_geom(A, X1c, X2f, axis, F2);
    double dg[4][4][4];
    mks_dmetric(A, X1c, X2c, dg);
    mks_conn(dg, C, cn);
    source_weights(dg, C.sg, sw);
    rc = mks_point(A, X1c, X2c).r;
  }
  A.C[t] = C; A.F1[t] = F1; A.F2[t] = F2;
  for (int s = 0; s < 40; s++) A.conn[(size_t)t * 40 + s] = cn[s];
  for (int s = 0; s < 14; s++) A.srcw[(size_t)t * 14 + s] = sw[s];
  A.floors[2 * t + 0] = fmax(A.rho_fl_abs, A.rho_fl_coef * pow(rc, A.rho_fl_pow));  // eq. 35 (A9)
  A.floors[2 * t + 1] = fmax(A.u_fl_abs, A.u_fl_coef * pow(rc, A.u_fl_pow));
  double* rec = A.rec + (size_t)t * 36;
  const double* cg = reinterpret_cast<const double*>(&A.C[t]);
  for (int s = 0; s < 20; s++) rec[s] = cg[s];
  for (int s = 0; s < 14; s++) rec[20 + s] = sw[s];
  rec[34] = A.floors[2 * t + 0];
  rec[35] = A.floors[2 * t + 1];
}

// expand a table to the caller's SoA layout (include/cuharm.h, cuharm_get_geom)
__global__ void geom_export_kernel(const Geom* tab, const double* conn, int loc, int n, double* out) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  if (loc < 3) {
    const Geom G = tab[t];
    const double cov[10] = {G.g00, G.g01, 0.0, G.g03, G.g11, 0.0, G.g13, G.g22, 0.0, G.g33};
    const double con[10] = {G.c00, G.c01, 0.0, G.c03, G.c11, 0.0, G.c13, G.c22, 0.0, G.c33};
    for (int s = 0; s < 10; s++) { out[(size_t)s * n + t] = cov[s]; out[(size_t)(10 + s) * n + t] = con[s]; }
    out[(size_t)20 * n + t] = G.sg;
    out[(size_t)21 * n + t] = G.alpha;
  } else {
    for (int s = 0; s < 40; s++) out[(size_t)s * n + t] = conn[(size_t)t * 40 + s];
  }
}

}  // namespace cuharm
