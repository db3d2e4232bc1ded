// cuharm_kernels.cuh — grid kernels of the hot path (S1-S11 of DESIGN.md) other than the flux kernels
// (cuharm_flux.cuh): ghost fill, flux-CT EMFs, fused source+update+inversion+floors, repair of failed zones, CFL and div B
// reductions.  fp64, SoA prim[8][n1g][n2g][n3g] with k (phi) fastest: a warp runs along k at fixed (i,j), so
// every geometry read is a broadcast (the metric is phi-independent).
#pragma once
#include "cuharm_flux.cuh"

namespace cuharm {

// ---------------------------------------------------------------------------------------------------------
// S1  Boundary conditions (A15).  Order X1, X2, X3, each over the full extended range of the others.
// kind: 0 outflow (+ inflow check in MKS X1), 1 periodic, 2 polar reflection, 3 fixed (kernel not launched).
// `gate`: if non-null and *gate == 0 the kernel does nothing (second ghost fill, needed only after repairs).
// ---------------------------------------------------------------------------------------------------------
struct BcArgs {
  Dims d;
  double* P;
  const Geom* C;
  int kind, coords;
  double gamma_max;
  const unsigned long long* gate;
};

__device__ __forceinline__ void inflow_check(double q[8], const Geom& G, bool inner, double gamma_max) {
  State S;
  fluid_state(q, G, S);
  const bool bad = inner ? (S.u1 > 0.0) : (S.u1 < 0.0);
  if (!bad) return;
  const double il = 1.0 / S.lor;
  const double v1 = G.alpha * G.c01;  // beta^1/alpha: makes u^1 = 0
  const double v2 = q[3] * il, v3 = q[4] * il;
  double vsq = G.g11 * v1 * v1 + G.g22 * v2 * v2 + G.g33 * v3 * v3 + 2.0 * (G.g13 * v1 * v3);
  const double gmax = gamma_max > 0.0 ? gamma_max : 50.0;
  const double vmax = 1.0 - 1.0 / (gmax * gmax);
  vsq = vsq > vmax ? vmax : vsq;
  const double ln = 1.0 / sqrt(1.0 - vsq);
  q[2] = ln * v1; q[3] = ln * v2; q[4] = ln * v3;
}

__global__ void bc_x1_kernel(BcArgs a) {
  if (a.gate && *a.gate == 0ull) return;
  const Dims& d = a.d;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= d.n3g) return;
  const int j = blockIdx.y;
  const int g = blockIdx.z >> 1, side = blockIdx.z & 1;
  const int ig = side ? (d.ng + d.n1 + g) : (d.ng - 1 - g);
  int is;
  if (a.kind == 1) {
    const int I = side ? (d.n1 + g) : (-1 - g);
    is = d.ng + ((I % d.n1) + d.n1) % d.n1;  // wraps repeatedly when n1 < ng
  } else {
    is = side ? (d.ng + d.n1 - 1) : d.ng;
  }
  double q[8];
  const long long src = is * d.s1 + j * d.s2 + k, dst = ig * d.s1 + j * d.s2 + k;
#pragma unroll
  for (int v = 0; v < 8; v++) q[v] = a.P[v * d.nz + src];
  if (a.kind == 0) {
    const Geom Gg = load_geom(a.C, ig * d.n2g + j);
    const double ratio = __ldg(&a.C[is * d.n2g + j].sg) / Gg.sg;  // sqrt(-g) B^i constant across the copy
    q[5] *= ratio; q[6] *= ratio; q[7] *= ratio;
    if (a.coords == 0) inflow_check(q, Gg, side == 0, a.gamma_max);
  }
#pragma unroll
  for (int v = 0; v < 8; v++) a.P[v * d.nz + dst] = q[v];
}

__global__ void bc_x2_kernel(BcArgs a) {
  if (a.gate && *a.gate == 0ull) return;
  const Dims& d = a.d;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= d.n3g) return;
  const int i = blockIdx.y;
  const int g = blockIdx.z >> 1, side = blockIdx.z & 1;
  const int jg = side ? (d.ng + d.n2 + g) : (d.ng - 1 - g);
  int js;
  if (a.kind == 1) {
    const int J = side ? (d.n2 + g) : (-1 - g);
    js = d.ng + ((J % d.n2) + d.n2) % d.n2;
  } else if (a.kind == 2) js = side ? (d.ng + d.n2 - 1 - g) : (d.ng + g);
  else js = side ? (d.ng + d.n2 - 1) : d.ng;
  const long long src = i * d.s1 + js * d.s2 + k, dst = i * d.s1 + jg * d.s2 + k;
  double q[8];
#pragma unroll
  for (int v = 0; v < 8; v++) q[v] = a.P[v * d.nz + src];
  if (a.kind == 2) { q[3] = -q[3]; q[6] = -q[6]; }  // utilde^2, B^2 change sign
  if (a.kind == 0) {
    const double ratio = __ldg(&a.C[i * d.n2g + js].sg) / __ldg(&a.C[i * d.n2g + jg].sg);
    q[5] *= ratio; q[6] *= ratio; q[7] *= ratio;
  }
#pragma unroll
  for (int v = 0; v < 8; v++) a.P[v * d.nz + dst] = q[v];
}

__global__ void bc_x3_kernel(BcArgs a) {
  if (a.gate && *a.gate == 0ull) return;
  const Dims& d = a.d;
  const int t = blockIdx.x * blockDim.x + threadIdx.x;  // over (i,j) columns and the 2*ng ghost slots
  const int ncol = d.n1g * d.n2g;
  if (t >= ncol * 2 * d.ng) return;
  const int slot = t % (2 * d.ng), col = t / (2 * d.ng);
  const int g = slot >> 1, side = slot & 1;
  const int kg = side ? (d.ng + d.n3 + g) : (d.ng - 1 - g);
  int ks;
  if (a.kind == 1) {
    const int K = side ? (d.n3 + g) : (-1 - g);
    ks = d.ng + ((K % d.n3) + d.n3) % d.n3;  // wraps repeatedly when n3 < ng
  } else {
    ks = side ? (d.ng + d.n3 - 1) : d.ng;
  }
  const long long base = (long long)col * d.n3g;
#pragma unroll
  for (int v = 0; v < 8; v++) a.P[v * d.nz + base + kg] = a.P[v * d.nz + base + ks];
}

// ---------------------------------------------------------------------------------------------------------
// S4  Flux-CT edge EMFs (eq. 21).  E^1 on (I, J-1/2, K-1/2), E^2 on (I-1/2, J, K-1/2),
// E^3 on (I-1/2, J-1/2, K), each stored at zone (I,J,K).  Range ng..ng+N inclusive in every direction.
// ---------------------------------------------------------------------------------------------------------
struct EmfArgs {
  Dims d;
  const double *F1, *F2, *F3;  // [7][nz] each
  double* E;                   // [3][nz]
};

__global__ void __launch_bounds__(128) emf_kernel(EmfArgs a) {
  const Dims& d = a.d;
  const int k = d.ng + blockIdx.x * 128 + threadIdx.x;
  if (k > d.ng + d.n3) return;
  const int j = d.ng + blockIdx.y, i = d.ng + blockIdx.z;
  const long long idx = i * d.s1 + j * d.s2 + k;
  // component slots: F1: [5] = B2, [6] = B3;  F2: [5] = B3, [6] = B1;  F3: [5] = B1, [6] = B2
  const double* F1B2 = a.F1 + 5 * d.nz; const double* F1B3 = a.F1 + 6 * d.nz;
  const double* F2B3 = a.F2 + 5 * d.nz; const double* F2B1 = a.F2 + 6 * d.nz;
  const double* F3B1 = a.F3 + 5 * d.nz; const double* F3B2 = a.F3 + 6 * d.nz;
  a.E[idx] = 0.25 * (F2B3[idx] + F2B3[idx - 1] - F3B2[idx] - F3B2[idx - d.s2]);
  a.E[d.nz + idx] = 0.25 * (F3B1[idx] + F3B1[idx - d.s1] - F1B3[idx] - F1B3[idx - 1]);
  a.E[2 * d.nz + idx] = 0.25 * (F1B2[idx] + F1B2[idx - d.s2] - F2B1[idx] - F2B1[idx - d.s1]);
}

// ---------------------------------------------------------------------------------------------------------
// S5-S7+S9  Fused source + conserved update + Noble inversion + floors, one thread per interior zone
// (eqs. 14, 22, 25, 27-31, 35-37; A5, A34, A35).  SAME: the flux state is the base state (predictor).
// ---------------------------------------------------------------------------------------------------------
struct UpdArgs {
  Dims d;
  const double* Pbase;  // P^n: supplies U^n and the Newton guess
  const double* Pflux;  // state the fluxes / source were built from
  double* Pout;
  const double *F1, *F2, *F3, *E;
  const Geom* C;
  const double* conn;
  const double* floors;
  int* flag;
  int* list;                    // failed zones of this substep
  unsigned long long* nfail;    // counter of this substep
  unsigned long long* stats;    // [8]
  double dtau, idx1, idx2, idx3, gam;
  NewtonCfg nc;
  FloorCfg fc;
};

template <bool SAME>
__global__ void __launch_bounds__(128) update_kernel(UpdArgs a) {
  const Dims& d = a.d;
  const int k = d.ng + blockIdx.x * 128 + threadIdx.x;
  const int j = d.ng + blockIdx.y, i = d.ng + blockIdx.z;
  int c_rho = 0, c_u = 0, c_ceil = 0, c_cap = 0, c_its = 0;
  if (k < d.ng + d.n3) {
    const long long idx = i * d.s1 + j * d.s2 + k;
    const int q2 = i * d.n2g + j;
    const Geom G = load_geom(a.C, q2);
    double pb[8];
#pragma unroll
    for (int v = 0; v < 8; v++) pb[v] = a.Pbase[v * d.nz + idx];
    State S;
    fluid_state(pb, G, S);
    double U[8];
    flux_vector<0>(pb, S, G, a.gam, U);
    double src[4];
    if (SAME) {
      source_term(pb, S, G, a.conn + (size_t)q2 * 40, a.gam, src);
    } else {
      double pf[8];
#pragma unroll
      for (int v = 0; v < 8; v++) pf[v] = a.Pflux[v * d.nz + idx];
      fluid_state(pf, G, S);
      source_term(pf, S, G, a.conn + (size_t)q2 * 40, a.gam, src);
    }
    // hydrodynamic components: face-flux differences (eq. 25)
#pragma unroll
    for (int v = 0; v < 5; v++) {
      const double* f1 = a.F1 + v * d.nz + idx;
      const double* f2 = a.F2 + v * d.nz + idx;
      const double* f3 = a.F3 + v * d.nz + idx;
      const double div = (f1[d.s1] - f1[0]) * a.idx1 + (f2[d.s2] - f2[0]) * a.idx2 + (f3[1] - f3[0]) * a.idx3;
      const double s = (v >= 1) ? src[v - 1] : 0.0;
      U[v] = U[v] + a.dtau * (s - div);
    }
    // induction: flux-CT replacement fluxes from the edge EMFs (eq. 22; A3)
    {
      const double* E1 = a.E + idx; const double* E2 = a.E + d.nz + idx; const double* E3 = a.E + 2 * d.nz + idx;
      const double e1_00 = E1[0], e1_j = E1[d.s2], e1_k = E1[1], e1_jk = E1[d.s2 + 1];
      const double e2_00 = E2[0], e2_i = E2[d.s1], e2_k = E2[1], e2_ik = E2[d.s1 + 1];
      const double e3_00 = E3[0], e3_i = E3[d.s1], e3_j = E3[d.s2], e3_ij = E3[d.s1 + d.s2];
      // F~2(B1) = -1/2 (E3 + E3[i+1]) at faces j, j+1;  F~3(B1) = +1/2 (E2 + E2[i+1]) at faces k, k+1
      const double divB1 = ((-0.5 * (e3_j + e3_ij)) - (-0.5 * (e3_00 + e3_i))) * a.idx2 +
                           ((0.5 * (e2_k + e2_ik)) - (0.5 * (e2_00 + e2_i))) * a.idx3;
      // F~1(B2) = +1/2 (E3 + E3[j+1]) at faces i, i+1;  F~3(B2) = -1/2 (E1 + E1[j+1]) at faces k, k+1
      const double divB2 = ((0.5 * (e3_i + e3_ij)) - (0.5 * (e3_00 + e3_j))) * a.idx1 +
                           ((-0.5 * (e1_k + e1_jk)) - (-0.5 * (e1_00 + e1_j))) * a.idx3;
      // F~1(B3) = -1/2 (E2 + E2[k+1]) at faces i, i+1;  F~2(B3) = +1/2 (E1 + E1[k+1]) at faces j, j+1
      const double divB3 = ((-0.5 * (e2_i + e2_ik)) - (-0.5 * (e2_00 + e2_k))) * a.idx1 +
                           ((0.5 * (e1_j + e1_jk)) - (0.5 * (e1_00 + e1_k))) * a.idx2;
      U[5] = U[5] - a.dtau * divB1;
      U[6] = U[6] - a.dtau * divB2;
      U[7] = U[7] - a.dtau * divB3;
    }
    double pn[8];
#pragma unroll
    for (int v = 0; v < 8; v++) pn[v] = pb[v];  // A35: the guess is P^n
    const int flag = invert_2d(U, G, a.gam, pn, a.nc, c_its);
    if (flag == 0) {
      const int m = apply_floors(pn, G, a.C + q2, __ldg(a.floors + 2 * q2), __ldg(a.floors + 2 * q2 + 1), a.fc, a.gam, a.nc);
      c_rho = m & 1; c_u = (m >> 1) & 1; c_ceil = (m >> 2) & 1; c_cap = (m >> 3) & 1;
    } else {
      const unsigned long long pos = atomicAdd(a.nfail, 1ull);
      a.list[pos] = (int)idx;
    }
    a.flag[idx] = flag;
#pragma unroll
    for (int v = 0; v < 8; v++) a.Pout[v * d.nz + idx] = pn[v];
  }
  // statistics: warp sums, one atomic per warp and counter, zeros skipped
  c_rho = __reduce_add_sync(0xffffffffu, c_rho);
  c_u = __reduce_add_sync(0xffffffffu, c_u);
  c_ceil = __reduce_add_sync(0xffffffffu, c_ceil);
  c_cap = __reduce_add_sync(0xffffffffu, c_cap);
  c_its = __reduce_add_sync(0xffffffffu, c_its);
  __shared__ int sh[5];
  if (threadIdx.x < 5) sh[threadIdx.x] = 0;
  __syncthreads();
  if ((threadIdx.x & 31) == 0) {
    if (c_rho) atomicAdd(&sh[0], c_rho);
    if (c_u) atomicAdd(&sh[1], c_u);
    if (c_ceil) atomicAdd(&sh[2], c_ceil);
    if (c_cap) atomicAdd(&sh[3], c_cap);
    if (c_its) atomicAdd(&sh[4], c_its);
  }
  __syncthreads();
  if (threadIdx.x < 5 && sh[threadIdx.x]) atomicAdd(a.stats + 2 + threadIdx.x, (unsigned long long)sh[threadIdx.x]);
}

// ---------------------------------------------------------------------------------------------------------
// S8  Repair of zones whose inversion failed (eq. 34; A13): deterministic Jacobi passes over the
// (short) list of failed zones.  Pass m: a still-bad zone whose 4 face neighbours in the (I,J) plane were all
// good at the start of the pass takes their mean; else the 4 diagonal neighbours; else it waits; in the last
// pass leftovers take the mean of whatever good zones exist among the 8 neighbours.  Only rho, u, utilde^i are
// replaced; floors are re-applied to the repaired zone.  flag > 0: bad; flag = -(m+1): repaired in
// pass m, i.e. good from pass m+1 on — which is what makes the passes Jacobi without a snapshot: donors are
// zones that are not written in the current pass.  One block: failures are rare (none in the first 1000 steps
// of the torus workloads); the list has room for every zone, so a pathological step is slow but still right.
// ---------------------------------------------------------------------------------------------------------
struct FixArgs {
  Dims d;
  double* P;
  int* flag;
  const int* list;
  const unsigned long long* nfail;
  unsigned long long* stats;
  const Geom* C;
  const double* floors;
  int max_passes;
  double gam;
  NewtonCfg nc;
  FloorCfg fc;
};

__device__ __forceinline__ bool zone_good(int f, int pass) { return f == 0 || (f < 0 && -f - 1 < pass); }

__global__ void __launch_bounds__(1024) fixup_kernel(FixArgs a) {
  const Dims& d = a.d;
  const unsigned long long nf = *a.nfail;
  if (nf == 0ull) return;
  if (threadIdx.x == 0) atomicAdd(a.stats + 0, nf);
  const long long fo[4] = {d.s1, -d.s1, d.s2, -d.s2};
  const long long dg[4] = {d.s1 + d.s2, d.s1 - d.s2, -d.s1 + d.s2, -d.s1 - d.s2};
  unsigned long long repaired = 0ull, lastres = 0ull;
  for (int pass = 0; pass <= a.max_passes; pass++) {
    const bool last = pass == a.max_passes;
    int left = 0;
    for (unsigned long long e = threadIdx.x; e < nf; e += blockDim.x) {
      const long long idx = a.list[e];
      if (a.flag[idx] <= 0) continue;
      bool fg = true, dgood = true;
#pragma unroll
      for (int m = 0; m < 4; m++) {
        fg = fg && zone_good(a.flag[idx + fo[m]], pass);
        dgood = dgood && zone_good(a.flag[idx + dg[m]], pass);
      }
      double q[8];
      if (fg || dgood) {
        const long long* st = fg ? fo : dg;
#pragma unroll
        for (int v = 0; v < 5; v++) {
          double s = 0.0;
#pragma unroll
          for (int m = 0; m < 4; m++) s += a.P[v * d.nz + idx + st[m]];
          q[v] = 0.25 * s;
        }
      } else if (last) {
        int cnt = 0;
        double s[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        for (int di = -1; di <= 1; di++)
          for (int dj = -1; dj <= 1; dj++) {
            if (!di && !dj) continue;
            const long long n = idx + di * d.s1 + dj * d.s2;
            if (!zone_good(a.flag[n], pass)) continue;
            cnt++;
#pragma unroll
            for (int v = 0; v < 5; v++) s[v] += a.P[v * d.nz + n];
          }
#pragma unroll
        for (int v = 0; v < 5; v++) q[v] = cnt > 0 ? s[v] / cnt : a.P[v * d.nz + idx];
        lastres++;
      } else {
        left = 1;
        continue;
      }
#pragma unroll
      for (int v = 5; v < 8; v++) q[v] = a.P[v * d.nz + idx];
      const int q2 = (int)(idx / d.s2);  // = i * n2g + j
      const Geom G = load_geom(a.C, q2);
      apply_floors(q, G, a.C + q2, a.floors[2 * q2], a.floors[2 * q2 + 1], a.fc, a.gam, a.nc);
#pragma unroll
      for (int v = 0; v < 5; v++) a.P[v * d.nz + idx] = q[v];
      a.flag[idx] = -(pass + 1);
      repaired++;
    }
    __threadfence_block();
    if (!__syncthreads_or(left)) break;
  }
  if (repaired) atomicAdd(a.stats + 1, repaired);
  if (lastres) atomicAdd(a.stats + 7, lastres);
}

// ---------------------------------------------------------------------------------------------------------
// S11  Corner-centred divergence of sqrt(-g) B (eq. 23; A4): max |D| and max |D| / sum |terms|.
// ---------------------------------------------------------------------------------------------------------
struct DivbArgs {
  Dims d;
  const double* P;
  const Geom* C;
  double idx1, idx2, idx3;
  int khi;
  unsigned long long* out;  // [2]
};

__global__ void __launch_bounds__(128) divb_kernel(DivbArgs a) {
  const Dims& d = a.d;
  const int k = d.ng + blockIdx.x * 128 + threadIdx.x;
  const int j = d.ng + blockIdx.y, i = d.ng + blockIdx.z;
  double mabs = 0.0, mnorm = 0.0;
  if (k <= a.khi) {
    const bool two_d = d.n3 == 1;
    const double w = two_d ? 0.5 : 0.25;
    double D = 0.0, A = 0.0;
    for (int l1 = 0; l1 < 2; l1++)
      for (int l2 = 0; l2 < 2; l2++) {
        const double sg = __ldg(&a.C[(i + l1) * d.n2g + j + l2].sg);
        for (int l3 = 0; l3 < (two_d ? 1 : 2); l3++) {
          const long long n = (i + l1) * d.s1 + (j + l2) * d.s2 + k + l3;
          const double t1 = (l1 ? 1.0 : -1.0) * sg * a.P[5 * d.nz + n] * w * a.idx1;
          const double t2 = (l2 ? 1.0 : -1.0) * sg * a.P[6 * d.nz + n] * w * a.idx2;
          D += t1 + t2;
          A += fabs(t1) + fabs(t2);
          if (!two_d) {
            const double t3 = (l3 ? 1.0 : -1.0) * sg * a.P[7 * d.nz + n] * w * a.idx3;
            D += t3;
            A += fabs(t3);
          }
        }
      }
    mabs = fabs(D);
    mnorm = A > 0.0 ? fabs(D) / A : 0.0;
  }
  atomic_max_nonneg(a.out + 0, mabs);
  atomic_max_nonneg(a.out + 1, mnorm);
}

// ---------------------------------------------------------------------------------------------------------
// Full-grid primitive <-> conserved (eqs. 27-31), centre geometry, ghosts included.
// ---------------------------------------------------------------------------------------------------------
struct ConvArgs {
  Dims d;
  const double* in;   // prim (p2c) or U (c2p)
  double* out;        // U (p2c) or prim guess-in/answer-out (c2p)
  int* flag;
  const Geom* C;
  double gam;
  NewtonCfg nc;
};

__global__ void __launch_bounds__(128) prim_to_cons_kernel(ConvArgs a) {
  const Dims& d = a.d;
  const int k = blockIdx.x * 128 + threadIdx.x;
  if (k >= d.n3g) return;
  const int j = blockIdx.y, i = blockIdx.z;
  const long long idx = i * d.s1 + j * d.s2 + k;
  const Geom G = load_geom(a.C, i * d.n2g + j);
  double q[8], U[8];
#pragma unroll
  for (int v = 0; v < 8; v++) q[v] = a.in[v * d.nz + idx];
  State S;
  fluid_state(q, G, S);
  flux_vector<0>(q, S, G, a.gam, U);
#pragma unroll
  for (int v = 0; v < 8; v++) a.out[v * d.nz + idx] = U[v];
}

__global__ void __launch_bounds__(128) cons_to_prim_kernel(ConvArgs a) {
  const Dims& d = a.d;
  const int k = blockIdx.x * 128 + threadIdx.x;
  if (k >= d.n3g) return;
  const int j = blockIdx.y, i = blockIdx.z;
  const long long idx = i * d.s1 + j * d.s2 + k;
  const Geom G = load_geom(a.C, i * d.n2g + j);
  double q[8], U[8];
#pragma unroll
  for (int v = 0; v < 8; v++) { U[v] = a.in[v * d.nz + idx]; q[v] = a.out[v * d.nz + idx]; }
  int its;
  const int f = invert_2d(U, G, a.gam, q, a.nc, its);
#pragma unroll
  for (int v = 0; v < 8; v++) a.out[v * d.nz + idx] = q[v];
  if (a.flag) a.flag[idx] = f;
}

}  // namespace cuharm
