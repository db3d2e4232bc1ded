// cuharm_kernels.cuh — grid kernels of the hot path (S1-S11 of DESIGN.md) other than the flux kernels
// (cuharm_flux.cuh): ghost fill, flux-CT EMFs, fused source+update+inversion+floors, repair of failed zones, CFL and div B
// reductions.  fp64, SoA prim[8][n1g][n2g][n3g] with k (phi) fastest: a warp runs along k at fixed (i,j), so
// every geometry read is a broadcast (the metric is phi-independent).
#pragma once
#include "cuharm_flux.cuh"
#include "cuharm_chain.cuh"

namespace cuharm {

// ---------------------------------------------------------------------------------------------------------
// S1  Boundary conditions (A15).  Order X1, X2, X3, each over the full extended range of the others.
// kind: 0 outflow (+ inflow check in MKS X1), 1 periodic, 2 polar reflection, 3 fixed (ghosts never written).
// `gate`: if non-null and *gate == 0 the kernel does nothing (second ghost fill, needed only after repairs).
// ---------------------------------------------------------------------------------------------------------
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

// ---------------------------------------------------------------------------------------------------------
// S1 in one launch.  The rule (A15) is three fills run one after the other -- X1, then X2, then X3, each over
// the full extended range of the other two directions (the oracle does exactly that) -- so the final content of a
// ghost zone (i, j, k) is a composition: X3 copies from
// (i, j, ks) what X2 left there, which X2 took (with its sign flips / rescaling) from (i, js, ks) as X1 left it,
// which X1 made from the interior zone (is, js, ks).  Every source of that chain is a zone no fill writes
// (interior, or a ghost of a `fixed` direction), so all ghost zones can be produced at once, in place, from the
// same inputs and by the same arithmetic in the same order as the three sequential fills.
// Block rows: first the (i, j) rows that are ghosts in X1 or X2 (whole k range), then the rows interior in (i, j)
// (their 2 ng ghost zones in k only), 21 of those rows per block.
// ---------------------------------------------------------------------------------------------------------
struct BcAllArgs {
  Dims d;
  double* P;
  const Geom* C;
  int kind1, kind2, kind3, coords;
  int kind1_lo, kind1_hi;  // the X1 rule per side: kind1, or 3 (never written) on an internal slab boundary
  double gamma_max;
  const unsigned long long* gate;
  int nrows_a;  // (i, j) rows with a ghost index in X1 or X2
};

__device__ __forceinline__ int bc_source(int x, int n, int ng, int kind, bool reflect_ok) {
  // source index of ghost index x (extended numbering) in a direction with n interior zones
  if (x >= ng && x < ng + n) return x;
  if (kind == 1) {
    const int I = x - ng;
    return ng + ((I % n) + n) % n;
  }
  if (kind == 2 && reflect_ok) return x < ng ? 2 * ng - 1 - x : 2 * (ng + n) - 1 - x;
  return x < ng ? ng : ng + n - 1;
}

__device__ __forceinline__ void bc_zone(const BcAllArgs& a, int i, int j, int k) {
  const Dims& d = a.d;
  const bool gi = (i < d.ng && a.kind1_lo != 3) || (i >= d.ng + d.n1 && a.kind1_hi != 3);
  const bool gj = (j < d.ng || j >= d.ng + d.n2) && a.kind2 != 3;
  const bool gk = (k < d.ng || k >= d.ng + d.n3) && a.kind3 != 3;
  if (!(gi || gj || gk)) return;
  const int is = gi ? bc_source(i, d.n1, d.ng, a.kind1, false) : i;
  const int js = gj ? bc_source(j, d.n2, d.ng, a.kind2, true) : j;
  const int ks = gk ? bc_source(k, d.n3, d.ng, a.kind3, false) : k;
  double q[8];
  const long long src = is * d.s1 + js * d.s2 + ks;
#pragma unroll
  for (int v = 0; v < 8; v++) q[v] = a.P[v * d.nz + src];
  if (gi && a.kind1 == 0) {  // X1 outflow, as seen in row js
    const Geom Gg = load_geom(a.C, i * d.n2g + js);
    const double ratio = __ldg(&a.C[is * d.n2g + js].sg) / Gg.sg;  // sqrt(-g) B^i constant across the copy
    q[5] *= ratio; q[6] *= ratio; q[7] *= ratio;
    if (a.coords == 0) inflow_check(q, Gg, i < d.ng, a.gamma_max);
  }
  if (gj) {  // X2, as seen in column i
    if (a.kind2 == 2) { q[3] = -q[3]; q[6] = -q[6]; }  // utilde^2, B^2 change sign
    if (a.kind2 == 0) {
      const double ratio = __ldg(&a.C[i * d.n2g + js].sg) / __ldg(&a.C[i * d.n2g + j].sg);
      q[5] *= ratio; q[6] *= ratio; q[7] *= ratio;
    }
  }
  const long long dst = i * d.s1 + j * d.s2 + k;
#pragma unroll
  for (int v = 0; v < 8; v++) a.P[v * d.nz + dst] = q[v];
}

__global__ void __launch_bounds__(128) bc_all_kernel(BcAllArgs a) {
  if (a.gate && *a.gate == 0ull) return;
  const Dims& d = a.d;
  const int b = blockIdx.x;
  const int kchunks = (d.n3g + 127) / 128;
  if (b < a.nrows_a * kchunks) {
    // family A: rows with a ghost index in X1 or X2, enumerated as the extended (i, j) plane minus its interior
    const int row = b / kchunks, k = (b - row * kchunks) * 128 + threadIdx.x;
    if (k >= d.n3g) return;
    int i, j;
    const int top = d.ng * d.n2g;                 // rows with i < ng
    const int mid = d.n1 * 2 * d.ng;              // interior i, ghost j
    if (row < top) { i = row / d.n2g; j = row - i * d.n2g; }
    else if (row < top + mid) {
      const int r = row - top;
      i = d.ng + r / (2 * d.ng);
      const int jj = r - (i - d.ng) * 2 * d.ng;
      j = jj < d.ng ? jj : d.n2 + jj;
    } else {
      const int r = row - top - mid;
      i = d.ng + d.n1 + r / d.n2g;
      j = r - (i - d.ng - d.n1) * d.n2g;
    }
    bc_zone(a, i, j, k);
  } else {
    // family B: interior (i, j) rows, their 2 ng ghost zones in k; 21 rows x 6 zones per block (ng = 3)
    const int per = 128 / (2 * d.ng);
    const int slot = threadIdx.x / (2 * d.ng), g = threadIdx.x - slot * 2 * d.ng;
    if (slot >= per) return;
    const long long row = (long long)(b - a.nrows_a * kchunks) * per + slot;
    if (row >= (long long)d.n1 * d.n2) return;
    const int i = d.ng + (int)(row / d.n2), j = d.ng + (int)(row % d.n2);
    const int k = g < d.ng ? g : d.n3 + g;
    bc_zone(a, i, j, k);
  }
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
  const double* srcw;   // [n1g*n2g][14] source weights
  const double* floors;
  int* flag;
  int* list;                    // failed zones of this substep
  unsigned long long* nfail;    // counter of this substep
  unsigned long long* stats;    // [8]
  const double* dt;  // device scalar: the step size of this RK2 step (written before the step by set_dt / dt_from_cw)
  double dtfac;      // dtau = dtfac * *dt: 1/2 in the predictor, 1 in the corrector (eq. 25)
  double idx1, idx2, idx3, gam;
  NewtonCfg nc;
  FloorCfg fc;
  ChainCfg cc;    // fallback chain: when on, U* of every LISTED zone goes to ustar ([8][nz], written sparsely) and
  double* ustar;  // the zones of eq. 33 are listed without trying the 2D method; chain_kernel then works through the list
};

// Per-zone work once the streamed operands are in registers.  pb = P^n, pf = the state the fluxes were built from
// (pf is pb in the predictor), fx[6v..6v+5] = F1[i+1], F1[i], F2[j+1], F2[j], F3[k+1], F3[k] of hydro component v,
// ex = E1 at (0, +j, +k, +j+k), E2 at (0, +i, +k, +i+k), E3 at (0, +i, +j, +i+j).
// -div F of one zone (eq. 25) from its face fluxes and edge EMFs (eq. 22; A3)
__device__ __forceinline__ void zone_divergence(const UpdArgs& a, const double fx[30], const double ex[12], double dU[8]) {
#pragma unroll
  for (int v = 0; v < 5; v++)
    dU[v] = -fma(fx[6 * v] - fx[6 * v + 1], a.idx1,
                 fma(fx[6 * v + 2] - fx[6 * v + 3], a.idx2, (fx[6 * v + 4] - fx[6 * v + 5]) * a.idx3));
  // induction: flux-CT replacement fluxes from the edge EMFs (eq. 22; A3)
  {
    const double e1_00 = ex[0], e1_j = ex[1], e1_k = ex[2], e1_jk = ex[3];
    const double e2_00 = ex[4], e2_i = ex[5], e2_k = ex[6], e2_ik = ex[7];
    const double e3_00 = ex[8], e3_i = ex[9], e3_j = ex[10], e3_ij = ex[11];
    // F~2(B1) = -1/2 (E3 + E3[i+1]) at faces j, j+1;  F~3(B1) = +1/2 (E2 + E2[i+1]) at faces k, k+1
    const double divB1 = ((-0.5 * (e3_j + e3_ij)) - (-0.5 * (e3_00 + e3_i))) * a.idx2 +
                         ((0.5 * (e2_k + e2_ik)) - (0.5 * (e2_00 + e2_i))) * a.idx3;
    // F~1(B2) = +1/2 (E3 + E3[j+1]) at faces i, i+1;  F~3(B2) = -1/2 (E1 + E1[j+1]) at faces k, k+1
    const double divB2 = ((0.5 * (e3_i + e3_ij)) - (0.5 * (e3_00 + e3_j))) * a.idx1 +
                         ((-0.5 * (e1_k + e1_jk)) - (-0.5 * (e1_00 + e1_j))) * a.idx3;
    // F~1(B3) = -1/2 (E2 + E2[k+1]) at faces i, i+1;  F~2(B3) = +1/2 (E1 + E1[k+1]) at faces j, j+1
    const double divB3 = ((-0.5 * (e2_i + e2_ik)) - (-0.5 * (e2_00 + e2_k))) * a.idx1 +
                         ((0.5 * (e1_j + e1_jk)) - (0.5 * (e1_00 + e1_k))) * a.idx2;
    dU[5] = -divB1;
    dU[6] = -divB2;
    dU[7] = -divB3;
  }
}

template <bool SAME, bool CHAIN>
__device__ __forceinline__ void update_zone(const UpdArgs& a, const double pb[8], const double pf[8], const double dU[8],
                                            const Geom& G, const double* cn, double rfl, double ufl, double dtau,
                                            long long idx, int q2, bool live, int cnt[5]) {
  const Dims& d = a.d;
  // U^n, source, update
  State S;
  fluid_state(pb, G, S);
  double U[8];
  flux_vector<0>(pb, S, G, a.gam, U);
  bool ent_first = false;
  if (CHAIN && a.cc.beta_min > 0.0) {  // eq. 33: beta of P^n, p_g / (p_g + b^2/2), IEEE division
    const double pg = (a.gam - 1.0) * pb[1];
    ent_first = pg / (pg + 0.5 * S.bsq) < a.cc.beta_min;
  }
  double src[4];
  if (SAME) {
    source_term(pb, S, G, cn, a.gam, src);
  } else {
    fluid_state(pf, G, S);
    source_term(pf, S, G, cn, a.gam, src);
  }
  U[0] = fma(dtau, dU[0], U[0]);
#pragma unroll
  for (int v = 1; v < 5; v++) U[v] = fma(dtau, src[v - 1] + dU[v], U[v]);
#pragma unroll
  for (int v = 5; v < 8; v++) U[v] = fma(dtau, dU[v], U[v]);
  double pn[8];
#pragma unroll
  for (int v = 0; v < 8; v++) pn[v] = pb[v];  // A35: the guess is P^n
  int its = 0;
  int flag;
  if (CHAIN) {
    if (ent_first) {
      flag = KIND_ENTROPY_FIRST;
      pn[5] = U[5] * G.isg; pn[6] = U[6] * G.isg; pn[7] = U[7] * G.isg;
    } else {
      flag = invert_2d(U, G, a.gam, pn, a.nc, its);
    }
  } else {
    flag = invert_2d(U, G, a.gam, pn, a.nc, its);
  }
  int m = 0;
  if (flag == 0) {
    m = apply_floors(pn, G, a.C + q2, rfl, ufl, a.fc, a.gam, a.nc);
  } else if (live) {
    const unsigned long long pos = atomicAdd(a.nfail, 1ull);
    a.list[pos] = (int)idx;
    if (CHAIN) {  // U* of the LISTED zones only: chain_kernel reads it for no other zone
#pragma unroll
      for (int v = 0; v < 8; v++) a.ustar[v * d.nz + idx] = U[v];
    }
  }
  if (live) {
    a.flag[idx] = flag;
#pragma unroll
    for (int v = 0; v < 8; v++) a.Pout[v * d.nz + idx] = pn[v];
    cnt[0] = m & 1; cnt[1] = (m >> 1) & 1; cnt[2] = (m >> 2) & 1; cnt[3] = (m >> 3) & 1; cnt[4] = its;
  }
}

// statistics: warp sums, one shared-memory atomic per warp and counter, one global atomic per block and counter
__device__ __forceinline__ void update_stats(const UpdArgs& a, const int cnt[5]) {
  __shared__ int sh[5];
  if (threadIdx.x < 5) sh[threadIdx.x] = 0;
  __syncthreads();
#pragma unroll
  for (int c = 0; c < 5; c++) {
    const int s = __reduce_add_sync(0xffffffffu, cnt[c]);
    if ((threadIdx.x & 31) == 0 && s) atomicAdd(&sh[c], s);
  }
  __syncthreads();
  if (threadIdx.x < 5 && sh[threadIdx.x]) atomicAdd(a.stats + 2 + threadIdx.x, (unsigned long long)sh[threadIdx.x]);
}

// Generic kernel: per-thread loads (any n3, any alignment).  One thread per interior zone; out-of-range lanes of the
// ragged tail work on a clamped copy of the last zone and store nothing.
template <bool SAME, bool CHAIN>
__global__ void __launch_bounds__(128, 3) update_kernel(UpdArgs a) {
  const Dims& d = a.d;
  const int k = d.ng + blockIdx.x * 128 + threadIdx.x;
  const int j = d.ng + blockIdx.y, i = d.ng + blockIdx.z;
  const bool live = k < d.ng + d.n3;
  const int kc = live ? k : d.ng + d.n3 - 1;
  const long long idx = i * d.s1 + j * d.s2 + kc;
  const int q2 = i * d.n2g + j;
  double pb[8], pf[8], fx[30], ex[12];
#pragma unroll
  for (int v = 0; v < 8; v++) pb[v] = a.Pbase[v * d.nz + idx];
#pragma unroll
  for (int v = 0; v < 8; v++) pf[v] = SAME ? pb[v] : a.Pflux[v * d.nz + idx];
#pragma unroll
  for (int v = 0; v < 5; v++) {
    const double* f1 = a.F1 + v * d.nz + idx;
    const double* f2 = a.F2 + v * d.nz + idx;
    const double* f3 = a.F3 + v * d.nz + idx;
    fx[6 * v + 0] = __ldg(f1 + d.s1); fx[6 * v + 1] = __ldg(f1);
    fx[6 * v + 2] = __ldg(f2 + d.s2); fx[6 * v + 3] = __ldg(f2);
    fx[6 * v + 4] = __ldg(f3 + 1);    fx[6 * v + 5] = __ldg(f3);
  }
  {
    const double* E1 = a.E + idx; const double* E2 = a.E + d.nz + idx; const double* E3 = a.E + 2 * d.nz + idx;
    ex[0] = __ldg(E1); ex[1] = __ldg(E1 + d.s2); ex[2] = __ldg(E1 + 1); ex[3] = __ldg(E1 + d.s2 + 1);
    ex[4] = __ldg(E2); ex[5] = __ldg(E2 + d.s1); ex[6] = __ldg(E2 + 1); ex[7] = __ldg(E2 + d.s1 + 1);
    ex[8] = __ldg(E3); ex[9] = __ldg(E3 + d.s1); ex[10] = __ldg(E3 + d.s2); ex[11] = __ldg(E3 + d.s1 + d.s2);
  }
  const Geom G = load_geom(a.C, q2);
  double cn[14];
#pragma unroll
  for (int s = 0; s < 7; s++) {
    const double2 v = __ldg(reinterpret_cast<const double2*>(a.srcw + (size_t)q2 * 14) + s);
    cn[2 * s] = v.x; cn[2 * s + 1] = v.y;
  }
  int cnt[5] = {0, 0, 0, 0, 0};
  double dU[8];
  zone_divergence(a, fx, ex, dU);
  update_zone<SAME, CHAIN>(a, pb, pf, dU, G, cn, __ldg(a.floors + 2 * q2), __ldg(a.floors + 2 * q2 + 1), a.dtfac * __ldg(a.dt), idx, q2,
                    live, cnt);
  update_stats(a, cnt);
}

// TMA kernel (n3g even, 16-byte aligned arrays).  The streamed operands of the 128 zones of a block are 63 row
// segments (55 in the predictor) of TB + 4 doubles each, contiguous along k: the lanes of warps 0 and 1 issue one
// 1D bulk copy (cp.async.bulk, global -> shared, completion on an mbarrier) per row, so the whole DRAM footprint of
// the block is in flight at once and holds no registers while it flies.  Every thread then reads its zone (and the
// k-1, k+1 neighbours) from shared memory.  Segment = zones k0-1 .. k0+TB+1 of the row (k0 = first zone of
// the block; the -1 makes the start even, i.e. 16-byte aligned, because ng is odd).
//
// Flux-CT is fused in: instead of the three edge-EMF arrays of emf_kernel the block stages the 22 rows of
// transverse induction fluxes its 12 EMFs per zone are made of and evaluates eq. 21 in place, with the same
// expression (same operand order) wherever an EMF is needed, so every zone that shares an edge gets the same bits
// and div B stays at round-off exactly as with the stored EMFs.
__host__ __device__ constexpr int upd_row(int tb) { return tb + 4; }  // doubles per staged row: 1 + TB + 1 (k+1) + 2 pad, a multiple of 16 B
constexpr int UPD_NROW = 63;   // 8 P^n, 8 P-flux, 10 F1, 10 F2, 5 F3 (hydro), 22 induction-flux rows
constexpr int UPD_TAB = 36;    // doubles of per-(i,j) records staged behind the rows: Geom 20, source weights 14, floors 2
__host__ __device__ constexpr int upd_smem(int tb) { return (UPD_NROW * upd_row(tb) + 2 * 64) * 8; }  // dynamic shared memory per block

// Stage rows: 0..7 P^n; 8..15 P-flux; 16..25 F1 hydro, (i+1, i) per component; 26..35 F2 hydro, (j+1, j) per component;
// 36..40 F3 hydro; induction fluxes (component slots F1: [5] = B2, [6] = B3;  F2: [5] = B3, [6] = B1;  F3: [5] = B1,
// [6] = B2): 41, 42 F2(B3) at j, j+1; 43..45 F3(B2) at j-1, j, j+1; 46..48 F3(B1) at i-1, i, i+1; 49, 50 F1(B3) at
// i, i+1; 51..56 F1(B2) on (i, i+1) x (j-1, j, j+1); 57..62 F2(B1) on (j, j+1) x (i-1, i, i+1).
struct TileIdx { int i, j, c; };  // zone-row (i, j) (interior numbering) and 128-zone chunk of a tile
struct TileCnt { int s, i, jj, c; };  // mixed-radix tile counter: j-strip, i, j within the strip, chunk

// The tile walk of the two staged update kernels (update_tma_kernel here, update_tmap_kernel in cuharm_update_tmap.cuh).
// Tile order: strips of wj rows j; inside a strip i runs slower than j, the chunk fastest.  The blocks resident at one
// time then cover a patch of (several i) x (wj j) rows, so the rows a tile shares with its i- and j-neighbours (F1[i+1],
// F2[j+1], the induction fluxes around each edge) are re-read while still in L2.  The first tile of a block and the
// stride G between its tiles are decomposed once; after that the counter is carried (no division in the tile loop).
struct TileWalk {
  TileCnt cur, dlt;
  int nch, wj, n1;
  __device__ __forceinline__ TileWalk(int tile, int G, int nch_, int wj_, int n1_) : nch(nch_), wj(wj_), n1(n1_) {
    int r = tile;
    cur.c = r % nch; r /= nch; cur.jj = r % wj; r /= wj; cur.i = r % n1; cur.s = r / n1;
    r = G;
    dlt.c = r % nch; r /= nch; dlt.jj = r % wj; r /= wj; dlt.i = r % n1; dlt.s = r / n1;
  }
  __device__ __forceinline__ void advance() {
    TileCnt y{cur.s + dlt.s, cur.i + dlt.i, cur.jj + dlt.jj, cur.c + dlt.c};
    if (y.c >= nch) { y.c -= nch; y.jj++; }
    if (y.jj >= wj) { y.jj -= wj; y.i++; }
    if (y.i >= n1) { y.i -= n1; y.s++; }
    cur = y;
  }
  __device__ __forceinline__ TileIdx idx() const { return TileIdx{cur.i, cur.s * wj + cur.jj, cur.c}; }
};

// Eq. 21 (A3) on the twelve edges of a zone, from the staged induction fluxes: the expressions and the
// operand order of emf_kernel, written once for both staged kernels.  `S` maps a logical operand -- which induction
// flux, and its offsets from the zone in the two directions it is indexed by here -- to the kernel's own stage layout:
//   S::template at<ARRAY, A, B>()   ARRAY = one of the EMF_* below; (A, B) = (dj, dk) for F2B3 / F3B2, (di, dk) for
//                                   F3B1 / F1B3, (di, dj) for F1B2 / F2B1
// ex[0..3] = E1 at (j, k), (j+1, k), (j, k+1), (j+1, k+1); ex[4..7] = E2 at (i, k), (i+1, k), (i, k+1), (i+1, k+1);
// ex[8..11] = E3 at (i, j), (i+1, j), (i, j+1), (i+1, j+1).
enum { EMF_F2B3 = 0, EMF_F3B2, EMF_F3B1, EMF_F1B3, EMF_F1B2, EMF_F2B1 };
template <int A, int B, class S>
__device__ __forceinline__ void edge_emf_triple(const S& st, double ex[12]) {
  // E1(j',k') = (F2B3[j'][k'] + F2B3[j'][k'-1] - F3B2[j'][k'] - F3B2[j'-1][k']) / 4
  ex[A + 2 * B] = 0.25 * (st.template at<EMF_F2B3, A, B>() + st.template at<EMF_F2B3, A, B - 1>() -
                          st.template at<EMF_F3B2, A, B>() - st.template at<EMF_F3B2, A - 1, B>());
  // E2(i',k') = (F3B1[i'][k'] + F3B1[i'-1][k'] - F1B3[i'][k'] - F1B3[i'][k'-1]) / 4
  ex[4 + A + 2 * B] = 0.25 * (st.template at<EMF_F3B1, A, B>() + st.template at<EMF_F3B1, A - 1, B>() -
                              st.template at<EMF_F1B3, A, B>() - st.template at<EMF_F1B3, A, B - 1>());
  // E3(i',j') = (F1B2[i'][j'] + F1B2[i'][j'-1] - F2B1[i'][j'] - F2B1[i'-1][j']) / 4
  ex[8 + A + 2 * B] = 0.25 * (st.template at<EMF_F1B2, A, B>() + st.template at<EMF_F1B2, A, B - 1>() -
                              st.template at<EMF_F2B1, A, B>() - st.template at<EMF_F2B1, A - 1, B>());
}
template <class S>
__device__ __forceinline__ void edge_emfs(const S& st, double ex[12]) {
  edge_emf_triple<0, 0>(st, ex);
  edge_emf_triple<1, 0>(st, ex);
  edge_emf_triple<0, 1>(st, ex);
  edge_emf_triple<1, 1>(st, ex);
}

// stage layout of update_tma_kernel (row table above): rows of UPD_ROW doubles, z = this zone in row 0
template <int UPD_ROW>
struct RowStage {
  const double* z;
  template <int ARR, int A, int B>
  __device__ __forceinline__ double at() const {
    constexpr int row = ARR == EMF_F2B3 ? 41 + A : ARR == EMF_F3B2 ? 44 + A : ARR == EMF_F3B1 ? 47 + A : ARR == EMF_F1B3 ? 49 + A
                        : ARR == EMF_F1B2 ? 51 + 3 * A + (B + 1) : 57 + 3 * B + (A + 1);
    constexpr int off = ARR == EMF_F1B2 || ARR == EMF_F2B1 ? 0 : B;   // E3's operands sit at the zone's own k
    return z[row * UPD_ROW + off];
  }
};

// Persistent blocks: block b takes tiles b, b + gridDim.x, ...; tile = (i, j, 128-zone chunk of the row), chunk
// fastest.  One stage per block: the stage is free again as soon as every thread has moved its operands to
// registers, which is the first thing a tile does, so the copies of tile n+1 fly during the whole of tile n's
// arithmetic; UPD_TMA_MINB blocks of 128 threads per SM keep that many tiles in flight and enough warps for the
// (serial) Newton iteration.
constexpr int UPD_TMA_MINB = 3;
// TB = zones (threads) per tile: 128, or 64 for short rows (n3 <= 64), which would leave half a 128-zone tile idle.
template <bool SAME, int TB, bool CHAIN>
__global__ void __launch_bounds__(TB, (UPD_TMA_MINB * 128) / TB) update_tma_kernel(UpdArgs a, int ntiles, int nch, int wj) {
  constexpr int UPD_ROW = upd_row(TB);
  extern __shared__ __align__(128) double rows[];  // [UPD_NROW][UPD_ROW]
  __shared__ __align__(8) unsigned long long mbar[2];  // [0] copies landed (tx count), [1] stage released (TB arrivals)
  const Dims& d = a.d;
  const int t = threadIdx.x;
  const int G = gridDim.x;
  const unsigned bar0 = smem_u32(&mbar[0]);
  if (t == 0) {
    mbar_init(bar0, 1);
    mbar_init(bar0 + 8, TB);
    mbar_fence_init();
  }
  __syncthreads();
  int tile = blockIdx.x;
  TileWalk walk(tile, G, nch, wj, d.n1);  // strip order (see TileWalk)
  TileIdx cur = walk.idx(), nxt;
  auto tile_base = [&](const TileIdx& x) {  // element offset of the first staged zone of the tile's row
    return (long long)(d.ng + x.i) * d.s1 + (long long)(d.ng + x.j) * d.s2 + (d.ng + x.c * TB - 1);
  };
  auto tile_bytes = [&](const TileIdx& x) {  // staged zones per row (even count) x 8
    return (unsigned)min(UPD_ROW - 2, d.n3g - (d.ng + x.c * TB - 1)) * 8u;
  };
  // Every warp issues its share of the tile's copies with warp-uniform operands (addresses from kernel parameters
  // and the tile indices), so each bulk copy is a handful of uniform-datapath instructions; per-lane operands would
  // make the compiler serialise the lanes in an elect loop that waits on the previous copy.
  constexpr int NWARP = TB / 32;
  double* const tab = rows + UPD_NROW * UPD_ROW;  // two slots of [20] geometry record, [14] source weights, [2] floors
  // Rows are dealt to the warps in four groups of contiguous stage rows (two groups for 64-thread blocks), and
  // inside a group the source addresses are walked with running byte pointers (one 64-bit add per row or less),
  // following the row table above.
  const long long nz8 = d.nz * 8, s18 = d.s1 * 8, s28 = d.s2 * 8;
  const unsigned rowb = UPD_ROW * 8u;
  const unsigned stage0 = smem_u32(rows);
  auto put = [&](int r, const char* src, unsigned bytes) { bulk_g2s(stage0 + r * rowb, src, bytes, bar0); };
  auto issue_group = [&](int grp, unsigned bytes, long long base8) {
    if (grp == 0) {  // rows 0..15: P^n, P-flux
      const char* pb = reinterpret_cast<const char*>(a.Pbase) + base8;
#pragma unroll
      for (int v = 0; v < 8; v++) { put(v, pb, bytes); pb += nz8; }
      if (!SAME) {
        const char* pf = reinterpret_cast<const char*>(a.Pflux) + base8;
#pragma unroll
        for (int v = 0; v < 8; v++) { put(8 + v, pf, bytes); pf += nz8; }
      }
    } else if (grp == 1) {  // rows 16..35: hydro fluxes of directions 1 and 2, (upper face, lower face) per component
      const char* f1 = reinterpret_cast<const char*>(a.F1) + base8;
      const char* f2 = reinterpret_cast<const char*>(a.F2) + base8;
#pragma unroll
      for (int v = 0; v < 5; v++) {
        put(16 + 2 * v, f1 + s18, bytes); put(17 + 2 * v, f1, bytes); f1 += nz8;
        put(26 + 2 * v, f2 + s28, bytes); put(27 + 2 * v, f2, bytes); f2 += nz8;
      }
    } else if (grp == 2) {  // rows 36..50: hydro fluxes of direction 3; induction fluxes F2(B3), F3(B2), F3(B1), F1(B3)
      const char* f3 = reinterpret_cast<const char*>(a.F3) + base8;
#pragma unroll
      for (int v = 0; v < 5; v++) { put(36 + v, f3, bytes); f3 += nz8; }
      // f3 now points at component 5 = F3(B1); component 6 = F3(B2) is one array further
      put(46, f3 - s18, bytes); put(47, f3, bytes); put(48, f3 + s18, bytes);
      f3 += nz8;
      put(43, f3 - s28, bytes); put(44, f3, bytes); put(45, f3 + s28, bytes);
      const char* f2b3 = reinterpret_cast<const char*>(a.F2) + base8 + 5 * nz8;
      put(41, f2b3, bytes); put(42, f2b3 + s28, bytes);
      const char* f1b3 = reinterpret_cast<const char*>(a.F1) + base8 + 6 * nz8;
      put(49, f1b3, bytes); put(50, f1b3 + s18, bytes);
    } else {  // rows 51..62: F1(B2) on (i..i+1) x (j-1..j+1), F2(B1) on (i-1..i+1) x (j..j+1)
      const char* f1b2 = reinterpret_cast<const char*>(a.F1) + base8 + 5 * nz8 - s28;
#pragma unroll
      for (int q = 0; q < 3; q++) { put(51 + q, f1b2, bytes); put(54 + q, f1b2 + s18, bytes); f1b2 += s28; }
      const char* f2b1 = reinterpret_cast<const char*>(a.F2) + base8 + 6 * nz8 - s18;
#pragma unroll
      for (int q = 0; q < 3; q++) { put(57 + q, f2b1, bytes); put(60 + q, f2b1 + s28, bytes); f2b1 += s18; }
    }
  };
  auto issue = [&](const TileIdx& x, int slot) {  // all warps; lane 0 of each issues
    if ((t & 31) != 0) return;
    const unsigned bytes = tile_bytes(x);
    const long long base8 = tile_base(x) * 8;
    const int w = t >> 5;
    if (w == 0) mbar_expect_tx(bar0, bytes * (SAME ? UPD_NROW - 8 : UPD_NROW) + UPD_TAB * 8u);
    if (NWARP == 4) {
      issue_group(w, bytes, base8);
    } else {  // two warps: groups (0, 2) and (1, 3)
      issue_group(w, bytes, base8);
      issue_group(w + 2, bytes, base8);
    }
    if (w == NWARP - 1) {
      const size_t q = (size_t)(d.ng + x.i) * d.n2g + (d.ng + x.j);
      double* const tb = tab + slot * 64;
      bulk_g2s(smem_u32(tb), a.C + q, 160u, bar0);
      bulk_g2s(smem_u32(tb + 20), a.srcw + q * 14, 112u, bar0);
      bulk_g2s(smem_u32(tb + 34), a.floors + q * 2, 16u, bar0);
    }
  };
  if (tile < ntiles) issue(cur, 0);
  const double dtau = a.dtfac * __ldg(a.dt);
  int cnt_acc[5] = {0, 0, 0, 0, 0};
  for (int n = 0; tile < ntiles; tile += G, n++, cur = nxt) {
    walk.advance();
    nxt = walk.idx();
    const int j = d.ng + cur.j, i = d.ng + cur.i;
    const int k0 = d.ng + cur.c * TB;
    const bool live = k0 + t < d.ng + d.n3;
    const int tc = live ? t : d.ng + d.n3 - 1 - k0;  // clamped lane position
    const long long idx = i * d.s1 + j * d.s2 + k0 + tc;
    const int q2 = i * d.n2g + j;
    mbar_wait(bar0, n & 1);
    const double* z = rows + 1 + tc;  // this zone in row 0 of the stage
#define ROWZ(r, o) z[(r) * UPD_ROW + (o)]
    double pb[8], pf[8], fx[30], ex[12];
#pragma unroll
    for (int v = 0; v < 8; v++) pb[v] = ROWZ(v, 0);
#pragma unroll
    for (int v = 0; v < 8; v++) pf[v] = SAME ? pb[v] : ROWZ(8 + v, 0);
#pragma unroll
    for (int v = 0; v < 5; v++) {
      fx[6 * v + 0] = ROWZ(16 + 2 * v, 0); fx[6 * v + 1] = ROWZ(17 + 2 * v, 0);
      fx[6 * v + 2] = ROWZ(26 + 2 * v, 0); fx[6 * v + 3] = ROWZ(27 + 2 * v, 0);
      fx[6 * v + 4] = ROWZ(36 + v, 1);     fx[6 * v + 5] = ROWZ(36 + v, 0);
    }
    edge_emfs(RowStage<UPD_ROW>{z}, ex);  // eq. 21
#undef ROWZ
    // Every thread now holds its operands: once all have arrived the stage can be refilled.  The barrier is split
    // (arrive here, wait after the divergence arithmetic), so nobody idles while the last warp finishes its reads.
    mbar_arrive(bar0 + 8);
    double dU[8];
    zone_divergence(a, fx, ex, dU);
    mbar_wait(bar0 + 8, n & 1);
    if (tile + G < ntiles) issue(nxt, (n + 1) & 1);
    int cnt[5] = {0, 0, 0, 0, 0};
    // the per-(i,j) records of this tile stay valid in their own (double-buffered) slot for the whole tile
    const double* tb = tab + (n & 1) * 64;
    const Geom Gc = load_geom_shared(tb);
    update_zone<SAME, CHAIN>(a, pb, pf, dU, Gc, tb + 20, tb[34], tb[35], dtau, idx, q2, live, cnt);
#pragma unroll
    for (int q = 0; q < 5; q++) cnt_acc[q] += cnt[q];
  }
  update_stats(a, cnt_acc);
}

// ---------------------------------------------------------------------------------------------------------
// S8  Repair of zones whose inversion failed (eq. 34; A13): deterministic Jacobi passes over the
// list of failed zones.  Pass m: a still-bad zone whose 4 face neighbours in the (I,J) plane were all
// good at the start of the pass takes their mean; else the 4 diagonal neighbours; else it waits; in the last
// pass leftovers take the mean of whatever good zones exist among the 8 neighbours.  Only rho, u, utilde^i are
// replaced; floors are re-applied to the repaired zone.  flag > 0: bad; flag = -(m+1): repaired in
// pass m, i.e. good from pass m+1 on -- which is what makes the passes Jacobi without a snapshot: donors are
// zones that are not written in the current pass.
//
// Grid-wide: the list is dealt to min(gridDim.x, ceil(nf / 512)) blocks (the others leave at once), and the passes
// are separated by a grid barrier on a device counter (monotonic, zeroed with the per-step counters).  The kernel is
// launched COOPERATIVELY (cuharm_api.cu: launch_fixup), with at most one block per multiprocessor, so the driver
// guarantees that the participating blocks are resident together -- also when several contexts repair on several
// streams at once.  With nothing failed (every step of the torus workloads' first
// 1000) the kernel is one read and an exit; with a handful of failures one block does the work without touching the
// barrier; a step with 1e6 failures is spread over the whole device.  Reads of flags and donors bypass L1 (other
// blocks write them between passes).
// ---------------------------------------------------------------------------------------------------------
struct FixArgs {
  Dims d;
  double* P;
  int* flag;
  const int* list;
  const unsigned long long* nfail;   // entries of the list
  const unsigned long long* nbad;    // zones still failed after the fallback chain (null: every entry of the list)
  unsigned long long* stats;
  unsigned long long* sync;          // [0] barrier counter, [1 + pass] zones left waiting after pass
  const Geom* C;
  const double* floors;
  int max_passes;
  double gam;
  NewtonCfg nc;
  FloorCfg fc;
};

__device__ __forceinline__ bool zone_good(int f, int pass) { return f == 0 || (f < 0 && -f - 1 < pass); }

constexpr int FIX_THREADS = 512;

__device__ __forceinline__ void fix_grid_barrier(unsigned long long* bar, unsigned long long target) {
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(bar, 1ull);
    while (*reinterpret_cast<volatile unsigned long long*>(bar) < target) __nanosleep(64);
    __threadfence();
  }
  __syncthreads();
}

// One zone of the list in one pass: 0 nothing to do (already repaired), 1 repaired, 2 repaired by the last-resort rule,
// 3 left waiting.
__device__ __forceinline__ int fix_one(const FixArgs& a, long long idx, int pass, bool last) {
  const Dims& d = a.d;
  if (__ldcg(a.flag + idx) <= 0) return 0;
  const long long fo[4] = {d.s1, -d.s1, d.s2, -d.s2};
  const long long dg[4] = {d.s1 + d.s2, d.s1 - d.s2, -d.s1 + d.s2, -d.s1 - d.s2};
  bool fg = true, dgood = true;
#pragma unroll
  for (int m = 0; m < 4; m++) {
    fg = fg && zone_good(__ldcg(a.flag + idx + fo[m]), pass);
    dgood = dgood && zone_good(__ldcg(a.flag + idx + dg[m]), pass);
  }
  double q[8];
  int what = 1;
  if (fg || dgood) {
    const long long* st = fg ? fo : dg;
#pragma unroll
    for (int v = 0; v < 5; v++) {
      double s = 0.0;
#pragma unroll
      for (int m = 0; m < 4; m++) s += __ldcg(a.P + v * d.nz + idx + st[m]);
      q[v] = 0.25 * s;
    }
  } else if (last) {
    int cnt = 0;
    double s[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    for (int di = -1; di <= 1; di++)
      for (int dj = -1; dj <= 1; dj++) {
        if (!di && !dj) continue;
        const long long n = idx + di * d.s1 + dj * d.s2;
        if (!zone_good(__ldcg(a.flag + n), pass)) continue;
        cnt++;
#pragma unroll
        for (int v = 0; v < 5; v++) s[v] += __ldcg(a.P + v * d.nz + n);
      }
#pragma unroll
    for (int v = 0; v < 5; v++) q[v] = cnt > 0 ? s[v] / cnt : __ldcg(a.P + v * d.nz + idx);
    what = 2;
  } else {
    return 3;
  }
#pragma unroll
  for (int v = 5; v < 8; v++) q[v] = __ldcg(a.P + v * d.nz + idx);
  const int q2 = (int)(idx / d.s2);  // = i * n2g + j
  const Geom G = load_geom(a.C, q2);
  apply_floors(q, G, a.C + q2, a.floors[2 * q2], a.floors[2 * q2 + 1], a.fc, a.gam, a.nc);
#pragma unroll
  for (int v = 0; v < 5; v++) a.P[v * d.nz + idx] = q[v];
  a.flag[idx] = -(pass + 1);
  return what;
}

__global__ void __launch_bounds__(FIX_THREADS) fixup_kernel(FixArgs a) {
  const unsigned long long nf = *a.nfail;
  if (nf == 0ull) return;
  const unsigned long long want = (nf + FIX_THREADS - 1) / FIX_THREADS;
  const unsigned nb = (unsigned)(want < gridDim.x ? want : gridDim.x);  // participating blocks
  if (blockIdx.x >= nb) return;
  if (blockIdx.x == 0 && threadIdx.x == 0) atomicAdd(a.stats + 0, a.nbad ? *a.nbad : nf);
  unsigned long long repaired = 0ull, lastres = 0ull;
  const unsigned long long stride = (unsigned long long)nb * FIX_THREADS;
  for (int pass = 0; pass <= a.max_passes; pass++) {
    const bool last = pass == a.max_passes;
    int left = 0;
    for (unsigned long long e = (unsigned long long)blockIdx.x * FIX_THREADS + threadIdx.x; e < nf; e += stride) {
      const int w = fix_one(a, a.list[e], pass, last);
      repaired += w == 1 || w == 2;
      lastres += w == 2;
      left |= w == 3;
    }
    if (last) break;
    // anything left waiting anywhere?  (one atomic per block that has some; read after the barrier)
    const int any = __syncthreads_or(left);
    if (nb == 1) {
      __threadfence_block();
      if (!any) break;
    } else {
      if (any && threadIdx.x == 0) atomicAdd(a.sync + 1 + pass, 1ull);
      fix_grid_barrier(a.sync, (unsigned long long)nb * (pass + 1));
      if (__ldcg(a.sync + 1 + pass) == 0ull) break;
    }
  }
  if (repaired) atomicAdd(a.stats + 1, repaired);
  if (lastres) atomicAdd(a.stats + 7, lastres);
}

// One Jacobi pass as a launch of its own (cuharm_repair_pass): for a caller that refreshes the halo planes of the
// primitives and of the flags between the passes (slab decomposition), so that a repair next to an internal boundary sees
// its neighbours exactly as the single-domain repair does.  out[0] = entries of the list, out[1] = zones left waiting.
__global__ void __launch_bounds__(256) fixup_pass_kernel(FixArgs a, int pass, unsigned long long* out) {
  const unsigned long long nf = *a.nfail;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    out[0] = nf;
    if (pass == 0 && nf) atomicAdd(a.stats + 0, a.nbad ? *a.nbad : nf);
  }
  unsigned long long repaired = 0ull, lastres = 0ull, left = 0ull;
  for (unsigned long long e = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; e < nf;
       e += (unsigned long long)gridDim.x * blockDim.x) {
    const int w = fix_one(a, a.list[e], pass, pass == a.max_passes);
    repaired += w == 1 || w == 2;
    lastres += w == 2;
    left += w == 3;
  }
  if (repaired) atomicAdd(a.stats + 1, repaired);
  if (lastres) atomicAdd(a.stats + 7, lastres);
  if (left) atomicAdd(out + 1, left);
}

// P:L311 (A16): utilde^2 of the two zones nearest each pole <- the straight line in X^2 through zero at the pole and
// the value of the third zone of the same (i, k): weights (m + 1/2) / (2 + 1/2), m = 0, 1 (uniform spacing in X^2).
// One thread per (i, k) and pole.  Runs on the output of the update kernel, before the ghost fill.
__global__ void __launch_bounds__(128) polar_damp_kernel(Dims d, double* P) {
  const int k = d.ng + blockIdx.x * 128 + threadIdx.x;
  if (k >= d.ng + d.n3) return;
  const int i = d.ng + blockIdx.y;
  double* u2 = P + 3 * d.nz + i * d.s1 + k;
  const bool south = blockIdx.z != 0;
  const int j2 = south ? d.ng + d.n2 - 3 : d.ng + 2;   // anchor row
  const int step = south ? 1 : -1;                      // towards the pole
  const double a = u2[j2 * d.s2];
  u2[(j2 + step) * d.s2] = a * (1.5 / 2.5);
  u2[(j2 + 2 * step) * d.s2] = a * (0.5 / 2.5);
}

// Stage-level test helper (cuharm_repair): the list of failed zones from a caller's flag array (interior zones with
// flag > 0 -> list, everything else -> 0 in the library's own flag array), so that fixup_kernel can be run on any
// pattern of failures.  The order of the list is irrelevant: the passes are Jacobi.
__global__ void __launch_bounds__(128) repair_list_kernel(Dims d, const int* flag_in, int* flag, int* list, unsigned long long* nfail) {
  const int k = blockIdx.x * 128 + threadIdx.x;
  if (k >= d.n3g) return;
  const int j = blockIdx.y, i = blockIdx.z;
  const long long idx = i * d.s1 + j * d.s2 + k;
  const bool in = i >= d.ng && i < d.ng + d.n1 && j >= d.ng && j < d.ng + d.n2 && k >= d.ng && k < d.ng + d.n3;
  const int f = in && flag_in[idx] > 0 ? flag_in[idx] : 0;
  flag[idx] = f;
  if (f) list[atomicAdd(nfail, 1ull)] = (int)idx;
}

// ---------------------------------------------------------------------------------------------------------
// S10  The step size lives in a device scalar, so that one recorded CUDA graph serves every dt (eq. 26 gives a new
// one every step).  clock[0] = dt of the current step, clock[1] = time integrated so far.
// set_dt_kernel: dt chosen by the caller.  dt_from_cw_kernel: eq. 26 from the c_w maxima the predictor of the
// previous step recorded ("the next time step"), with the host formula of cuharm_last_cfl_dt written out in
// the same order (IEEE divisions, no contraction possible) and with the same guard, so host and device agree bit for bit.
// ---------------------------------------------------------------------------------------------------------
__global__ void set_dt_kernel(double* clock, double dt) {
  clock[0] = dt;
  clock[1] += dt;
}

__global__ void dt_from_cw_kernel(double* clock, const unsigned long long* cw, double xi, double dx1, double dx2, double dx3,
                                  double dt_max) {
  const double dx[3] = {dx1, dx2, dx3};
  double inv = 0.0;
  for (int c = 0; c < 3; c++) {
    const double cwc = __longlong_as_double((long long)cw[c]);
    const double dtl = xi * dx[c] / cwc;  // dt^l = xi dx^l / max c_w
    inv += 1.0 / dtl;                     // eq. 26
  }
  double dt = 1.0 / inv;
  if (dt_max > 0.0 && dt > dt_max) dt = dt_max;
  // the host's guard (dt_of_cw): a non-finite speed (a NaN enters the maxima as +inf) or no speed at all with no cap
  // gives dt = 0 -- the step that follows leaves the state where it is and the clock does not advance, which
  // cuharm_get_time shows as dt_last = 0
  if (!(dt > 0.0) || isinf(dt)) dt = 0.0;
  clock[0] = dt;
  clock[1] += dt;
}

// ---------------------------------------------------------------------------------------------------------
// S9 as a stage of its own (test helper cuharm_apply_floors): eq. 35 floors, eqs. 36-37 ceilings, Lorentz cap on
// every interior zone of an arbitrary primitive array; mask[zone] = the bit mask of apply_floors.
// ---------------------------------------------------------------------------------------------------------
struct FloorArgs {
  Dims d;
  double* P;
  int* mask;
  const Geom* C;
  const double* floors;
  double gam;
  NewtonCfg nc;
  FloorCfg fc;
};

__global__ void __launch_bounds__(128) floors_kernel(FloorArgs a) {
  const Dims& d = a.d;
  const int k = d.ng + blockIdx.x * 128 + threadIdx.x;
  if (k >= d.ng + d.n3) return;
  const int j = d.ng + blockIdx.y, i = d.ng + blockIdx.z;
  const long long idx = i * d.s1 + j * d.s2 + k;
  const int q2 = i * d.n2g + j;
  const Geom G = load_geom(a.C, q2);
  double q[8];
#pragma unroll
  for (int v = 0; v < 8; v++) q[v] = a.P[v * d.nz + idx];
  const int m = apply_floors(q, G, a.C + q2, __ldg(a.floors + 2 * q2), __ldg(a.floors + 2 * q2 + 1), a.fc, a.gam, a.nc);
#pragma unroll
  for (int v = 0; v < 8; v++) a.P[v * d.nz + idx] = q[v];
  if (a.mask) a.mask[idx] = m;
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
    // corners whose terms sum to < 1e-290 are skipped (A4): subnormal-range terms carry no relative precision
    mnorm = A > 1e-290 ? fabs(D) / A : 0.0;
  }
  atomic_max_nonneg(a.out + 0, mabs);
  atomic_max_nonneg(a.out + 1, mnorm);
}

// ---------------------------------------------------------------------------------------------------------
// Fluxes through the shell of zone centres of radial index i (eqs. 43-46):
// Mdot = sum sqrt(-g) rho u^1, phi_B = 1/2 sum sqrt(-g) |B^1|, Ldot = sum sqrt(-g) T^1_phi, Edot = -sum sqrt(-g) T^1_t,
// each times dX2 dX3.  Deterministic two-level sum: block j reduces its row along k in a fixed tree order into
// partial[j][4]; shell_sum_kernel (one block) reduces over j the same way.  No floating-point atomics.
// ---------------------------------------------------------------------------------------------------------
struct ShellArgs {
  Dims d;
  const double* P;
  const Geom* C;
  int i;        // zone index including ghosts
  double gam, dA;
  double* partial;  // [n2][4]
  double* out;      // [4]
};

__device__ __forceinline__ void block_sum4(double v[4], double (*sh)[4]) {
  // fixed-order tree over the 128 threads of the block; result in sh[0]
  const int t = threadIdx.x;
#pragma unroll
  for (int c = 0; c < 4; c++) sh[t][c] = v[c];
  __syncthreads();
  for (int s = 64; s > 0; s >>= 1) {
    if (t < s) {
#pragma unroll
      for (int c = 0; c < 4; c++) sh[t][c] += sh[t + s][c];
    }
    __syncthreads();
  }
}

__global__ void __launch_bounds__(128) shell_flux_kernel(ShellArgs a) {
  __shared__ double sh[128][4];
  const Dims& d = a.d;
  const int j = d.ng + blockIdx.x;
  const Geom G = load_geom(a.C, a.i * d.n2g + j);
  double acc[4] = {0.0, 0.0, 0.0, 0.0};
  for (int k = d.ng + threadIdx.x; k < d.ng + d.n3; k += 128) {
    const long long idx = a.i * d.s1 + j * d.s2 + k;
    double q[8], F[8];
#pragma unroll
    for (int v = 0; v < 8; v++) q[v] = a.P[v * d.nz + idx];
    State S;
    fluid_state(q, G, S);
    flux_vector<1>(q, S, G, a.gam, F);  // sqrt(-g) x (rho u^1, T^1_t, T^1_1, T^1_2, T^1_3, ...)
    acc[0] += F[0] * a.dA;
    acc[1] += 0.5 * G.sg * fabs(q[5]) * a.dA;
    acc[2] += F[4] * a.dA;
    acc[3] += -F[1] * a.dA;
  }
  block_sum4(acc, sh);
  if (threadIdx.x < 4) a.partial[blockIdx.x * 4 + threadIdx.x] = sh[0][threadIdx.x];
}

__global__ void __launch_bounds__(128) shell_sum_kernel(ShellArgs a) {
  __shared__ double sh[128][4];
  double acc[4] = {0.0, 0.0, 0.0, 0.0};
  for (int j = threadIdx.x; j < a.d.n2; j += 128) {
#pragma unroll
    for (int c = 0; c < 4; c++) acc[c] += a.partial[j * 4 + c];
  }
  block_sum4(acc, sh);
  if (threadIdx.x < 4) a.out[threadIdx.x] = sh[0][threadIdx.x];
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
