// cuharm_flux.cuh — S2+S3: reconstruction + Riemann flux of one direction (eqs. 15-20; PPM: A20).
//
// Face (i,j,k) = LOWER DIR-face of zone (i,j,k); its left state is the upper-edge value of zone -1 along DIR, its
// right state the lower-edge value of the zone itself (eq. 16).  Faces lo..hi of the direction, one transverse
// ghost layer (for the EMF average).  Output F[c][zone]: c = 0..4 hydro components, c = 5,6 the induction fluxes of
// B^{DIR+1}, B^{DIR+2} (cyclic); the flux of B^{DIR} is replaced by zero in flux-CT (eq. 22) and never stored.
// STAGE = true (test helper cuharm_flux_dir): all 8 components + c_w per face.
//
// The fp64 pipe bounds these kernels, so the thread mapping follows the direction in a way
// that reconstructs every cell ONCE:
//   directions 1, 2: a thread owns one (transverse index, k) column and MARCHES along the direction, carrying the
//     MC slope, the unlimited PPM edge value and the limited upper-edge state of the previous cell in registers;
//     k is the lane index, so every load and store is coalesced and the face geometry is a broadcast;
//   direction 3: a lane owns one cell along k; the neighbour's slope, edge value and limited state arrive by warp
//     shuffle; a warp of 32 cells yields 29 (PPM) or 31 (PLM) faces, consecutive warps overlap by the difference.
#pragma once
#include "cuharm_phys.cuh"

namespace cuharm {

struct Dims {
  int n1, n2, n3, ng;
  int n1g, n2g, n3g;
  long long s1, s2;  // element strides of i and j (k has stride 1)
  long long nz;      // zones per variable, ghosts included
};

__device__ __forceinline__ unsigned long long warp_max_ull(unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long w = __shfl_xor_sync(0xffffffffu, v, o);
    v = w > v ? w : v;
  }
  return v;
}

// max of non-negative doubles through their order-preserving integer image; no floating-point atomics anywhere.
// Must be reached by all 32 lanes of the warp.
__device__ __forceinline__ void atomic_max_nonneg(unsigned long long* addr, double v) {
  const unsigned long long m = warp_max_ull((unsigned long long)__double_as_longlong(v >= 0.0 ? v : 0.0));
  if ((threadIdx.x & 31) == 0 && m > *reinterpret_cast<volatile unsigned long long*>(addr)) atomicMax(addr, m);
}

struct FluxArgs {
  Dims d;
  const double* P;
  const Geom* Gf;  // geometry at this direction's faces
  double* F;       // [7][nz] (or [8][nz] if STAGE)
  double* cw;      // STAGE only (may be null)
  unsigned long long* cwmax;
  double gam;
  int lo1, lo2, lo3, hi1, hi2, hi3;  // inclusive face ranges in i, j, k
  int seg;                           // marching kernels: faces per segment (blockIdx.y = segment)
};

template <int DIR, bool STAGE>
__device__ __forceinline__ void store_flux(const FluxArgs& a, long long idx, const double F[8], double cwv) {
  const long long nz = a.d.nz;
  if (STAGE) {
#pragma unroll
    for (int v = 0; v < 8; v++) a.F[v * nz + idx] = F[v];
    if (a.cw) a.cw[idx] = cwv;
  } else {
#pragma unroll
    for (int v = 0; v < 5; v++) a.F[v * nz + idx] = F[v];
    a.F[5 * nz + idx] = F[5 + (DIR % 3)];        // B^{DIR+1}
    a.F[6 * nz + idx] = F[5 + ((DIR + 1) % 3)];  // B^{DIR+2}
  }
}

// ---------------------------------------------------------------------------------------------------------
// Directions 1 and 2: marching.  grid.x covers the flattened (transverse index, k) plane, grid.y the segments.
// ---------------------------------------------------------------------------------------------------------
template <int DIR, int RECON, int RIEMANN, bool STAGE>
__global__ void __launch_bounds__(128) flux_march_kernel(FluxArgs a) {
  static_assert(DIR == 1 || DIR == 2, "marching kernel: directions 1 and 2");
  const Dims& d = a.d;
  const int nk = a.hi3 - a.lo3 + 1;
  const int nt = DIR == 1 ? (a.hi2 - a.lo2 + 1) : (a.hi1 - a.lo1 + 1);
  const int q = blockIdx.x * 128 + threadIdx.x;
  double cwv = 0.0;
  if (q < nt * nk) {
    const int t = (DIR == 1 ? a.lo2 : a.lo1) + q / nk;
    const int k = a.lo3 + q % nk;
    const long long sd = DIR == 1 ? d.s1 : d.s2;
    const long long nz = d.nz;
    const int flo = DIR == 1 ? a.lo1 : a.lo2, fhi = DIR == 1 ? a.hi1 : a.hi2;
    const int fa = flo + blockIdx.y * a.seg;
    const int fb = min(fa + a.seg, fhi + 1);
    // element offset of cell fa in this column; geometry index of face fa and its stride
    const double* y = a.P + (DIR == 1 ? (long long)t * d.s2 : (long long)t * d.s1) + k + (long long)fa * sd;
    long long idx = (DIR == 1 ? (long long)t * d.s2 : (long long)t * d.s1) + k + (long long)fa * sd;
    int gq = DIR == 1 ? fa * d.n2g + t : t * d.n2g + fa;
    const int gstep = DIR == 1 ? d.n2g : 1;
    double rprev[8], sc[8], elo[8];
    // prologue: limited upper-edge state of cell fa-1 (and, for PPM, slope of cell fa and edge value fa-1/2)
#pragma unroll
    for (int v = 0; v < 8; v++) {
      const double* yv = y + v * nz;
      if (RECON == 0) {
        const double ym2 = yv[-2 * sd], ym1 = yv[-sd], y0 = yv[0];
        rprev[v] = fma(0.5, slope_mc(ym2, ym1, y0), ym1);
      } else {
        const double ym3 = yv[-3 * sd], ym2 = yv[-2 * sd], ym1 = yv[-sd], y0 = yv[0], y1 = yv[sd];
        const double sm2 = slope_mc(ym3, ym2, ym1), sm1 = slope_mc(ym2, ym1, y0);
        sc[v] = slope_mc(ym1, y0, y1);
        double l = ppm_edge(ym2, ym1, sm2, sm1);
        double r = ppm_edge(ym1, y0, sm1, sc[v]);
        elo[v] = r;
        ppm_mono(ym1, l, r);
        rprev[v] = r;
      }
    }
    for (int f = fa; f < fb; f++) {
      double pl[8], pr[8];
#pragma unroll
      for (int v = 0; v < 8; v++) {
        const double* yv = y + v * nz;
        if (RECON == 0) {
          const double ym1 = yv[-sd], y0 = yv[0], y1 = yv[sd];
          const double hs = 0.5 * slope_mc(ym1, y0, y1);  // eq. 16
          pl[v] = rprev[v];
          pr[v] = y0 - hs;
          rprev[v] = y0 + hs;
        } else {
          const double y0 = yv[0], y1 = yv[sd], y2 = yv[2 * sd];
          const double s1 = slope_mc(y0, y1, y2);
          const double ehi = ppm_edge(y0, y1, sc[v], s1);
          double l = elo[v], r = ehi;
          ppm_mono(y0, l, r);
          pl[v] = rprev[v];
          pr[v] = l;
          rprev[v] = r;
          sc[v] = s1;
          elo[v] = ehi;
        }
      }
      const Geom G = load_geom(a.Gf, gq);
      double F[8], c;
      face_flux<DIR, RIEMANN>(pl, pr, G, a.gam, F, c);
      cwv = fmax(cwv, c);
      store_flux<DIR, STAGE>(a, idx, F, c);
      y += sd;
      idx += sd;
      gq += gstep;
    }
  }
  atomic_max_nonneg(a.cwmax, cwv);
}

// ---------------------------------------------------------------------------------------------------------
// Direction 3: one lane per cell along k, neighbours by shuffle.  Warp w of a row covers faces
// lo3 + w*FPW .. lo3 + w*FPW + FPW - 1; its lanes hold the cells from HALO below the first face.
// ---------------------------------------------------------------------------------------------------------
template <int RECON>
struct FluxK {
  static constexpr int HALO = RECON == 0 ? 1 : 2;   // lanes below the first valid face
  static constexpr int FPW = RECON == 0 ? 31 : 29;  // faces per warp
};

template <int RECON, int RIEMANN, bool STAGE>
__global__ void __launch_bounds__(128) flux_k_kernel(FluxArgs a) {
  const Dims& d = a.d;
  constexpr int HALO = FluxK<RECON>::HALO, FPW = FluxK<RECON>::FPW;
  const unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const int nfaces = a.hi3 - a.lo3 + 1;
  const int wpr = (nfaces + FPW - 1) / FPW;  // warps per row
  const int nj = a.hi2 - a.lo2 + 1;
  const long long nrows = (long long)(a.hi1 - a.lo1 + 1) * nj;
  const long long gw = (long long)blockIdx.x * 4 + (threadIdx.x >> 5);
  if (gw >= nrows * wpr) return;  // whole warp
  const int row = (int)(gw / wpr), w = (int)(gw % wpr);
  const int i = a.lo1 + row / nj, j = a.lo2 + row % nj;
  const int f0 = a.lo3 + w * FPW;
  const int c = f0 - HALO + lane;  // this lane's cell = the cell whose lower face is face c
  const int cc = min(max(c, 1), d.n3g - 2);  // clamped for loads; clamped lanes never produce output
  const long long nz = d.nz;
  const long long rowoff = i * d.s1 + j * d.s2;
  const double* y = a.P + rowoff + cc;
  double pl[8], pr[8];
#pragma unroll
  for (int v = 0; v < 8; v++) {
    const double* yv = y + v * nz;
    const double ym1 = yv[-1], y0 = yv[0], y1 = yv[1];
    const double s = slope_mc(ym1, y0, y1);
    double l, r;
    if (RECON == 0) {
      l = fma(-0.5, s, y0);
      r = fma(0.5, s, y0);
    } else {
      const double sup = __shfl_down_sync(FULL, s, 1);   // slope of cell c+1 (lane 31: garbage)
      const double ehi = ppm_edge(y0, y1, s, sup);
      const double elo = __shfl_up_sync(FULL, ehi, 1);   // edge value c-1/2 (lane 0: garbage)
      l = elo;
      r = ehi;
      ppm_mono(y0, l, r);
    }
    pl[v] = __shfl_up_sync(FULL, r, 1);  // upper-edge state of cell c-1
    pr[v] = l;
  }
  const bool valid = lane >= HALO && lane < HALO + FPW && c <= a.hi3;
  double cwv = 0.0;
  if (valid) {
    const Geom G = load_geom(a.Gf, i * d.n2g + j);
    double F[8];
    face_flux<3, RIEMANN>(pl, pr, G, a.gam, F, cwv);
    store_flux<3, STAGE>(a, rowoff + c, F, cwv);
  }
  atomic_max_nonneg(a.cwmax, cwv);
}

}  // namespace cuharm
