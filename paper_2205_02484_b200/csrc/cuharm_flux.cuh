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
//     shuffle; a warp of 32 cells yields 29 (PPM) or 31 (PLM) faces, consecutive warps overlap by the difference;
//     the 4 warps of a block take 4 consecutive rows j at the same position along k.
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
// A NaN enters as +infinity.  Must be reached by all 32 lanes of the warp.
__device__ __forceinline__ void atomic_max_nonneg(unsigned long long* addr, double v) {
  const double vv = v >= 0.0 ? v : (v != v ? __longlong_as_double(0x7ff0000000000000LL) : 0.0);
  const unsigned long long m = warp_max_ull((unsigned long long)__double_as_longlong(vv));
  if ((threadIdx.x & 31) == 0 && m > *reinterpret_cast<volatile unsigned long long*>(addr)) atomicMax(addr, m);
}

// ---------------------------------------------------------------------------------------------------------
// Asynchronous 1D bulk copies global -> shared (the TMA engine's cp.async.bulk) completing on an mbarrier.
// Source, destination and size must be multiples of 16 bytes.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  unsigned done = 0;
  while (!done) {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(done)
                 : "r"(bar), "r"(parity)
                 : "memory");
  }
}

// Running maximum of the face speeds c_w of a thread, kept as the integer image of |c_w| (order-preserving for
// non-negative doubles; the sign bit is cleared, so a NaN of either sign ranks above +infinity and is never lost the
// way fmax would lose it).  atomic_max_image folds the warp's maxima into the global slot, reporting anything above
// +infinity as +infinity.  Integer pipe only: nothing here competes with the fp64 pipe.
__device__ __forceinline__ void cw_track(unsigned long long& acc, double c) {
  const unsigned long long m = (unsigned long long)__double_as_longlong(c) & 0x7fffffffffffffffull;
  acc = m > acc ? m : acc;
}
__device__ __forceinline__ void atomic_max_image(unsigned long long* addr, unsigned long long acc) {
  unsigned long long m = warp_max_ull(acc);
  m = m > 0x7ff0000000000000ull ? 0x7ff0000000000000ull : m;
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
  int geo_rows;                      // marching kernels: transverse rows whose face geometry a block stages in
                                     // shared memory (0: read it from global memory face by face)
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
// Per variable a thread carries, for the face f it is about to do: yc = y_f, yn = y_{f+1}, dn = y_{f+1} - y_f,
// the doubled MC slope sc of cell f, the unlimited edge value elo at f-1/2, the limited upper-edge state rprev of
// cell f-1, and `pre` = y_{f+2}, loaded one iteration ahead so that its DRAM latency hides behind a whole face.
// ---------------------------------------------------------------------------------------------------------
// software prefetch distance (faces beyond the register look-ahead) per marching direction; measured on B200 at
// 256^3: along X1 (plane stride) 2 faces is best, along X2 (row stride) 1 face; into L1
constexpr int MARCH_PF1 = 2, MARCH_PF2 = 1;
__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

// 128 threads x 2 blocks per multiprocessor = the full register file at 255 registers per thread.  Measured on B200
// (256^3, PPM + LLF, ms per launch): 128 x 2 at 254 registers 0.59; capped at 232 registers 0.59; 64-thread blocks at
// 224 / 200 registers (no spills, 8 / 10 warps) 0.63 / 0.67; 168 registers (12 warps, 440 bytes spilled) 0.80 -- the
// kernel lives on instruction-level parallelism inside a warp, not on occupancy.
constexpr int MARCH_T = 128, MARCH_MINB = 2;
template <int DIR, int RECON, int RIEMANN, bool STAGE, bool GEO>
__global__ void __launch_bounds__(MARCH_T, MARCH_MINB) flux_march_kernel(FluxArgs a) {
  static_assert(DIR == 1 || DIR == 2, "marching kernel: directions 1 and 2");
  const Dims& d = a.d;
  const int nk = a.hi3 - a.lo3 + 1;
  const int nt = DIR == 1 ? (a.hi2 - a.lo2 + 1) : (a.hi1 - a.lo1 + 1);
  const int q = blockIdx.x * MARCH_T + threadIdx.x;
  unsigned long long cwv = 0ull;
  // The face geometry the block will need -- the records of (faces of its segment) x (the transverse rows its 128
  // columns touch) -- is staged in shared memory once, so the march reads it with shared-memory latency.
  extern __shared__ __align__(16) double2 geo[];  // [face in segment][row][10]
  const int t_first = (DIR == 1 ? a.lo2 : a.lo1) + (blockIdx.x * MARCH_T) / nk;
  if (GEO) {
    const int f0 = (DIR == 1 ? a.lo1 : a.lo2) + blockIdx.y * a.seg;
    const int f1 = min(f0 + a.seg, (DIR == 1 ? a.hi1 : a.hi2) + 1);
    const int t_max = DIR == 1 ? a.hi2 : a.hi1;
    const int nrec = (f1 - f0) * a.geo_rows;
    for (int e = threadIdx.x; e < nrec * 10; e += MARCH_T) {
      const int rec = e / 10, w = e - rec * 10;
      const int f = f0 + rec / a.geo_rows, tt = min(t_first + rec % a.geo_rows, t_max);
      const int g = DIR == 1 ? f * d.n2g + tt : tt * d.n2g + f;
      geo[e] = __ldg(reinterpret_cast<const double2*>(a.Gf + g) + w);
    }
    __syncthreads();
  }
  if (q < nt * nk) {
    const int t = (DIR == 1 ? a.lo2 : a.lo1) + q / nk;
    const int k = a.lo3 + q % nk;
    const long long sd = DIR == 1 ? d.s1 : d.s2;
    const long long nz = d.nz;
    const int flo = DIR == 1 ? a.lo1 : a.lo2, fhi = DIR == 1 ? a.hi1 : a.hi2;
    const int fa = flo + blockIdx.y * a.seg;
    const int fb = min(fa + a.seg, fhi + 1);
    const int nd = DIR == 1 ? d.n1g : d.n2g;  // extent of the marching direction (for the look-ahead clamp)
    // element offset of cell fa in this column; geometry index of face fa and its stride
    long long idx = (DIR == 1 ? (long long)t * d.s2 : (long long)t * d.s1) + k + (long long)fa * sd;
    const double* y = a.P + idx;
    int gq = DIR == 1 ? fa * d.n2g + t : t * d.n2g + fa;
    const int gstep = DIR == 1 ? d.n2g : 1;
    double yc[8], yn[8], dn[8], sc[8], elo[8], rprev[8], pre[8];
    // prologue: state of the carried quantities at face fa
#pragma unroll
    for (int v = 0; v < 8; v++) {
      const double* yv = y + v * nz;
      if (RECON == 0) {
        const double ym2 = yv[-2 * sd], ym1 = yv[-sd];
        yc[v] = yv[0];
        yn[v] = yv[sd];
        double l;
        plm_faces(ym1, slope2_mc(ym1 - ym2, yc[v] - ym1), l, rprev[v]);
        dn[v] = yc[v] - ym1;  // PLM carries the LOWER difference of cell f
        pre[v] = yv[(fa + 2 < nd ? 2 : 1) * sd];
      } else {
        const double ym3 = yv[-3 * sd], ym2 = yv[-2 * sd], ym1 = yv[-sd];
        yc[v] = yv[0];
        yn[v] = yv[sd];
        const double d32 = ym2 - ym3, d21 = ym1 - ym2, d10 = yc[v] - ym1;
        dn[v] = yn[v] - yc[v];
        const double sm2 = slope2_mc(d32, d21), sm1 = slope2_mc(d21, d10);
        sc[v] = slope2_mc(d10, dn[v]);
        double l = ppm_edge(ym2, ym1, sm2, sm1);
        double r = ppm_edge(ym1, yc[v], sm1, sc[v]);
        elo[v] = r;
        ppm_mono(ym1, l, r);
        rprev[v] = r;
        pre[v] = yv[2 * sd];
      }
    }
    // unrolled by 2 (measured at 256^3, ms per substep of the X1 kernel: x1 1.25, x2 1.19, x3 1.22, x4 1.20)
#pragma unroll 2
    for (int f = fa; f < fb; f++) {
      double pl[8], pr[8];
      // look-ahead load for the next face (clamped at the end of the array; the clamped value is never used)
      const long long ahead = (f + 3 < nd ? 3 : 2) * sd;
      {
        constexpr int PFD = DIR == 1 ? MARCH_PF1 : MARCH_PF2;
        const long long far = (f + 3 + PFD < nd ? 3 + PFD : 2) * sd;
#pragma unroll
        for (int v = 0; v < 8; v++) prefetch_l1(y + v * nz + far);
        if (!GEO) {
          prefetch_l1(reinterpret_cast<const char*>(a.Gf + gq + gstep));
          prefetch_l1(reinterpret_cast<const char*>(a.Gf + gq + gstep) + 128);
        }
      }
#pragma unroll
      for (int v = 0; v < 8; v++) {
        // (read-only path along X1 only -- measured at 256^3: X1 1.20 -> 1.17 ms per substep with it, X2 1.17 -> 1.30)
        const double nxt = DIR == 1 ? __ldg(y + v * nz + ahead) : y[v * nz + ahead];
        if (RECON == 0) {
          // cell f: slope from (y_f - y_{f-1}, y_{f+1} - y_f)
          const double dp = yn[v] - yc[v];
          double l, r;
          plm_faces(yc[v], slope2_mc(dn[v], dp), l, r);
          pl[v] = rprev[v];
          pr[v] = l;
          rprev[v] = r;
          dn[v] = dp;
          yc[v] = yn[v];
          yn[v] = pre[v];
        } else {
          const double y2 = pre[v];
          const double d2 = y2 - yn[v];
          const double s1 = slope2_mc(dn[v], d2);            // cell f+1
          const double ehi = ppm_edge_d(yc[v], dn[v], sc[v], s1);  // edge f+1/2
          double l = elo[v], r = ehi;
          ppm_mono(yc[v], l, r);
          pl[v] = rprev[v];
          pr[v] = l;
          rprev[v] = r;
          sc[v] = s1;
          elo[v] = ehi;
          dn[v] = d2;
          yc[v] = yn[v];
          yn[v] = y2;
        }
        pre[v] = nxt;
      }
      const Geom G = GEO ? load_geom_shared(reinterpret_cast<const double*>(geo + ((f - fa) * a.geo_rows + (t - t_first)) * 10))
                         : load_geom(a.Gf, gq);
      double F[8], c;
      face_flux<DIR, RIEMANN>(pl, pr, G, a.gam, F, c);
      cw_track(cwv, c);
      store_flux<DIR, STAGE>(a, idx, F, c);
      y += sd;
      idx += sd;
      gq += gstep;
    }
  }
  atomic_max_image(a.cwmax, cwv);
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
__global__ void __launch_bounds__(128, 4) flux_k_kernel(FluxArgs a) {
  const Dims& d = a.d;
  constexpr int HALO = FluxK<RECON>::HALO, FPW = FluxK<RECON>::FPW;
  const unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  // grid: x = warp slot along the row, y = groups of 4 rows j (one per warp of the block), z = i: no divisions
  const int w = blockIdx.x;
  const int j = a.lo2 + blockIdx.y * 4 + (threadIdx.x >> 5);
  const int i = a.lo1 + blockIdx.z;
  if (j > a.hi2) return;  // whole warp
  const int f0 = a.lo3 + w * FPW;
  const int c = f0 - HALO + lane;  // this lane's cell = the cell whose lower face is face c
  const int cc = min(max(c, 1), d.n3g - 2);  // clamped for the loads; clamped lanes never produce output
  const long long nz = d.nz;
  const long long rowoff = i * d.s1 + j * d.s2;
  const double* y = a.P + rowoff + cc;
  double pl[8], pr[8];
#pragma unroll
  for (int v = 0; v < 8; v++) {
    const double* yv = y + v * nz;
    const double ym1 = yv[-1], y0 = yv[0], y1 = yv[1];
    const double dp = y1 - y0;
    const double s = slope2_mc(y0 - ym1, dp);
    double l, r;
    if (RECON == 0) {
      plm_faces(y0, s, l, r);
    } else {
      const double sup = __shfl_down_sync(FULL, s, 1);   // slope of cell c+1 (lane 31: garbage)
      const double ehi = ppm_edge_d(y0, dp, s, sup);
      const double elo = __shfl_up_sync(FULL, ehi, 1);   // edge value c-1/2 (lane 0: garbage)
      l = elo;
      r = ehi;
      ppm_mono(y0, l, r);
    }
    pl[v] = __shfl_up_sync(FULL, r, 1);  // upper-edge state of cell c-1
    pr[v] = l;
  }
  const bool ok = lane >= HALO && lane < HALO + FPW && c <= a.hi3;
  unsigned long long cwi = 0ull;
  if (ok) {
    const Geom G = load_geom(a.Gf, i * d.n2g + j);
    double F[8], cwv;
    face_flux<3, RIEMANN>(pl, pr, G, a.gam, F, cwv);
    store_flux<3, STAGE>(a, rowoff + c, F, cwv);
    cw_track(cwi, cwv);
  }
  atomic_max_image(a.cwmax, cwi);
}

// ---------------------------------------------------------------------------------------------------------
// Direction 3, whole-row version (n3g even, 16-byte aligned P): persistent blocks of NW warps.  A work item is one
// (i, j) row: its 8 variables arrive as 8 bulk copies of the whole row (n3g doubles each) into one of two stages,
// and warp w of the block takes the chunks w, w + NW, ... of the row (29 / 31 faces each, as above).  Compared with
// per-thread loads nothing waits on DRAM with a scoreboard (the copies of the next two rows fly during the
// arithmetic of this one), and whole rows keep the copy count low: a warp issues its bulk copies one after the
// other at ~8 issue slots each.
// ---------------------------------------------------------------------------------------------------------
constexpr int KROW_STAGES = 3;  // rows in the ring of a block
template <int RECON, int RIEMANN, bool STAGE>
__global__ void __launch_bounds__(128, 4) flux_k_row_kernel(FluxArgs a, int wpr) {
  constexpr int NS = KROW_STAGES;
  extern __shared__ __align__(128) double rowbuf[];  // [NS][8][n3g]
  __shared__ __align__(8) unsigned long long mbar2[2 * NS];  // full[NS] (tx count), empty[NS] (one arrival per warp)
  const Dims& d = a.d;
  constexpr int HALO = FluxK<RECON>::HALO, FPW = FluxK<RECON>::FPW;
  const unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int rs = d.n3g;
  const unsigned bar0 = smem_u32(&mbar2[0]);
  const int ni = a.hi1 - a.lo1 + 1, nj = a.hi2 - a.lo2 + 1;
  const int nrows = ni * nj, G = gridDim.x;
  int row = blockIdx.x;
  int ci = row / nj, cj = row % nj;          // carried (i, j) of the current row
  const int di = G / nj, dj = G % nj;
  auto issue = [&](int r, int stage) {  // lanes 0..7 of warp 0, one variable each; r = row index
    const int i = r / nj, j = r - i * nj;
    const double* src = a.P + (long long)(a.lo1 + i) * d.s1 + (long long)(a.lo2 + j) * d.s2 + lane * d.nz;
    const unsigned bar = bar0 + 8 * stage;
    if (lane == 0) mbar_expect_tx(bar, 8u * rs * 8u);
    __syncwarp(0xffu);
    bulk_g2s(smem_u32(rowbuf + (stage * 8 + lane) * rs), src, (unsigned)rs * 8u, bar);
  };
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < NS; s++) { mbar_init(bar0 + 8 * s, 1); mbar_init(bar0 + 8 * (NS + s), nw); }
    mbar_fence_init();
  }
  __syncthreads();
  if (wib == 0 && lane < 8) {
    for (int s = 0; s < NS; s++)
      if (row + (long long)s * G < nrows) issue(row + s * G, s);
  }
  unsigned long long cwmax = 0ull;
  for (int n = 0; row < nrows; row += G, n++) {
    const int s = n % NS;
    const int i = a.lo1 + ci, j = a.lo2 + cj;
    const double* st = rowbuf + s * 8 * rs;
    mbar_wait(bar0 + 8 * s, (n / NS) & 1);
    for (int w = wib; w < wpr; w += nw) {
      const int f0 = a.lo3 + w * FPW;
      const int c = f0 - HALO + lane;            // this lane's cell = the cell whose lower face is face c
      const int cc = min(max(c, 1), d.n3g - 2);  // clamped for the reads; clamped lanes never produce output
      double pl[8], pr[8];
#pragma unroll
      for (int v = 0; v < 8; v++) {
        const double ym1 = st[v * rs + cc - 1], y0 = st[v * rs + cc], y1 = st[v * rs + cc + 1];
        const double dp = y1 - y0;
        const double sl = slope2_mc(y0 - ym1, dp);
        double l, r;
        if (RECON == 0) {
          plm_faces(y0, sl, l, r);
        } else {
          const double sup = __shfl_down_sync(FULL, sl, 1);   // slope of cell c+1 (lane 31: garbage)
          const double ehi = ppm_edge_d(y0, dp, sl, sup);
          const double elo = __shfl_up_sync(FULL, ehi, 1);    // edge value c-1/2 (lane 0: garbage)
          l = elo;
          r = ehi;
          ppm_mono(y0, l, r);
        }
        pl[v] = __shfl_up_sync(FULL, r, 1);  // upper-edge state of cell c-1
        pr[v] = l;
      }
      const bool ok = lane >= HALO && lane < HALO + FPW && c <= a.hi3;
      if (ok) {
        const Geom G3 = load_geom(a.Gf, i * d.n2g + j);
        double F[8], cwv;
        face_flux<3, RIEMANN>(pl, pr, G3, a.gam, F, cwv);
        store_flux<3, STAGE>(a, i * d.s1 + j * d.s2 + c, F, cwv);
        cw_track(cwmax, cwv);
      }
    }
    // This warp is done with stage s (one arrival per warp; no block-wide barrier: the warps of a block may be a row
    // apart).  The stage released ONE ROW AGO, which every warp has normally long left, is then refilled by warp 0 with
    // the row NS - 1 iterations ahead: NS - 1 rows are in flight or landed while a row is being worked on.
    __syncwarp();
    if (lane == 0) mbar_arrive(bar0 + 8 * (NS + s));
    // (the wait is executed by every thread -- a spin loop under a thread-dependent condition would cost the warp its
    // convergence guarantee and every shuffle above an explicit re-synchronisation)
    const long long rnext = (long long)row + (long long)(NS - 1) * G;  // row of iteration n - 1 + NS
    if (n >= 1 && rnext < nrows) {
      mbar_wait(bar0 + 8 * (NS + (n - 1) % NS), ((n - 1) / NS) & 1);
      if (wib == 0 && lane < 8) issue((int)rnext, (n - 1) % NS);
    }
    ci += di;
    cj += dj;
    if (cj >= nj) { cj -= nj; ci++; }
  }
  atomic_max_image(a.cwmax, cwmax);
}

}  // namespace cuharm
