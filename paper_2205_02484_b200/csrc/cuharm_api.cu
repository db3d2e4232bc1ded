// cuharm_api.cu — host side of libcuharm.so: the C ABI of include/cuharm.h, workspace carving, launch
// sequencing of one RK2 step (eq. 25), optional CUDA-graph replay.  No torch types, no device
// allocation: the caller owns every device byte.  There is no CPU path: without a device every call fails.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/cuharm.h"
#include "cuharm_geom.cuh"
#include "cuharm_kernels.cuh"
#include "cuharm_update_tmap.cuh"

using namespace cuharm;

namespace {

thread_local char g_errtext[256] = "no CUDA error recorded";

int cuda_fail(cudaError_t e, const char* what) {
  snprintf(g_errtext, sizeof(g_errtext), "%s: %s", what, cudaGetErrorString(e));
  (void)cudaGetLastError();  // clear the non-sticky error state so that later calls report their own
  return CUHARM_ECUDA;
}
#define CK(call)                                          \
  do {                                                    \
    cudaError_t e_ = (call);                              \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call);   \
  } while (0)

size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

// counters block (unsigned long long slots)
// [CNT_NFAIL, CNT_STEP_END) is zeroed at the start of every step: failure counts of the two substeps, the c_w maxima of
// predictor and corrector, and per substep CNT_FIXW slots of repair / fallback-chain scratch ([0] grid-barrier counter of
// the repair, [1..] zones left waiting after each repair pass, [CNT_FIXW - 1] zones still failed after the chain).
// CNT_CLOCK: two doubles, the step size of the current step and the integrated time (set_dt_kernel, dt_from_cw_kernel).
// CNT_CHAIN: the four counters of cuharm_get_chain_stats.
enum { CNT_STATS = 0, CNT_NFAIL = 8, CNT_CWPRED = 10, CNT_CWSCR = 13, CNT_FIX = 16, CNT_FIXW = 24, CNT_STEP_END = 64,
       CNT_DIVB = 64, CNT_CLOCK = 66, CNT_CHAIN = 68, CNT_TOTAL = 80 };
constexpr int FIXUP_MAX_PASSES_CAP = CNT_FIXW - 3;

}  // namespace

struct cuharm_ctx {
  cuharm_params p;
  Dims d;
  cudaStream_t stream;
  int dev = 0;  // CUDA device the context was created on; every entry point runs with it current
  double dx[3], x0[3];
  // borrowed device memory
  double* prim = nullptr;
  char* ws = nullptr;
  Geom *gC = nullptr, *gF1 = nullptr, *gF2 = nullptr;
  double *conn = nullptr, *srcw = nullptr, *rec = nullptr, *floors = nullptr, *F[3] = {nullptr, nullptr, nullptr}, *E = nullptr, *Phalf = nullptr, *ustar = nullptr;
  int *flag = nullptr, *list = nullptr;
  unsigned long long* cnt = nullptr;
  bool bound = false, have_geom = false, stepped = false;
  bool dt_set = false, half_done = false;  // cuharm_set_dt / cuharm_substep sequencing
  int64_t launches = 0;
  // optional per-kernel-class timing with CUDA events on the library's stream (cuharm_set_timing)
  bool timing = false, capturing = false;
  std::vector<cudaEvent_t> ev;
  std::vector<int> ev_cat;
  size_t ev_used = 0;
  double t_ms[CUHARM_NCLASS] = {0};
  int64_t t_n[CUHARM_NCLASS] = {0};
  // graph
  bool upd_tma = false;  // update_tma_kernel usable (shared-memory opt-in succeeded)
  bool upd_tmap = false; // update_tmap_kernel usable (opt-in succeeded, tensor maps of the bound arrays encoded)
  bool tmap_enable = true;
  int tmap_blocks = 0, tmap_blocks64 = 0;
  bool maps_ok = false;
  UpdMaps maps;
  int upd_blocks = 0, upd_blocks64 = 0;  // its persistent grid sizes (128- and 64-zone tiles)
  int sms = 148;         // multiprocessors of the device
  bool coop = false;     // cooperative launches available (device attribute; decided at grid_init)
  double xb = 0.0;       // eq. 39: X1 of the exponential -> hyper-exponential transition
  int nx = 0;            // its exponent (0: plain exponential)
  bool fluxk_row = true; // prefer the whole-row pipeline (flux_k_row_kernel)
  bool use_graph = false;
  cudaGraphExec_t gexec = nullptr;
  cudaStream_t cap_stream = nullptr;
  cudaStream_t side[2] = {nullptr, nullptr};  // branches of the recorded graph (flux kernels of directions 2, 3)
  cudaEvent_t fj[3] = {nullptr, nullptr, nullptr};  // fork / join events of those branches
  int64_t graph_nodes = 0;
};

// update_tma_kernel: tiles are ordered in strips of this many rows j (shared rows are then re-read from L2)
constexpr int UPD_STRIP = 8;

// Makes the context's device current for the duration of an entry point and restores the caller's.
struct DevGuard {
  int prev = -1;
  bool changed = false;
  explicit DevGuard(const cuharm_ctx* h) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != h->dev) changed = cudaSetDevice(h->dev) == cudaSuccess;
  }
  ~DevGuard() {
    if (changed) cudaSetDevice(prev);
  }
};

namespace {

struct WsLayout {
  size_t gC, gF1, gF2, conn, srcw, rec, floors, F[3], E, Phalf, flag, list, cnt, ustar, total;
};

WsLayout layout(const Dims& d, bool chain) {
  WsLayout L;
  size_t off = 0;
  const size_t ncol = (size_t)d.n1g * d.n2g, nz = (size_t)d.nz;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
  L.gC = take(ncol * sizeof(Geom));
  L.gF1 = take(ncol * sizeof(Geom));
  L.gF2 = take(ncol * sizeof(Geom));
  L.conn = take(ncol * 40 * sizeof(double));
  L.srcw = take(ncol * 14 * sizeof(double));
  L.rec = take(ncol * 36 * sizeof(double));
  L.floors = take(ncol * 2 * sizeof(double));
  for (int k = 0; k < 3; k++) L.F[k] = take(7 * nz * sizeof(double));
  L.E = take(3 * nz * sizeof(double));
  L.Phalf = take(8 * nz * sizeof(double));
  L.flag = take(nz * sizeof(int));
  L.list = take(nz * sizeof(int));
  L.cnt = take(CNT_TOTAL * sizeof(unsigned long long));
  L.ustar = take(chain ? 8 * nz * sizeof(double) : 0);  // U* of every zone, only with the fallback chain on
  L.total = off;
  return L;
}

// Tensor maps of the bound arrays for update_tmap_kernel (box list in cuharm_update_tmap.cuh): 4-D [component][i][j][k],
// 8-byte elements, zero fill outside the array.  The driver's encoder is reached through the runtime
// (cudaGetDriverEntryPoint), so the library keeps linking against the CUDA runtime only.
bool encode_update_maps(cuharm_ctx* h) {
  typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static EncodeFn encode = nullptr;
  if (!encode) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) {
      (void)cudaGetLastError();
      return false;
    }
    encode = (EncodeFn)fn;
  }
  const Dims& d = h->d;
  if (d.n3g % 2) return false;  // strides must be multiples of 16 bytes
  const int tb = d.n3 <= 64 ? 64 : 128;
  struct Box { double* base; int ncomp; unsigned bj, bi, bc; };
  const Box boxes[TMAP_NBOX] = {
      {h->prim, 8, 1, 1, 8}, {h->Phalf, 8, 1, 1, 8},
      {h->F[0], 7, 1, 2, 5}, {h->F[1], 7, 2, 1, 5}, {h->F[2], 7, 1, 1, 5},
      {h->F[1], 7, 2, 1, 1}, {h->F[2], 7, 3, 1, 1}, {h->F[2], 7, 1, 3, 1}, {h->F[0], 7, 1, 2, 1},
      {h->F[0], 7, 3, 2, 1}, {h->F[1], 7, 2, 3, 1}};
  for (int b = 0; b < TMAP_NBOX; b++) {
    if ((uintptr_t)boxes[b].base % 16) return false;
    const cuuint64_t dims[4] = {(cuuint64_t)d.n3g, (cuuint64_t)d.n2g, (cuuint64_t)d.n1g, (cuuint64_t)boxes[b].ncomp};
    const cuuint64_t strides[3] = {(cuuint64_t)d.s2 * 8, (cuuint64_t)d.s1 * 8, (cuuint64_t)d.nz * 8};
    const cuuint32_t box[4] = {(cuuint32_t)(tb + 2), boxes[b].bj, boxes[b].bi, boxes[b].bc};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    if (tmap_rows(b) != (int)(boxes[b].bj * boxes[b].bi * boxes[b].bc)) return false;
    const CUresult r = encode(&h->maps.m[b], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, boxes[b].base, dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return false;
  }
  return true;
}

NewtonCfg newton_cfg(const cuharm_params& p) { return NewtonCfg{p.newton_tol, p.newton_maxit, p.newton_extra}; }
ChainCfg chain_cfg(const cuharm_params& p) { return ChainCfg{p.inv_chain, p.brent_maxit, p.beta_min, p.brent_tol}; }
FloorCfg floor_cfg(const cuharm_params& p) {
  return FloorCfg{p.sigma_max, p.b2_over_u_max, p.gamma_max, p.sigma_max > 0.0 ? 1.0 / p.sigma_max : 0.0,
                  p.b2_over_u_max > 0.0 ? 1.0 / p.b2_over_u_max : 0.0};
}

// RAII pair of events around one launch (or one group of launches) of a kernel class
struct Timed {
  cuharm_ctx* h;
  bool live;
  Timed(cuharm_ctx* h_, int cat) : h(h_), live(false) {
    if (!h->timing || h->capturing || h->ev_used + 2 > h->ev.size()) return;
    if (cudaEventRecord(h->ev[h->ev_used], h->stream) != cudaSuccess) return;
    h->ev_cat.push_back(cat);
    live = true;
  }
  ~Timed() {
    if (!live) return;
    cudaEventRecord(h->ev[h->ev_used + 1], h->stream);
    h->ev_used += 2;
  }
};

// The repair kernel separates its Jacobi passes by a grid barrier, so its participating blocks must be resident together.
// A COOPERATIVE launch makes the driver guarantee that (and keeps two such kernels from different streams from holding
// multiprocessors against each other); it is also what a recorded graph stores.  Devices / drivers without cooperative
// launch get a plain launch of one block (no barrier needed).
int launch_fixup(cuharm_ctx* h, const FixArgs& a) {
  if (h->coop) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)h->sms);
    cfg.blockDim = dim3(FIX_THREADS);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = h->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, fixup_kernel, a);
    if (e == cudaSuccess) { h->launches++; return CUHARM_OK; }
    if (h->capturing) return cuda_fail(e, "cudaLaunchKernelEx(fixup_kernel, cooperative)");
    (void)cudaGetLastError();
    h->coop = false;  // not supported here after all: plain launches from now on
  }
  // without the cooperative attribute nothing makes several blocks co-resident, and blocks spinning at the kernel's
  // grid barrier could wait for one that never starts (other streams may hold the multiprocessors): ONE block, which
  // takes the barrier-free path of the kernel -- slow for many failed zones, never a deadlock
  fixup_kernel<<<1, FIX_THREADS, 0, h->stream>>>(a);
  h->launches++;
  CK(cudaGetLastError());
  return CUHARM_OK;
}

int launch_bc(cuharm_ctx* h, double* P, const unsigned long long* gate) {
  Timed t_(h, CUHARM_K_BC);
  const Dims& d = h->d;
  // one launch for the whole ghost fill (the composition of the X1 -> X2 -> X3 fills, cuharm_kernels.cuh)
  if (h->p.bc_x1 == 3 && h->p.bc_x2 == 3 && h->p.bc_x3 == 3) return CUHARM_OK;
  const int nrows_a = d.n1g * d.n2g - d.n1 * d.n2;
  const int kchunks = (d.n3g + 127) / 128;
  const int per = 128 / (2 * d.ng);
  const long long nb = (long long)nrows_a * kchunks + ((long long)d.n1 * d.n2 + per - 1) / per;
  const bool slab = h->p.n1_global > 0;
  BcAllArgs b{d, P, h->gC, h->p.bc_x1, h->p.bc_x2, h->p.bc_x3, h->p.coords, (slab && h->p.slab_lo) ? 3 : h->p.bc_x1,
              (slab && h->p.slab_hi) ? 3 : h->p.bc_x1, h->p.gamma_max, gate, nrows_a};
  bc_all_kernel<<<(unsigned)nb, 128, 0, h->stream>>>(b);
  h->launches++;
  CK(cudaGetLastError());
  return CUHARM_OK;
}

// Faces per marching segment.  A block costs (faces + ~0.6) face-times (the prologue of a segment reconstructs one
// extra cell) and the 2 x SMs resident blocks run in waves, so the segment count is chosen to minimise
// waves x (faces per segment + 0.6) among the counts that keep segments at least 16 faces long.
int march_seg(long long columns, int nfaces, int sms) {
  const long long col_blocks = (columns + MARCH_T - 1) / MARCH_T;
  const long long slots = (long long)MARCH_MINB * (sms > 0 ? sms : 148);
  const int maxseg = nfaces >= 32 ? nfaces / 16 : 1;
  int best = 1;
  double best_cost = 1e300;
  for (int nseg = 1; nseg <= maxseg; nseg++) {
    const int seg = (nfaces + nseg - 1) / nseg;
    const long long blocks = col_blocks * ((nfaces + seg - 1) / seg);
    const double waves = (double)((blocks + slots - 1) / slots);
    const double cost = waves * (seg + 0.6);
    if (cost < best_cost * 0.999) { best_cost = cost; best = nseg; }
  }
  return (nfaces + best - 1) / best;  // faces per segment
}

template <int RECON, int RIEMANN, bool STAGE>
void launch_flux_t(cuharm_ctx* h, FluxArgs& a, int dir) {
  const int ni = a.hi1 - a.lo1 + 1, nj = a.hi2 - a.lo2 + 1, nk = a.hi3 - a.lo3 + 1;
  if (dir == 3) {
    const int fpw = FluxK<RECON>::FPW;
    const int wpr = (nk + fpw - 1) / fpw;
    const Dims& d = a.d;
    const bool tma = h->fluxk_row && (d.n3g % 2 == 0) && ((uintptr_t)a.P % 16 == 0);
    const size_t row_smem = KROW_STAGES * 8 * (size_t)d.n3g * sizeof(double);
    bool row_ok = tma && row_smem <= 200 * 1024;
    if (row_ok && row_smem > 48 * 1024)
      row_ok = cudaFuncSetAttribute(flux_k_row_kernel<RECON, RIEMANN, STAGE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)row_smem) == cudaSuccess;
    if (row_ok) {
      // whole-row pipeline: warps per block chosen to divide the chunks of a row evenly
      const int nw = wpr % 3 == 0 ? 3 : (wpr % 4 == 0 ? 4 : (wpr % 2 == 0 ? 2 : (wpr >= 4 ? 4 : wpr)));
      int per = 0;
      if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, flux_k_row_kernel<RECON, RIEMANN, STAGE>, 32 * nw, row_smem) != cudaSuccess || per < 1) per = 1;
      const int nb = (int)std::min<long long>((long long)ni * nj, (long long)h->sms * per);
      flux_k_row_kernel<RECON, RIEMANN, STAGE><<<nb, 32 * nw, row_smem, h->stream>>>(a, wpr);
    } else {
      const dim3 grid((unsigned)wpr, (unsigned)((nj + 3) / 4), (unsigned)ni);
      flux_k_kernel<RECON, RIEMANN, STAGE><<<grid, 128, 0, h->stream>>>(a);
    }
  } else {
    const int nf = dir == 1 ? ni : nj;
    const int nt = dir == 1 ? nj : ni;
    const long long cols = (long long)nt * nk;
    a.seg = march_seg(cols, nf, h->sms);
    const dim3 grid((unsigned)((cols + MARCH_T - 1) / MARCH_T), (unsigned)((nf + a.seg - 1) / a.seg));
    // face geometry staged per block: (rows a block's 128 columns can touch) x (faces per segment) records
    a.geo_rows = std::min(nt, (MARCH_T - 1) / nk + 2);
    size_t gsm = (size_t)a.geo_rows * a.seg * sizeof(Geom);
    if (gsm > 40 * 1024) { a.geo_rows = 0; gsm = 0; }
    if (a.geo_rows > 0) {
      if (dir == 1) flux_march_kernel<1, RECON, RIEMANN, STAGE, true><<<grid, MARCH_T, gsm, h->stream>>>(a);
      else flux_march_kernel<2, RECON, RIEMANN, STAGE, true><<<grid, MARCH_T, gsm, h->stream>>>(a);
    } else {
      if (dir == 1) flux_march_kernel<1, RECON, RIEMANN, STAGE, false><<<grid, MARCH_T, 0, h->stream>>>(a);
      else flux_march_kernel<2, RECON, RIEMANN, STAGE, false><<<grid, MARCH_T, 0, h->stream>>>(a);
    }
  }
}

// fluxes of direction dir (1..3) of the primitive array P into F (and c_w max into cwmax)
template <bool STAGE>
int launch_flux(cuharm_ctx* h, const double* P, int dir, double* F, double* cw, unsigned long long* cwmax) {
  const Dims& d = h->d;
  int lo[3], hi[3];
  const int n[3] = {d.n1, d.n2, d.n3};
  for (int c = 0; c < 3; c++) {
    lo[c] = (c == dir - 1) ? d.ng : d.ng - 1;
    hi[c] = d.ng + n[c];
  }
  Timed t_(h, CUHARM_K_FLUX1 + dir - 1);
  FluxArgs a{d, P, dir == 1 ? h->gF1 : (dir == 2 ? h->gF2 : h->gC), F, cw, cwmax, h->p.gam,
             lo[0], lo[1], lo[2], hi[0], hi[1], hi[2], 0, 0};
  const int rc = h->p.recon, rm = h->p.riemann;
  if (rc == 0 && rm == 0) launch_flux_t<0, 0, STAGE>(h, a, dir);
  else if (rc == 0 && rm == 1) launch_flux_t<0, 1, STAGE>(h, a, dir);
  else if (rc == 1 && rm == 0) launch_flux_t<1, 0, STAGE>(h, a, dir);
  else launch_flux_t<1, 1, STAGE>(h, a, dir);
  h->launches++;
  CK(cudaGetLastError());
  return CUHARM_OK;
}

// one RK2 substep (A34 order): fluxes -> EMFs -> update+inversion+floors -> ghost fill -> repair -> ghost fill
// `with_repair` = false: stop after the first ghost fill (the caller drives the repair pass by pass: cuharm_repair_pass)
int substep(cuharm_ctx* h, const double* Pflux, const double* Pbase, double* Pout, double dtfac, int which, bool with_repair = true) {
  const Dims& d = h->d;
  unsigned long long* cwmax = h->cnt + (which == 0 ? CNT_CWPRED : CNT_CWSCR);
  // The three flux kernels are independent of one another.  While a graph is being recorded they go on three
  // branches (fork / join through events), so that the drain of one overlaps the ramp-up of the next; launched
  // directly they stay in stream order (that is also the mode in which per-kernel events time them).
  bool fork = false;
  if (h->capturing) {
    fork = true;
    for (int s = 0; s < 2 && fork; s++)
      if (!h->side[s] && cudaStreamCreateWithFlags(&h->side[s], cudaStreamNonBlocking) != cudaSuccess) fork = false;
    for (int e = 0; e < 3 && fork; e++)
      if (!h->fj[e] && cudaEventCreateWithFlags(&h->fj[e], cudaEventDisableTiming) != cudaSuccess) fork = false;
    if (!fork) cudaGetLastError();
  }
  if (fork) {
    cudaStream_t main_s = h->stream;
    CK(cudaEventRecord(h->fj[0], main_s));
    // launch order of the three directions (main branch first); measured best on B200: the persistent X3 kernel
    // first, the many-block marching kernels fill in behind it
    static const int od[3] = {3, 1, 2};
    int rc = launch_flux<false>(h, Pflux, od[0], h->F[od[0] - 1], nullptr, cwmax + od[0] - 1);
    for (int s = 0; s < 2 && !rc; s++) {
      CK(cudaStreamWaitEvent(h->side[s], h->fj[0], 0));
      h->stream = h->side[s];
      rc = launch_flux<false>(h, Pflux, od[1 + s], h->F[od[1 + s] - 1], nullptr, cwmax + od[1 + s] - 1);
      h->stream = main_s;
      CK(cudaEventRecord(h->fj[1 + s], h->side[s]));
      CK(cudaStreamWaitEvent(main_s, h->fj[1 + s], 0));
    }
    if (rc) return rc;
  } else {
    for (int dir = 1; dir <= 3; dir++) {
      int rc = launch_flux<false>(h, Pflux, dir, h->F[dir - 1], nullptr, cwmax + (dir - 1));
      if (rc) return rc;
    }
  }
  // bulk-copy (TMA) staging of the update kernel needs 16-byte aligned row segments: even n3g, aligned arrays.
  // That kernel evaluates the edge EMFs itself (flux-CT fused); otherwise they go through emf_kernel and h->E.
  const uintptr_t al = (uintptr_t)Pbase | (uintptr_t)Pflux | (uintptr_t)h->F[0] | (uintptr_t)h->F[1] |
                       (uintptr_t)h->F[2] | (uintptr_t)h->E;
  // (the staged row starts one zone below the tile, at ng - 1 + c TB: 16-byte aligned only for odd ng)
  // tensor-map staging: the same restriction (a box that starts 8 bytes off a 16-byte boundary faults on B200, measured);
  // it serves the library's own arrays (the maps hold their addresses)
  const bool tmap = h->maps_ok && (d.n3g % 2 == 0) && (d.ng % 2 == 1) && Pbase == h->prim &&
                    (Pflux == h->prim || Pflux == h->Phalf);
  const bool tma = !tmap && h->upd_tma && (d.n3g % 2 == 0) && (d.ng % 2 == 1) && (al % 16 == 0);
  if (!tma && !tmap) {
    Timed t_(h, CUHARM_K_EMF);
    EmfArgs a{d, h->F[0], h->F[1], h->F[2], h->E};
    emf_kernel<<<dim3((d.n3 + 1 + 127) / 128, d.n2 + 1, d.n1 + 1), 128, 0, h->stream>>>(a);
    h->launches++;
  }
  unsigned long long* nfail = h->cnt + CNT_NFAIL + which;
  {
    Timed t_(h, CUHARM_K_UPDATE);
    UpdArgs a{d, Pbase, Pflux, Pout, h->F[0], h->F[1], h->F[2], h->E, h->gC, h->srcw, h->floors, h->flag, h->list,
              nfail, h->cnt + CNT_STATS, reinterpret_cast<const double*>(h->cnt + CNT_CLOCK), dtfac, 1.0 / h->dx[0], 1.0 / h->dx[1], 1.0 / h->dx[2], h->p.gam,
              newton_cfg(h->p), floor_cfg(h->p), chain_cfg(h->p), h->ustar};
    dim3 grid((d.n3 + 127) / 128, d.n2, d.n1);
    if (tmap) {
      const int tb = d.n3 <= 64 ? 64 : 128;
      const size_t smem = tmap_smem(tb);
      const int nch = (d.n3 + tb - 1) / tb;
      const long long nt = (long long)d.n1 * d.n2 * nch;
      const int ntiles = (int)nt;
      const int nb = (int)std::min<long long>(nt, tb == 64 ? h->tmap_blocks64 : h->tmap_blocks);
      int wj = 1;  // strip width: the largest divisor of n2 not above UPD_STRIP
      for (int w = 1; w <= UPD_STRIP && w <= d.n2; w++)
        if (d.n2 % w == 0) wj = w;
      const bool same = Pflux == Pbase;
      auto go = [&](auto kern, int threads) { kern<<<nb, threads, smem, h->stream>>>(a, h->maps, h->rec, ntiles, nch, wj); };
      if (h->p.inv_chain) {
        if (tb == 64) same ? go(update_tmap_kernel<true, 64, true>, 64) : go(update_tmap_kernel<false, 64, true>, 64);
        else same ? go(update_tmap_kernel<true, 128, true>, 128) : go(update_tmap_kernel<false, 128, true>, 128);
      } else {
        if (tb == 64) same ? go(update_tmap_kernel<true, 64, false>, 64) : go(update_tmap_kernel<false, 64, false>, 64);
        else same ? go(update_tmap_kernel<true, 128, false>, 128) : go(update_tmap_kernel<false, 128, false>, 128);
      }
    } else if (tma) {
      const int tb = d.n3 <= 64 ? 64 : 128;
      const size_t smem = upd_smem(tb);
      const int nch = (d.n3 + tb - 1) / tb;
      const long long nt = (long long)d.n1 * d.n2 * nch;
      const int ntiles = (int)nt;
      const int nb = (int)std::min<long long>(nt, tb == 64 ? h->upd_blocks64 : h->upd_blocks);
      int wj = 1;  // strip width: the largest divisor of n2 not above UPD_STRIP
      for (int w = 1; w <= UPD_STRIP && w <= d.n2; w++)
        if (d.n2 % w == 0) wj = w;
      const bool same = Pflux == Pbase;
      auto go = [&](auto kern, int threads) { kern<<<nb, threads, smem, h->stream>>>(a, ntiles, nch, wj); };
      if (h->p.inv_chain) {
        if (tb == 64) same ? go(update_tma_kernel<true, 64, true>, 64) : go(update_tma_kernel<false, 64, true>, 64);
        else same ? go(update_tma_kernel<true, 128, true>, 128) : go(update_tma_kernel<false, 128, true>, 128);
      } else {
        if (tb == 64) same ? go(update_tma_kernel<true, 64, false>, 64) : go(update_tma_kernel<false, 64, false>, 64);
        else same ? go(update_tma_kernel<true, 128, false>, 128) : go(update_tma_kernel<false, 128, false>, 128);
      }
    } else {
      const bool same = Pflux == Pbase;
      if (h->p.inv_chain) {
        if (same) update_kernel<true, true><<<grid, 128, 0, h->stream>>>(a);
        else update_kernel<false, true><<<grid, 128, 0, h->stream>>>(a);
      } else {
        if (same) update_kernel<true, false><<<grid, 128, 0, h->stream>>>(a);
        else update_kernel<false, false><<<grid, 128, 0, h->stream>>>(a);
      }
    }
    h->launches++;
  }
  CK(cudaGetLastError());
  if (h->p.inv_chain) {  // 1D-W and entropy methods on the listed zones, before anything reads Pout
    Timed t_(h, CUHARM_K_FIXUP);
    ChainArgs a{d, Pflux, Pout, h->gC, h->gF1, h->gF2, h->floors, h->flag, h->list, h->ustar, nfail,
                h->cnt + CNT_FIX + which * CNT_FIXW + CNT_FIXW - 1, h->cnt + CNT_STATS, h->cnt + CNT_CHAIN,
                reinterpret_cast<const double*>(h->cnt + CNT_CLOCK), dtfac, 1.0 / h->dx[0], 1.0 / h->dx[1], 1.0 / h->dx[2], h->p.gam,
                newton_cfg(h->p), floor_cfg(h->p), chain_cfg(h->p)};
    const int nb = 2 * h->sms, rc_ = h->p.recon, rm_ = h->p.riemann;
    if (rc_ == 0 && rm_ == 0) chain_kernel<0, 0><<<nb, 128, 0, h->stream>>>(a);
    else if (rc_ == 0) chain_kernel<0, 1><<<nb, 128, 0, h->stream>>>(a);
    else if (rm_ == 0) chain_kernel<1, 0><<<nb, 128, 0, h->stream>>>(a);
    else chain_kernel<1, 1><<<nb, 128, 0, h->stream>>>(a);
    h->launches++;
    CK(cudaGetLastError());
  }
  if (h->p.polar_damp) {  // P:L311; A16
    Timed t_(h, CUHARM_K_BC);
    polar_damp_kernel<<<dim3((d.n3 + 127) / 128, d.n1, 2), 128, 0, h->stream>>>(d, Pout);
    h->launches++;
    CK(cudaGetLastError());
  }
  int rc = launch_bc(h, Pout, nullptr);
  if (rc || !with_repair) return rc;
  {
    Timed t_(h, CUHARM_K_FIXUP);
    unsigned long long* fixw = h->cnt + CNT_FIX + which * CNT_FIXW;
    FixArgs a{d, Pout, h->flag, h->list, nfail, h->p.inv_chain ? fixw + CNT_FIXW - 1 : nullptr, h->cnt + CNT_STATS, fixw, h->gC,
              h->floors, h->p.fixup_max_passes, h->p.gam, newton_cfg(h->p), floor_cfg(h->p)};
    const int rf = launch_fixup(h, a);
    if (rf) return rf;
  }
  CK(cudaGetLastError());
  return launch_bc(h, Pout, nfail);
}

// the step size is read by the kernels from the device scalar cnt[CNT_CLOCK] (written just before by set_dt_kernel or
// dt_from_cw_kernel), so this sequence -- and the graph recorded from it -- is the same for every dt
int enqueue_step(cuharm_ctx* h) {
  // per-step counters: failure counts of the two substeps, the c_w maxima of predictor and corrector
  CK(cudaMemsetAsync(h->cnt + CNT_NFAIL, 0, (CNT_STEP_END - CNT_NFAIL) * sizeof(unsigned long long), h->stream));
  int rc = substep(h, h->prim, h->prim, h->Phalf, 0.5, 0);  // predictor: fluxes and source from P^n, dtau = dt/2
  if (rc) return rc;
  return substep(h, h->Phalf, h->prim, h->prim, 1.0, 1);    // corrector: from the half-step state, in place, dtau = dt
}

// one step with the step size already in the device scalar: plain launches, or replay of the recorded graph
int run_step(cuharm_ctx* h) {
  h->stepped = true;
  if (!h->use_graph) return enqueue_step(h);
  if (!h->gexec) {  // record once; dt is not part of the graph
    cudaGraph_t g = nullptr;
    const int64_t before = h->launches;
    // record on a private stream (the caller's may be the legacy default stream, which cannot be captured);
    // the instantiated graph is then launched on the caller's stream
    if (!h->cap_stream) CK(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
    cudaStream_t user = h->stream;
    CK(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal));
    h->stream = h->cap_stream;
    h->capturing = true;
    int rc = enqueue_step(h);
    h->capturing = false;
    h->stream = user;
    cudaError_t e = cudaStreamEndCapture(h->cap_stream, &g);  // also ends a capture that failed half way
    h->graph_nodes = h->launches - before;
    h->launches = before;
    if (rc) { if (g) cudaGraphDestroy(g); (void)cudaGetLastError(); return rc; }
    if (e != cudaSuccess) { if (g) cudaGraphDestroy(g); return cuda_fail(e, "cudaStreamEndCapture"); }
    e = cudaGraphInstantiate(&h->gexec, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { h->gexec = nullptr; return cuda_fail(e, "cudaGraphInstantiate"); }
  }
  CK(cudaGraphLaunch(h->gexec, h->stream));
  h->launches += h->graph_nodes;
  return CUHARM_OK;
}

int check_params(const cuharm_params* p) {
  if (p->struct_bytes != (int32_t)sizeof(cuharm_params)) return CUHARM_EINVAL;
  if (p->n1 < 1 || p->n2 < 1 || p->n3 < 1 || p->ng < 3 || p->ng > 8) return CUHARM_EINVAL;
  if (p->coords < 0 || p->coords > 1 || p->recon < 0 || p->recon > 1 || p->riemann < 0 || p->riemann > 1) return CUHARM_EINVAL;
  const int bcs[3] = {p->bc_x1, p->bc_x2, p->bc_x3};
  for (int c = 0; c < 3; c++)
    if (bcs[c] < 0 || bcs[c] > 3) return CUHARM_EINVAL;
  if (p->bc_x1 == 2 || p->bc_x3 == 2) return CUHARM_EINVAL;  // the polar reflection belongs to X2
  if (p->bc_x2 == 2 && p->n2 < p->ng) return CUHARM_EINVAL;  // a mirror image needs ng interior zones
  if (!(p->gam > 1.0) || !(p->newton_tol > 0.0) || p->newton_maxit < 1 || p->newton_extra < 0 || p->fixup_max_passes < 0 ||
      p->fixup_max_passes > FIXUP_MAX_PASSES_CAP)
    return CUHARM_EINVAL;
  if (p->coords == 0) {
    if (!(p->r_in - p->R0 > 0.0) || !(p->r_out > p->r_in) || !(std::fabs(p->a) <= 1.0)) return CUHARM_EINVAL;
    if (p->n_x < 0 || p->n_x > 16 || !std::isfinite(p->r_break)) return CUHARM_EINVAL;
  } else {
    for (int c = 0; c < 3; c++)
      if (!(p->xmax[c] > p->xmin[c])) return CUHARM_EINVAL;
  }
  if (p->polar_damp < 0 || p->polar_damp > 1 || p->reserved != 0) return CUHARM_EINVAL;
  if (p->n1_global < 0 || (p->n1_global > 0 && (p->i_offset < 0 || p->i_offset + p->n1 > p->n1_global || p->slab_lo < 0 ||
                                                p->slab_lo > 1 || p->slab_hi < 0 || p->slab_hi > 1)))
    return CUHARM_EINVAL;
  if (p->n1_global > 0 && (p->slab_lo || p->slab_hi) && p->n1 < p->ng) return CUHARM_EINVAL;  // a halo is ng interior planes
  if (p->polar_damp && (p->bc_x2 != 2 || p->n2 < 6)) return CUHARM_EINVAL;
  if (p->inv_chain < 0 || p->inv_chain > 1) return CUHARM_EINVAL;
  if (p->inv_chain && (p->brent_maxit < 1 || !(p->brent_tol >= 0.0) || !std::isfinite(p->beta_min))) return CUHARM_EINVAL;
  if ((long long)(p->n1 + 2 * p->ng) * (p->n2 + 2 * p->ng) * (p->n3 + 2 * p->ng) > 2000000000LL) return CUHARM_EINVAL;
  return CUHARM_OK;
}

}  // namespace

extern "C" {

int cuharm_grid_init(cuharm_handle* out, const cuharm_params* p, void* cuda_stream) {
  if (!out || !p) return CUHARM_EINVAL;
  int rc = check_params(p);
  if (rc) return rc;
  int ndev = 0;
  CK(cudaGetDeviceCount(&ndev));
  if (ndev < 1) return cuda_fail(cudaErrorNoDevice, "cuharm_grid_init");
  cuharm_ctx* h = new (std::nothrow) cuharm_ctx();
  if (!h) return CUHARM_ENOMEM;
  h->p = *p;
  h->stream = (cudaStream_t)cuda_stream;
  {  // the device current at creation owns the stream and every later launch
    const cudaError_t e = cudaGetDevice(&h->dev);
    if (e != cudaSuccess) { delete h; return cuda_fail(e, "cudaGetDevice"); }
  }
  Dims& d = h->d;
  d.n1 = p->n1; d.n2 = p->n2; d.n3 = p->n3; d.ng = p->ng;
  d.n1g = p->n1 + 2 * p->ng; d.n2g = p->n2 + 2 * p->ng; d.n3g = p->n3 + 2 * p->ng;
  d.s2 = d.n3g; d.s1 = (long long)d.n2g * d.n3g; d.nz = (long long)d.n1g * d.s1;
  if (p->coords == 0) {  // eq. 39: uniform in X1 = ln(r - R0), X2 in [-1,1], X3 in [0, 2 pi)
    const double PI = 3.14159265358979323846;
    h->x0[0] = std::log(p->r_in - p->R0);
    // outer edge: the X1 at which eq. 39's radial map reaches r_out.  On the hyper-exponential branch that is the
    // root of X + (X - x_b)^n = ln(r_out - R0), found by Newton from above (the function is convex and increasing)
    double x_out = std::log(p->r_out - p->R0);
    h->xb = 0.0;
    h->nx = 0;
    if (p->n_x >= 2 && p->r_break > p->R0) {
      h->nx = p->n_x;
      h->xb = std::log(p->r_break - p->R0);
      const double target = x_out;
      if (target > h->xb) {
        double x = target;
        for (int it = 0; it < 100; it++) {
          const double y = x - h->xb;
          const double f = x + std::pow(y, h->nx) - target;
          const double fp = 1.0 + h->nx * std::pow(y, h->nx - 1);
          const double xn = x - f / fp;
          if (std::fabs(xn - x) <= 1e-16 * std::fabs(x)) { x = xn; break; }
          x = xn;
        }
        x_out = x;
      }
    }
    h->dx[0] = (x_out - h->x0[0]) / (p->n1_global > 0 ? p->n1_global : p->n1);
    h->x0[1] = -1.0; h->dx[1] = 2.0 / p->n2;
    h->x0[2] = 0.0;  h->dx[2] = 2.0 * PI / p->n3;
  } else {
    const int n[3] = {p->n1_global > 0 ? p->n1_global : p->n1, p->n2, p->n3};
    for (int c = 0; c < 3; c++) { h->x0[c] = p->xmin[c]; h->dx[c] = (p->xmax[c] - p->xmin[c]) / n[c]; }
  }
  {  // opt in to the dynamic shared memory of the bulk-copy update kernel (67.5 KB per block)
    auto setup = [&](auto kern_t, auto kern_f, int tb, int& blocks, int smem_bytes = 0) {
      const int smem = smem_bytes ? smem_bytes : upd_smem(tb);
      int dev = 0, sms = 0, per = 0;
      if (cudaFuncSetAttribute(kern_t, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return false;
      if (cudaFuncSetAttribute(kern_f, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return false;
      cudaGetDevice(&dev);
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
      if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, kern_f, tb, smem) != cudaSuccess || per < 1) return false;
      blocks = sms * per;  // persistent grid: every SM filled with as many blocks as fit
      return true;
    };
    h->upd_tma = p->inv_chain
                     ? setup(update_tma_kernel<true, 128, true>, update_tma_kernel<false, 128, true>, 128, h->upd_blocks) &&
                           setup(update_tma_kernel<true, 64, true>, update_tma_kernel<false, 64, true>, 64, h->upd_blocks64)
                     : setup(update_tma_kernel<true, 128, false>, update_tma_kernel<false, 128, false>, 128, h->upd_blocks) &&
                           setup(update_tma_kernel<true, 64, false>, update_tma_kernel<false, 64, false>, 64, h->upd_blocks64);
    if (!h->upd_tma) cudaGetLastError();
    // the tensor-map version of the same kernel (the maps themselves are encoded at bind time, for the bound arrays)
    h->upd_tmap = p->inv_chain
                      ? setup(update_tmap_kernel<true, 128, true>, update_tmap_kernel<false, 128, true>, 128, h->tmap_blocks, tmap_smem(128)) &&
                            setup(update_tmap_kernel<true, 64, true>, update_tmap_kernel<false, 64, true>, 64, h->tmap_blocks64, tmap_smem(64))
                      : setup(update_tmap_kernel<true, 128, false>, update_tmap_kernel<false, 128, false>, 128, h->tmap_blocks, tmap_smem(128)) &&
                            setup(update_tmap_kernel<true, 64, false>, update_tmap_kernel<false, 64, false>, 64, h->tmap_blocks64, tmap_smem(64));
    if (!h->upd_tmap) cudaGetLastError();
    h->tmap_enable = std::getenv("CUHARM_NO_TMAP") == nullptr;
    {
      int dev = 0, sms = 0;
      cudaGetDevice(&dev);
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
      if (sms > 0) h->sms = sms;
      int coop = 0, per = 0;
      if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) == cudaSuccess && coop &&
          cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, fixup_kernel, FIX_THREADS, 0) == cudaSuccess && per >= 1)
        h->coop = true;
    }
  }
  *out = h;
  return CUHARM_OK;
}

size_t cuharm_workspace_bytes(cuharm_handle h) { return h ? layout(h->d, h->p.inv_chain != 0).total : 0; }

int cuharm_bind(cuharm_handle h, double* d_prim, void* d_workspace, size_t ws_bytes) {
  if (!h || !d_prim || !d_workspace) return CUHARM_EINVAL;
  if (((uintptr_t)d_workspace & 255) || ((uintptr_t)d_prim & 15)) return CUHARM_EINVAL;
  const WsLayout L = layout(h->d, h->p.inv_chain != 0);
  if (ws_bytes < L.total) return CUHARM_ENOMEM;
  DevGuard dg_(h);
  const bool same_ws = h->ws == (char*)d_workspace;
  const bool same_prim = h->prim == d_prim;
  h->prim = d_prim;
  h->ws = (char*)d_workspace;
  h->gC = (Geom*)(h->ws + L.gC); h->gF1 = (Geom*)(h->ws + L.gF1); h->gF2 = (Geom*)(h->ws + L.gF2);
  h->conn = (double*)(h->ws + L.conn); h->srcw = (double*)(h->ws + L.srcw); h->rec = (double*)(h->ws + L.rec); h->floors = (double*)(h->ws + L.floors);
  for (int k = 0; k < 3; k++) h->F[k] = (double*)(h->ws + L.F[k]);
  h->E = (double*)(h->ws + L.E); h->Phalf = (double*)(h->ws + L.Phalf);
  h->flag = (int*)(h->ws + L.flag); h->list = (int*)(h->ws + L.list);
  h->cnt = (unsigned long long*)(h->ws + L.cnt);
  h->ustar = h->p.inv_chain ? (double*)(h->ws + L.ustar) : nullptr;
  if (!same_ws) h->have_geom = false;
  // a recorded graph holds the array addresses: it stays valid only if both are unchanged
  if (h->gexec && !(same_ws && same_prim)) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
  h->maps_ok = h->upd_tmap && h->tmap_enable && encode_update_maps(h);
  h->bound = true;
  h->stepped = false;
  h->dt_set = h->half_done = false;
  CK(cudaMemsetAsync(h->flag, 0, (size_t)h->d.nz * sizeof(int), h->stream));  // ghost zones always count as good
  CK(cudaMemsetAsync(h->cnt, 0, CNT_TOTAL * sizeof(unsigned long long), h->stream));
  if (h->have_geom) {
    int rc = launch_bc(h, h->prim, nullptr);
    if (rc) return rc;
    // the half-step array keeps the caller's ghost values where a boundary is `fixed`
    CK(cudaMemcpyAsync(h->Phalf, h->prim, 8 * (size_t)h->d.nz * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
  }
  return CUHARM_OK;
}

int cuharm_metric_precompute(cuharm_handle h) {
  if (!h) return CUHARM_EINVAL;
  if (!h->bound) return CUHARM_ESTATE;
  DevGuard dg_(h);
  const cuharm_params& p = h->p;
  const Dims& d = h->d;
  GeomArgs a{d.n1g, d.n2g, d.ng, d.n2, p.n1_global > 0 ? p.i_offset : 0, p.coords, (p.coords == 0 && p.bc_x2 == 2) ? 1 : 0, p.a, p.R0, p.hslope,
             h->xb, h->nx, h->x0[0], h->x0[1], h->dx[0], h->dx[1], p.rho_fl_coef, p.rho_fl_pow, p.rho_fl_abs, p.u_fl_coef,
             p.u_fl_pow, p.u_fl_abs, h->gC, h->gF1, h->gF2, h->conn, h->srcw, h->floors, h->rec};
  const int n = d.n1g * d.n2g;
  geom_kernel<<<(n + 63) / 64, 64, 0, h->stream>>>(a);
  h->launches++;
  CK(cudaGetLastError());
  h->have_geom = true;
  int rc = launch_bc(h, h->prim, nullptr);
  if (rc) return rc;
  CK(cudaMemcpyAsync(h->Phalf, h->prim, 8 * (size_t)d.nz * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
  return CUHARM_OK;
}

int cuharm_step(cuharm_handle h, double dt) {
  if (!h) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom) return CUHARM_ESTATE;
  if (!(dt > 0.0) || !std::isfinite(dt)) return CUHARM_EINVAL;
  DevGuard dg_(h);
  set_dt_kernel<<<1, 1, 0, h->stream>>>(reinterpret_cast<double*>(h->cnt + CNT_CLOCK), dt);
  h->launches++;
  CK(cudaGetLastError());
  return run_step(h);
}

int cuharm_set_dt(cuharm_handle h, double dt) {
  if (!h) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom) return CUHARM_ESTATE;
  if (!(dt > 0.0) || !std::isfinite(dt)) return CUHARM_EINVAL;
  DevGuard dg_(h);
  set_dt_kernel<<<1, 1, 0, h->stream>>>(reinterpret_cast<double*>(h->cnt + CNT_CLOCK), dt);
  h->launches++;
  CK(cudaGetLastError());
  h->dt_set = true;
  return CUHARM_OK;
}

int cuharm_substep(cuharm_handle h, int32_t which) {
  if (!h || which < 0 || which > 1) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom || !h->dt_set || (which == 1 && !h->half_done)) return CUHARM_ESTATE;
  DevGuard dg_(h);
  if (which == 0) {
    CK(cudaMemsetAsync(h->cnt + CNT_NFAIL, 0, (CNT_STEP_END - CNT_NFAIL) * sizeof(unsigned long long), h->stream));
    const int rc = substep(h, h->prim, h->prim, h->Phalf, 0.5, 0);
    if (rc) return rc;
    h->half_done = true;
    h->stepped = true;
    return CUHARM_OK;
  }
  h->half_done = false;
  h->dt_set = false;
  return substep(h, h->Phalf, h->prim, h->prim, 1.0, 1);
}

int cuharm_substep_update(cuharm_handle h, int32_t which) {
  if (!h || which < 0 || which > 1) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom || !h->dt_set || (which == 1 && !h->half_done)) return CUHARM_ESTATE;
  DevGuard dg_(h);
  if (which == 0) {
    CK(cudaMemsetAsync(h->cnt + CNT_NFAIL, 0, (CNT_STEP_END - CNT_NFAIL) * sizeof(unsigned long long), h->stream));
    const int rc = substep(h, h->prim, h->prim, h->Phalf, 0.5, 0, false);
    if (rc) return rc;
    h->half_done = true;
    h->stepped = true;
    return CUHARM_OK;
  }
  h->half_done = false;
  h->dt_set = false;
  return substep(h, h->Phalf, h->prim, h->prim, 1.0, 1, false);
}

int cuharm_repair_pass(cuharm_handle h, int32_t which, int32_t pass, int64_t out[2]) {
  if (!h || !out || which < 0 || which > 1 || pass < 0 || pass > h->p.fixup_max_passes) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom || !h->stepped) return CUHARM_ESTATE;
  DevGuard dg_(h);
  const Dims& d = h->d;
  unsigned long long* fixw = h->cnt + CNT_FIX + which * CNT_FIXW;
  unsigned long long* nfail = h->cnt + CNT_NFAIL + which;
  CK(cudaMemsetAsync(fixw + 1, 0, 2 * sizeof(unsigned long long), h->stream));
  FixArgs a{d, which == 0 ? h->Phalf : h->prim, h->flag, h->list, nfail, h->p.inv_chain ? fixw + CNT_FIXW - 1 : nullptr,
            h->cnt + CNT_STATS, fixw, h->gC, h->floors, h->p.fixup_max_passes, h->p.gam, newton_cfg(h->p), floor_cfg(h->p)};
  fixup_pass_kernel<<<2 * h->sms, 256, 0, h->stream>>>(a, pass, fixw + 1);
  h->launches++;
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(out, fixw + 1, 2 * sizeof(int64_t), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return CUHARM_OK;
}

int cuharm_substep_finish(cuharm_handle h, int32_t which) {
  if (!h || which < 0 || which > 1) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom || !h->stepped) return CUHARM_ESTATE;
  DevGuard dg_(h);
  return launch_bc(h, which == 0 ? h->Phalf : h->prim, nullptr);
}

size_t cuharm_flag_offset(cuharm_handle h) { return h ? layout(h->d, h->p.inv_chain != 0).flag : 0; }

size_t cuharm_half_offset(cuharm_handle h) { return h ? layout(h->d, h->p.inv_chain != 0).Phalf : 0; }

int cuharm_step_cfl(cuharm_handle h, double xi, double dt_max) {
  if (!h || !(xi > 0.0) || !std::isfinite(xi) || dt_max != dt_max) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom || !h->stepped) return CUHARM_ESTATE;
  DevGuard dg_(h);
  dt_from_cw_kernel<<<1, 1, 0, h->stream>>>(reinterpret_cast<double*>(h->cnt + CNT_CLOCK), h->cnt + CNT_CWPRED, xi, h->dx[0],
                                            h->dx[1], h->dx[2], dt_max);
  h->launches++;
  CK(cudaGetLastError());
  return run_step(h);
}

int cuharm_get_time(cuharm_handle h, double* t, double* dt_last) {
  if (!h || (!t && !dt_last)) return CUHARM_EINVAL;
  if (!h->bound) return CUHARM_ESTATE;
  DevGuard dg_(h);
  double c[2];
  CK(cudaMemcpyAsync(c, h->cnt + CNT_CLOCK, sizeof(c), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  if (dt_last) *dt_last = c[0];
  if (t) *t = c[1];
  return CUHARM_OK;
}

int cuharm_use_graph(cuharm_handle h, int32_t on) {
  if (!h) return CUHARM_EINVAL;
  DevGuard dg_(h);
  h->use_graph = on != 0;
  if (!on && h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
  return CUHARM_OK;
}

int64_t cuharm_launch_count(cuharm_handle h) { return h ? h->launches : 0; }

int cuharm_set_timing(cuharm_handle h, int32_t on) {
  if (!h) return CUHARM_EINVAL;
  DevGuard dg_(h);
  if (on && h->ev.empty()) {
    h->ev.resize(2 * 8192);
    for (auto& e : h->ev) CK(cudaEventCreate(&e));
  }
  h->timing = on != 0;
  h->ev_used = 0;
  h->ev_cat.clear();
  for (int c = 0; c < CUHARM_NCLASS; c++) { h->t_ms[c] = 0.0; h->t_n[c] = 0; }
  return CUHARM_OK;
}

int cuharm_get_timing(cuharm_handle h, double ms[CUHARM_NCLASS], int64_t count[CUHARM_NCLASS]) {
  if (!h || !ms || !count) return CUHARM_EINVAL;
  DevGuard dg_(h);
  CK(cudaStreamSynchronize(h->stream));
  for (size_t q = 0; q + 1 < h->ev_used; q += 2) {
    float t = 0.f;
    CK(cudaEventElapsedTime(&t, h->ev[q], h->ev[q + 1]));
    const int c = h->ev_cat[q / 2];
    h->t_ms[c] += t;
    h->t_n[c] += 1;
  }
  h->ev_used = 0;
  h->ev_cat.clear();
  for (int c = 0; c < CUHARM_NCLASS; c++) { ms[c] = h->t_ms[c]; count[c] = h->t_n[c]; }
  return CUHARM_OK;
}

int cuharm_cons_to_prim(cuharm_handle h, const double* d_U, double* d_prim_inout, int32_t* d_flag) {
  if (!h || !d_U || !d_prim_inout) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom) return CUHARM_ESTATE;
  DevGuard dg_(h);
  const Dims& d = h->d;
  ConvArgs a{d, d_U, d_prim_inout, d_flag, h->gC, h->p.gam, newton_cfg(h->p)};
  cons_to_prim_kernel<<<dim3((d.n3g + 127) / 128, d.n2g, d.n1g), 128, 0, h->stream>>>(a);
  h->launches++;
  CK(cudaGetLastError());
  return CUHARM_OK;
}

int cuharm_invert_fallback(cuharm_handle h, int32_t method, const double* d_U, const double* d_US, double* d_prim_inout,
                           int32_t* d_flag) {
  if (!h || !d_U || !d_prim_inout || method < 1 || method > 2 || (method == 2 && !d_US)) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom) return CUHARM_ESTATE;
  if (h->p.brent_maxit < 1 || !(h->p.brent_tol >= 0.0)) return CUHARM_EINVAL;
  DevGuard dg_(h);
  const Dims& d = h->d;
  FallbackArgs a{d, d_U, d_US, d_prim_inout, d_flag, h->gC, h->p.gam, method, chain_cfg(h->p)};
  fallback_kernel<<<dim3((d.n3g + 127) / 128, d.n2g, d.n1g), 128, 0, h->stream>>>(a);
  h->launches++;
  CK(cudaGetLastError());
  return CUHARM_OK;
}

int cuharm_prim_to_cons(cuharm_handle h, const double* d_prim, double* d_U) {
  if (!h || !d_prim || !d_U) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom) return CUHARM_ESTATE;
  DevGuard dg_(h);
  const Dims& d = h->d;
  ConvArgs a{d, d_prim, d_U, nullptr, h->gC, h->p.gam, newton_cfg(h->p)};
  prim_to_cons_kernel<<<dim3((d.n3g + 127) / 128, d.n2g, d.n1g), 128, 0, h->stream>>>(a);
  h->launches++;
  CK(cudaGetLastError());
  return CUHARM_OK;
}

static int read_cw(cuharm_handle h, const unsigned long long* d_cw, double cw[3]) {
  unsigned long long m[3];
  CK(cudaMemcpyAsync(m, d_cw, sizeof(m), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  for (int c = 0; c < 3; c++) std::memcpy(&cw[c], &m[c], sizeof(double));
  return CUHARM_OK;
}

static double dt_of_cw(const cuharm_ctx* h, double xi, const double cw[3]) {
  double inv = 0.0;
  for (int c = 0; c < 3; c++) {
    const double dtl = xi * h->dx[c] / cw[c];  // dt^l = xi dx^l / max c_w
    inv += 1.0 / dtl;                          // eq. 26
  }
  const double dt = 1.0 / inv;
  return std::isfinite(dt) && dt > 0.0 ? dt : 0.0;  // a non-finite wave speed anywhere (a NaN enters as +inf): 0
}

static int dt_from_cw(cuharm_handle h, const unsigned long long* d_cw, double xi, double* dt_out) {
  double cw[3];
  const int rc = read_cw(h, d_cw, cw);
  if (rc) return rc;
  *dt_out = dt_of_cw(h, xi, cw);
  return CUHARM_OK;
}

int cuharm_dt_of_cw(cuharm_handle h, double xi, const double cw[3], double* dt_out) {
  if (!h || !cw || !dt_out || !(xi > 0.0)) return CUHARM_EINVAL;
  *dt_out = dt_of_cw(h, xi, cw);
  return CUHARM_OK;
}

int cuharm_last_cw(cuharm_handle h, double cw[3]) {
  if (!h || !cw) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom || !h->stepped) return CUHARM_ESTATE;
  DevGuard dg_(h);
  return read_cw(h, h->cnt + CNT_CWPRED, cw);
}

int cuharm_cfl_cw(cuharm_handle h, double cw[3]) {
  if (!h || !cw) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom) return CUHARM_ESTATE;
  DevGuard dg_(h);
  unsigned long long* d_cw = h->cnt + CNT_CWSCR;
  CK(cudaMemsetAsync(d_cw, 0, 3 * sizeof(unsigned long long), h->stream));
  for (int dir = 1; dir <= 3; dir++) {
    int rc = launch_flux<false>(h, h->prim, dir, h->F[dir - 1], nullptr, d_cw + (dir - 1));
    if (rc) return rc;
  }
  return read_cw(h, d_cw, cw);
}

int cuharm_cfl_dt(cuharm_handle h, double xi, double* dt_out) {
  if (!h || !dt_out || !(xi > 0.0)) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom) return CUHARM_ESTATE;
  DevGuard dg_(h);
  unsigned long long* cw = h->cnt + CNT_CWSCR;
  CK(cudaMemsetAsync(cw, 0, 3 * sizeof(unsigned long long), h->stream));
  for (int dir = 1; dir <= 3; dir++) {
    int rc = launch_flux<false>(h, h->prim, dir, h->F[dir - 1], nullptr, cw + (dir - 1));
    if (rc) return rc;
  }
  return dt_from_cw(h, cw, xi, dt_out);
}

int cuharm_last_cfl_dt(cuharm_handle h, double xi, double* dt_out) {
  if (!h || !dt_out || !(xi > 0.0)) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom || !h->stepped) return CUHARM_ESTATE;
  DevGuard dg_(h);
  return dt_from_cw(h, h->cnt + CNT_CWPRED, xi, dt_out);
}

int cuharm_shell_fluxes(cuharm_handle h, int32_t i, double out[4]) {
  if (!h || !out) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom) return CUHARM_ESTATE;
  const Dims& d = h->d;
  if (i < 0 || i >= d.n1) return CUHARM_EINVAL;
  DevGuard dg_(h);
  // scratch: the head of the EMF array (idle between steps): n2 x 4 partial sums + 4 results
  double* partial = h->E;
  double* res = h->E + (size_t)d.n2 * 4;
  ShellArgs a{d, h->prim, h->gC, d.ng + i, h->p.gam, h->dx[1] * h->dx[2], partial, res};
  shell_flux_kernel<<<d.n2, 128, 0, h->stream>>>(a);
  shell_sum_kernel<<<1, 128, 0, h->stream>>>(a);
  h->launches += 2;
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(out, res, 4 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return CUHARM_OK;
}

int cuharm_divb(cuharm_handle h, double* max_abs, double* max_norm) {
  if (!h || !max_abs || !max_norm) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom) return CUHARM_ESTATE;
  const Dims& d = h->d;
  DevGuard dg_(h);
  const bool two_d = d.n3 == 1;
  const int khi = two_d ? d.ng : ((h->p.bc_x3 == 1) ? d.ng + d.n3 - 1 : d.ng + d.n3 - 2);
  unsigned long long* out = h->cnt + CNT_DIVB;
  CK(cudaMemsetAsync(out, 0, 2 * sizeof(unsigned long long), h->stream));
  if (d.n1 >= 2 && d.n2 >= 2 && khi >= d.ng) {
    DivbArgs a{d, h->prim, h->gC, 1.0 / h->dx[0], 1.0 / h->dx[1], 1.0 / h->dx[2], khi, out};
    divb_kernel<<<dim3((khi - d.ng + 1 + 127) / 128, d.n2 - 1, d.n1 - 1), 128, 0, h->stream>>>(a);
    h->launches++;
    CK(cudaGetLastError());
  }
  unsigned long long m[2];
  CK(cudaMemcpyAsync(m, out, sizeof(m), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  std::memcpy(max_abs, &m[0], sizeof(double));
  std::memcpy(max_norm, &m[1], sizeof(double));
  return CUHARM_OK;
}

int cuharm_get_geom(cuharm_handle h, int32_t loc, double* d_out) {
  if (!h || !d_out || loc < 0 || loc > 3) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom) return CUHARM_ESTATE;
  DevGuard dg_(h);
  const int n = h->d.n1g * h->d.n2g;
  const Geom* tab = loc == 1 ? h->gF1 : (loc == 2 ? h->gF2 : h->gC);
  geom_export_kernel<<<(n + 127) / 128, 128, 0, h->stream>>>(tab, h->conn, loc, n, d_out);
  h->launches++;
  CK(cudaGetLastError());
  return CUHARM_OK;
}

int cuharm_apply_bc(cuharm_handle h, double* d_prim) {
  if (!h || !d_prim) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom) return CUHARM_ESTATE;
  DevGuard dg_(h);
  return launch_bc(h, d_prim, nullptr);
}

int cuharm_apply_floors(cuharm_handle h, double* d_prim, int32_t* d_mask) {
  if (!h || !d_prim) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom) return CUHARM_ESTATE;
  DevGuard dg_(h);
  const Dims& d = h->d;
  FloorArgs a{d, d_prim, d_mask, h->gC, h->floors, h->p.gam, newton_cfg(h->p), floor_cfg(h->p)};
  floors_kernel<<<dim3((d.n3 + 127) / 128, d.n2, d.n1), 128, 0, h->stream>>>(a);
  h->launches++;
  CK(cudaGetLastError());
  return CUHARM_OK;
}

int cuharm_repair(cuharm_handle h, double* d_prim, const int32_t* d_flag) {
  if (!h || !d_prim || !d_flag) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom) return CUHARM_ESTATE;
  DevGuard dg_(h);
  const Dims& d = h->d;
  unsigned long long* nfail = h->cnt + CNT_NFAIL;
  unsigned long long* fixw = h->cnt + CNT_FIX;
  // only the failure counts and the repair scratch: the c_w maxima of the last predictor (CNT_CWPRED) stay, so that a
  // cuharm_step_cfl / cuharm_last_cfl_dt after this call still sees them
  CK(cudaMemsetAsync(h->cnt + CNT_NFAIL, 0, (CNT_CWPRED - CNT_NFAIL) * sizeof(unsigned long long), h->stream));
  CK(cudaMemsetAsync(h->cnt + CNT_FIX, 0, (CNT_STEP_END - CNT_FIX) * sizeof(unsigned long long), h->stream));
  repair_list_kernel<<<dim3((d.n3g + 127) / 128, d.n2g, d.n1g), 128, 0, h->stream>>>(d, d_flag, h->flag, h->list, nfail);
  FixArgs a{d, d_prim, h->flag, h->list, nfail, nullptr, h->cnt + CNT_STATS, fixw, h->gC, h->floors, h->p.fixup_max_passes,
            h->p.gam, newton_cfg(h->p), floor_cfg(h->p)};
  h->launches++;
  CK(cudaGetLastError());
  const int rf = launch_fixup(h, a);
  if (rf) return rf;
  // the library's flag array goes back to "all good" (its state between steps)
  CK(cudaMemsetAsync(h->flag, 0, (size_t)d.nz * sizeof(int), h->stream));
  return CUHARM_OK;
}

int cuharm_flux_dir(cuharm_handle h, const double* d_prim, int32_t dir, double* d_F, double* d_cw) {
  if (!h || !d_prim || !d_F || dir < 1 || dir > 3) return CUHARM_EINVAL;
  if (!h->bound || !h->have_geom) return CUHARM_ESTATE;
  DevGuard dg_(h);
  CK(cudaMemsetAsync(d_F, 0, 8 * (size_t)h->d.nz * sizeof(double), h->stream));
  if (d_cw) CK(cudaMemsetAsync(d_cw, 0, (size_t)h->d.nz * sizeof(double), h->stream));
  return launch_flux<true>(h, d_prim, dir, d_F, d_cw, h->cnt + CNT_CWSCR + (dir - 1));
}

int cuharm_get_stats(cuharm_handle h, int64_t out[8]) {
  if (!h || !out) return CUHARM_EINVAL;
  if (!h->bound) return CUHARM_ESTATE;
  DevGuard dg_(h);
  CK(cudaMemcpyAsync(out, h->cnt + CNT_STATS, 8 * sizeof(int64_t), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return CUHARM_OK;
}

int cuharm_get_chain_stats(cuharm_handle h, int64_t out[4]) {
  if (!h || !out) return CUHARM_EINVAL;
  if (!h->bound) return CUHARM_ESTATE;
  DevGuard dg_(h);
  CK(cudaMemcpyAsync(out, h->cnt + CNT_CHAIN, 4 * sizeof(int64_t), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return CUHARM_OK;
}

int cuharm_destroy(cuharm_handle h) {
  if (!h) return CUHARM_EINVAL;
  {
  DevGuard dg_(h);
  if (h->gexec) cudaGraphExecDestroy(h->gexec);
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  for (int k = 0; k < 2; k++) if (h->side[k]) cudaStreamDestroy(h->side[k]);
  for (int k = 0; k < 3; k++) if (h->fj[k]) cudaEventDestroy(h->fj[k]);
  for (auto& e : h->ev) cudaEventDestroy(e);
  }
  delete h;
  return CUHARM_OK;
}

const char* cuharm_strerror(int code) {
  switch (code) {
    case CUHARM_OK: return "ok";
    case CUHARM_EINVAL: return "invalid argument";
    case CUHARM_ESTATE: return "call out of order (bind / metric_precompute / step)";
    case CUHARM_ECUDA: return g_errtext;
    case CUHARM_ENOMEM: return "workspace too small";
    default: return "unknown error code";
  }
}

}  // extern "C"
