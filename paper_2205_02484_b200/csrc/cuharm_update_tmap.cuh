// cuharm_update_tmap.cuh — the fused source + update + inversion + floors kernel (S4-S7, S9) fed by TENSOR-MAP bulk
// copies (cp.async.bulk.tensor, the TMA engine's tiled mode): the operands of a tile of TB zones are twelve boxes of the
// 4-D arrays [component][i][j][k] (8-byte elements) instead of 63 one-dimensional row copies, so a tile costs a
// dozen copy instructions instead of 66.  Same tiles, same strip order (TileWalk), same per-zone arithmetic (update_zone)
// and the same code for the edge EMFs (edge_emfs) as update_tma_kernel: results are bit-identical to it.
//
// Boxes (inner extent TB + 2 zones: k0 - 1 .. k0 + TB; zones past the end of the array are zero-filled by the engine
// and never used), in the order they sit in shared memory, rows = (component, i, j) combinations of the box:
//   0  P^n        comps 0..7                        8 rows   [c]
//   1  P-flux     comps 0..7 (corrector only)       8 rows   [c]
//   2  F1 hydro   comps 0..4, i..i+1               10 rows   [c][i']
//   3  F2 hydro   comps 0..4, j..j+1               10 rows   [c][j']
//   4  F3 hydro   comps 0..4                        5 rows   [c]
//   5  F2(B3)     comp 5, j..j+1                    2 rows   [j']
//   6  F3(B2)     comp 6, j-1..j+1                  3 rows   [j']
//   7  F3(B1)     comp 5, i-1..i+1                  3 rows   [i']
//   8  F1(B3)     comp 6, i..i+1                    2 rows   [i']
//   9  F1(B2)     comp 5, (i..i+1) x (j-1..j+1)     6 rows   [i'][j']
//  10  F2(B1)     comp 6, (i-1..i+1) x (j..j+1)     6 rows   [i'][j']
// plus the per-(i,j) record (geometry 20, source weights 14, floors 2 doubles) as one plain bulk copy.
#pragma once
#include <cuda.h>

#include "cuharm_kernels.cuh"

namespace cuharm {

constexpr int TMAP_NBOX = 11;
struct UpdMaps {
  CUtensorMap m[TMAP_NBOX];
};

__host__ __device__ constexpr int tmap_rows(int b) {
  return b == 0 ? 8 : b == 1 ? 8 : b == 2 ? 10 : b == 3 ? 10 : b == 4 ? 5 : b == 5 ? 2 : b == 6 ? 3 : b == 7 ? 3 : b == 8 ? 2 : 6;
}
// byte offset of box b in the stage: every box starts on a 128-byte boundary (a requirement of the tensor copies)
__host__ __device__ constexpr int tmap_off(int b, int tb) {
  int off = 0;
  for (int q = 0; q < b; q++) off = (off + tmap_rows(q) * (tb + 2) * 8 + 127) & ~127;
  return off;
}
constexpr int TMAP_REC = 36;  // doubles of the per-(i,j) record
__host__ __device__ constexpr int tmap_smem(int tb) { return tmap_off(TMAP_NBOX, tb) + 2 * 64 * 8; }

__device__ __forceinline__ void tensor_g2s_4d(unsigned dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, unsigned bar) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(dst),
      "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar)
      : "memory");
}

// stage layout of update_tmap_kernel for edge_emfs (cuharm_kernels.cuh): box 5 F2(B3) rows j, j+1; box 6 F3(B2) rows j-1,
// j, j+1; box 7 F3(B1) rows i-1, i, i+1; box 8 F1(B3) rows i, i+1; box 9 F1(B2) rows [i' - i][j' - (j-1)]; box 10 F2(B1)
// rows [i' - (i-1)][j' - j]; a staged row starts one zone below the tile
template <int TB>
struct BoxStage {
  const unsigned char* stage;
  int tc;
  template <int ARR, int A, int B>
  __device__ __forceinline__ double at() const {
    constexpr int box = 5 + ARR;
    constexpr int row = ARR == EMF_F2B3 ? A : ARR == EMF_F3B2 ? A + 1 : ARR == EMF_F3B1 ? A + 1 : ARR == EMF_F1B3 ? A
                        : ARR == EMF_F1B2 ? 3 * A + (B + 1) : 2 * (A + 1) + B;
    constexpr int off = ARR == EMF_F1B2 || ARR == EMF_F2B1 ? 0 : B;
    return reinterpret_cast<const double*>(stage + tmap_off(box, TB))[row * (TB + 2) + 1 + tc + off];
  }
};

template <bool SAME, int TB, bool CHAIN>
__global__ void __launch_bounds__(TB, (UPD_TMA_MINB * 128) / TB)
update_tmap_kernel(UpdArgs a, const __grid_constant__ UpdMaps maps, const double* __restrict__ rec, int ntiles, int nch, int wj) {
  constexpr int ROW = TB + 2;  // doubles per staged row
  extern __shared__ __align__(128) unsigned char stage[];
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
  TileWalk walk(tile, G, nch, wj, d.n1);  // strip order (cuharm_kernels.cuh)
  TileIdx cur = walk.idx(), nxt;
  double* const tab = reinterpret_cast<double*>(stage + tmap_off(TMAP_NBOX, TB));  // two slots of 64 doubles
  const unsigned st0 = smem_u32(stage);
  constexpr unsigned TX = (unsigned)((SAME ? 55 : 63) * ROW * 8 + TMAP_REC * 8);
  // one thread issues the dozen copies of a tile
  auto issue = [&](const TileIdx& x, int slot) {
    if (t != 0) return;
    const int k = d.ng + x.c * TB - 1, j = d.ng + x.j, i = d.ng + x.i;
    mbar_expect_tx(bar0, TX);
    tensor_g2s_4d(st0 + tmap_off(0, TB), &maps.m[0], k, j, i, 0, bar0);
    if (!SAME) tensor_g2s_4d(st0 + tmap_off(1, TB), &maps.m[1], k, j, i, 0, bar0);
    tensor_g2s_4d(st0 + tmap_off(2, TB), &maps.m[2], k, j, i, 0, bar0);
    tensor_g2s_4d(st0 + tmap_off(3, TB), &maps.m[3], k, j, i, 0, bar0);
    tensor_g2s_4d(st0 + tmap_off(4, TB), &maps.m[4], k, j, i, 0, bar0);
    tensor_g2s_4d(st0 + tmap_off(5, TB), &maps.m[5], k, j, i, 5, bar0);
    tensor_g2s_4d(st0 + tmap_off(6, TB), &maps.m[6], k, j - 1, i, 6, bar0);
    tensor_g2s_4d(st0 + tmap_off(7, TB), &maps.m[7], k, j, i - 1, 5, bar0);
    tensor_g2s_4d(st0 + tmap_off(8, TB), &maps.m[8], k, j, i, 6, bar0);
    tensor_g2s_4d(st0 + tmap_off(9, TB), &maps.m[9], k, j - 1, i, 5, bar0);
    tensor_g2s_4d(st0 + tmap_off(10, TB), &maps.m[10], k, j, i - 1, 6, bar0);
    bulk_g2s(smem_u32(tab + slot * 64), rec + ((size_t)i * d.n2g + j) * TMAP_REC, TMAP_REC * 8u, bar0);
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
    // this zone in row r of box b: the staged row starts one zone below the tile
#define BOXZ(b, r, o) (reinterpret_cast<const double*>(stage + tmap_off(b, TB))[(r) * ROW + 1 + tc + (o)])
    double pb[8], pf[8], fx[30], ex[12];
#pragma unroll
    for (int v = 0; v < 8; v++) pb[v] = BOXZ(0, v, 0);
#pragma unroll
    for (int v = 0; v < 8; v++) pf[v] = SAME ? pb[v] : BOXZ(1, v, 0);
#pragma unroll
    for (int v = 0; v < 5; v++) {
      fx[6 * v + 0] = BOXZ(2, 2 * v + 1, 0); fx[6 * v + 1] = BOXZ(2, 2 * v, 0);   // F1 at i+1, i
      fx[6 * v + 2] = BOXZ(3, 2 * v + 1, 0); fx[6 * v + 3] = BOXZ(3, 2 * v, 0);   // F2 at j+1, j
      fx[6 * v + 4] = BOXZ(4, v, 1);         fx[6 * v + 5] = BOXZ(4, v, 0);       // F3 at k+1, k
    }
    edge_emfs(BoxStage<TB>{stage, tc}, ex);  // eq. 21
#undef BOXZ
    // operands are in registers: release the stage (split barrier: arrive here, wait after the divergence arithmetic)
    mbar_arrive(bar0 + 8);
    double dU[8];
    zone_divergence(a, fx, ex, dU);
    mbar_wait(bar0 + 8, n & 1);
    if (tile + G < ntiles) issue(nxt, (n + 1) & 1);
    int cnt[5] = {0, 0, 0, 0, 0};
    const double* tb = tab + (n & 1) * 64;  // the per-(i,j) record of this tile stays valid in its own slot
    const Geom Gc = load_geom_shared(tb);
    update_zone<SAME, CHAIN>(a, pb, pf, dU, Gc, tb + 20, tb[34], tb[35], dtau, idx, q2, live, cnt);
#pragma unroll
    for (int q = 0; q < 5; q++) cnt_acc[q] += cnt[q];
  }
  update_stats(a, cnt_acc);
}

}  // namespace cuharm
