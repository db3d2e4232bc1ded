// cuharm_divb_noalloc: the eq. 23 divergence diagnostic (reading A4) for callers that have no way to obtain
// device memory of their own beyond the arrays they were handed.
//
// Who that is.  Every other call of libcuharm works on a context whose workspace the caller allocates (cuharm_bind wants
// cuharm_workspace_bytes of it: gigabytes at 256^3).  An in-situ monitor, an I/O or analysis plug-in, a checker hooked into
// somebody else's time loop is often in no position to do that: the host code has handed the whole device to its own pool
// (a framework's caching allocator, a simulation arena sized to the last byte), the plug-in interface passes it the
// primitive array and a sqrt(-g) table and nothing else, and cudaMalloc / cudaFree are off limits there anyway because
// they may fail on a full device and they stall every stream of the process while they run.  Such a caller still wants to
// know that div B sits at round-off.  This one entry point serves it: no context, no workspace, no allocation of any kind.
//
// How.  The reduction needs a little scratch (one pair of partial maxima per (i, j) corner row).  It lives in a file-scope
// static __device__ array of fixed size, CUHARM_DIVB_NOALLOC_MAX_ROWS rows = 2 MiB, which every GPU that loads the
// library carries until the process exits.  Grids with more corner rows than that are refused (CUHARM_ENOMEM).
//
// Sharing.  There is ONE scratch array per device and every call on that device uses it.  Calls whose kernels may overlap
// on the GPU (different streams, no ordering between them) race on it and return garbage; order them on one stream or
// with events.  The array keeps whatever the last call left there.  Nothing in it has to start at zero: the first kernel
// overwrites every slot the second kernel goes on to read (rows 0 .. nrows-1 of THIS call), and slots beyond are never
// read, so stale partials of an earlier, larger call cannot leak into a result.
//
// Set-up.  In host code the name of a __device__ array is only a host-side shadow of the symbol, not a device address; a
// kernel handed that name would fault or quietly scribble on host-mapped memory.  The first call on each device therefore
// asks the runtime for the real address (cudaGetSymbolAddress, with that device current) and keeps it per device ordinal.
// Because that first call talks to the runtime beyond plain launches, make it before you start capturing a stream.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "cuharm.h"

namespace {

constexpr int MAX_ROWS = CUHARM_DIVB_NOALLOC_MAX_ROWS;
constexpr int MAX_DEVICES = 64;

// [row][2]: order-preserving integer images of max |D| and max |D| / sum |terms| over the corners of one (i, j) row
static __device__ __align__(256) unsigned long long g_divb_scratch[2 * (size_t)MAX_ROWS];

std::mutex g_setup_mutex;
unsigned long long* g_scratch_addr[MAX_DEVICES] = {};  // device address of g_divb_scratch, per device ordinal

thread_local char g_text[256] = "no error recorded";

int fail(int code, const char* msg) {
  snprintf(g_text, sizeof(g_text), "%s", msg);
  return code;
}

int cuda_fail(cudaError_t e, const char* what) {
  snprintf(g_text, sizeof(g_text), "%s: %s", what, cudaGetErrorString(e));
  (void)cudaGetLastError();
  return CUHARM_ECUDA;
}

// Device address of the scratch array on the CURRENT device; looked up once per device.
int scratch_for_current_device(unsigned long long** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
  if (dev < 0 || dev >= MAX_DEVICES) return fail(CUHARM_EINVAL, "cuharm_divb_noalloc: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (!g_scratch_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_divb_scratch);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(g_divb_scratch)");
    if (!p) return fail(CUHARM_ECUDA, "cuharm_divb_noalloc: cudaGetSymbolAddress returned a null address");
    g_scratch_addr[dev] = static_cast<unsigned long long*>(p);
  }
  *out = g_scratch_addr[dev];
  return CUHARM_OK;
}

// a non-negative double as an integer that orders the same way; NaN counts as +infinity, anything negative as 0
__device__ __forceinline__ unsigned long long image_of(double v) {
  const double vv = v >= 0.0 ? v : (v != v ? __longlong_as_double(0x7ff0000000000000LL) : 0.0);
  return (unsigned long long)__double_as_longlong(vv);
}

__device__ __forceinline__ unsigned long long warp_max(unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long w = __shfl_xor_sync(0xffffffffu, v, o);
    v = w > v ? w : v;
  }
  return v;
}

struct RowArgs {
  const double* P;   // prim[8][n1g][n2g][n3g]; only B^1..3 (components 5..7) are read
  const double* sg;  // sqrt(-g) at zone centres, [n1g][n2g]
  int n2, n3, ng, n2g;
  long long s1, s2, nz;
  double idx1, idx2, idx3;
  int khi;           // last corner index along k (array index, ghosts included)
  unsigned long long* part;  // [nrows][2]
};

// Stage 1: block r handles the corners (i, j, k = ng .. khi) of row r = (i - ng) * (n2 - 1) + (j - ng); same expression,
// term by term, as the context-based cuharm_divb evaluates per corner.
__global__ void __launch_bounds__(128) divb_rows_kernel(RowArgs a) {
  const int row = blockIdx.x;
  const int i = a.ng + row / (a.n2 - 1), j = a.ng + row % (a.n2 - 1);
  const bool two_d = a.n3 == 1;
  const double w = two_d ? 0.5 : 0.25;
  double sg[2][2];
  for (int l1 = 0; l1 < 2; l1++)
    for (int l2 = 0; l2 < 2; l2++) sg[l1][l2] = __ldg(&a.sg[(i + l1) * a.n2g + j + l2]);
  unsigned long long mabs = 0ull, mnorm = 0ull;
  for (int k = a.ng + threadIdx.x; k <= a.khi; k += 128) {
    double D = 0.0, A = 0.0;
    for (int l1 = 0; l1 < 2; l1++)
      for (int l2 = 0; l2 < 2; l2++)
        for (int l3 = 0; l3 < (two_d ? 1 : 2); l3++) {
          const long long n = (i + l1) * a.s1 + (j + l2) * a.s2 + k + l3;
          const double t1 = (l1 ? 1.0 : -1.0) * sg[l1][l2] * a.P[5 * a.nz + n] * w * a.idx1;
          const double t2 = (l2 ? 1.0 : -1.0) * sg[l1][l2] * a.P[6 * a.nz + n] * w * a.idx2;
          D += t1 + t2;
          A += fabs(t1) + fabs(t2);
          if (!two_d) {
            const double t3 = (l3 ? 1.0 : -1.0) * sg[l1][l2] * a.P[7 * a.nz + n] * w * a.idx3;
            D += t3;
            A += fabs(t3);
          }
        }
    const unsigned long long ia = image_of(fabs(D));
    // corners whose terms sum to < 1e-290 do not enter the normalised measure (A4), as in cuharm_divb
    const unsigned long long in = image_of(A > 1e-290 ? fabs(D) / A : 0.0);
    mabs = ia > mabs ? ia : mabs;
    mnorm = in > mnorm ? in : mnorm;
  }
  __shared__ unsigned long long sh[4][2];
  mabs = warp_max(mabs);
  mnorm = warp_max(mnorm);
  if ((threadIdx.x & 31) == 0) { sh[threadIdx.x >> 5][0] = mabs; sh[threadIdx.x >> 5][1] = mnorm; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int wp = 1; wp < 4; wp++) {
      mabs = sh[wp][0] > mabs ? sh[wp][0] : mabs;
      mnorm = sh[wp][1] > mnorm ? sh[wp][1] : mnorm;
    }
    a.part[2 * (size_t)row + 0] = mabs;  // every row slot of this call is written before stage 2 reads it
    a.part[2 * (size_t)row + 1] = mnorm;
  }
}

// Stage 2: one block folds the nrows partial pairs and writes the two doubles the caller asked for.
__global__ void __launch_bounds__(1024) divb_fold_kernel(const unsigned long long* part, int nrows, double* out) {
  unsigned long long mabs = 0ull, mnorm = 0ull;
  for (int r = threadIdx.x; r < nrows; r += 1024) {
    const unsigned long long x = part[2 * (size_t)r], y = part[2 * (size_t)r + 1];
    mabs = x > mabs ? x : mabs;
    mnorm = y > mnorm ? y : mnorm;
  }
  __shared__ unsigned long long sh[32][2];
  mabs = warp_max(mabs);
  mnorm = warp_max(mnorm);
  if ((threadIdx.x & 31) == 0) { sh[threadIdx.x >> 5][0] = mabs; sh[threadIdx.x >> 5][1] = mnorm; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int wp = 1; wp < 32; wp++) {
      mabs = sh[wp][0] > mabs ? sh[wp][0] : mabs;
      mnorm = sh[wp][1] > mnorm ? sh[wp][1] : mnorm;
    }
    out[0] = __longlong_as_double((long long)mabs);
    out[1] = __longlong_as_double((long long)mnorm);
  }
}

}  // namespace

extern "C" {

int cuharm_divb_noalloc(const double* d_prim, const double* d_sqrtg, int32_t n1, int32_t n2, int32_t n3, int32_t ng,
                        const double dx[3], int32_t periodic_x3, void* cuda_stream, double* d_out) {
  if (!d_prim || !d_sqrtg || !dx || !d_out) return fail(CUHARM_EINVAL, "cuharm_divb_noalloc: null pointer");
  if (n1 < 1 || n2 < 1 || n3 < 1 || ng < 1 || ng > 8) return fail(CUHARM_EINVAL, "cuharm_divb_noalloc: bad grid shape");
  for (int c = 0; c < 3; c++)
    if (!(dx[c] > 0.0) || !(dx[c] < 1e300)) return fail(CUHARM_EINVAL, "cuharm_divb_noalloc: dx must be finite and > 0");
  const long long nrows = (long long)(n1 - 1) * (n2 - 1);
  if (nrows > MAX_ROWS) {
    snprintf(g_text, sizeof(g_text),
             "cuharm_divb_noalloc: (n1-1)*(n2-1) = %lld corner rows exceed the static scratch of %d rows "
             "(CUHARM_DIVB_NOALLOC_MAX_ROWS); use cuharm_divb on a context with a workspace for larger grids",
             nrows, MAX_ROWS);
    return CUHARM_ENOMEM;
  }
  unsigned long long* part = nullptr;
  const int rc = scratch_for_current_device(&part);
  if (rc != CUHARM_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int n2g = n2 + 2 * ng, n3g = n3 + 2 * ng;
  const bool two_d = n3 == 1;
  // corners whose 8 (2D: 4) cells are interior; a periodic X3 adds the corner between the last and the first zone,
  // whose upper cells are the first ghost layer (valid after a ghost fill)
  const int khi = two_d ? ng : (periodic_x3 ? ng + n3 - 1 : ng + n3 - 2);
  int rows = 0;
  if (nrows > 0 && khi >= ng) {
    rows = (int)nrows;
    RowArgs a{d_prim, d_sqrtg, n2, n3, ng, n2g, (long long)n2g * n3g, (long long)n3g, (long long)(n1 + 2 * ng) * n2g * n3g,
              1.0 / dx[0], 1.0 / dx[1], 1.0 / dx[2], khi, part};
    divb_rows_kernel<<<rows, 128, 0, st>>>(a);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "divb_rows_kernel launch");
  }
  divb_fold_kernel<<<1, 1024, 0, st>>>(part, rows, d_out);  // rows == 0: no corner to look at, both results are 0
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(e, "divb_fold_kernel launch");
  return CUHARM_OK;
}

const char* cuharm_divb_noalloc_errtext(void) { return g_text; }

}  // extern "C"
