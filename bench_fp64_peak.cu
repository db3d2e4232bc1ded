// fp64_peak.cu — DFMA micro-benchmark behind the "alu" roofline of DESIGN.md section 5: what the fp64 pipe of one B200
// delivers, as warp-level DFMA instructions per second, for a given instruction-level parallelism (independent
// dependency chains per thread) and number of resident warps per SM sub-partition.  Stand-alone (no library code):
//     nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o fp64_peak fp64_peak.cu && ./fp64_peak
// or  python -m paper_2205_02484_b200.fp64_peak     (builds, runs, prints the table and one JSON line)
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>

template <int ILP>
__global__ void dfma_kernel(double* out, double a, double b, int iters, long long* cycles) {
  double x[ILP];
#pragma unroll
  for (int q = 0; q < ILP; q++) x[q] = threadIdx.x * 1e-9 + q;
  const long long t0 = clock64();
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int r = 0; r < 16; r++) {
#pragma unroll
      for (int q = 0; q < ILP; q++) x[q] = fma(x[q], a, b);  // ILP independent chains, 16 links each per trip
    }
  }
  const long long t1 = clock64();
  double s = 0.0;
#pragma unroll
  for (int q = 0; q < ILP; q++) s += x[q];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
  if (threadIdx.x == 0 && blockIdx.x == 0) *cycles = t1 - t0;
}

template <int ILP>
void run(int sms, int warps_per_smsp, double* d_out, long long* d_cyc, double clock_ghz) {
  const int iters = 4096;
  const int threads = 32 * 4 * warps_per_smsp;  // one block per SM, its warps spread over the 4 sub-partitions
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  dfma_kernel<ILP><<<sms, threads>>>(d_out, 0.999999, 1e-9, 16, d_cyc);  // warm-up
  cudaEventRecord(e0);
  dfma_kernel<ILP><<<sms, threads>>>(d_out, 0.999999, 1e-9, iters, d_cyc);
  cudaEventRecord(e1);
  cudaEventSynchronize(e1);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  long long cyc = 0;
  cudaMemcpy(&cyc, d_cyc, sizeof(cyc), cudaMemcpyDeviceToHost);
  const double per_warp = (double)iters * 16 * ILP;                   // DFMA warp instructions per warp
  const double total = per_warp * warps_per_smsp * 4.0 * sms;         // on the whole device
  const double cyc_per_inst_smsp = (double)cyc / (per_warp * warps_per_smsp);  // cycles per DFMA per sub-partition
  printf("ILP %d  warps/sub-partition %d : %7.3f cycles per warp-DFMA per sub-partition, %.3e warp-DFMA/s (%.1f Tflop/s), "
         "%.0f %% of 1 per 2 cycles at %.3f GHz\n",
         ILP, warps_per_smsp, cyc_per_inst_smsp, total / (ms * 1e-3), total * 64.0 / (ms * 1e-3) / 1e12,
         100.0 * (total / (ms * 1e-3)) / (sms * 4.0 * clock_ghz * 1e9 / 2.0), clock_ghz);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
}

int main() {
  int dev = 0, sms = 0, khz = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { fprintf(stderr, "no CUDA device\n"); return 1; }
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
  const double ghz = khz * 1e-6;
  double* d_out;
  long long* d_cyc;
  cudaMalloc(&d_out, sizeof(double) * sms * 1024);
  cudaMalloc(&d_cyc, sizeof(long long));
  printf("device %d: %d SMs, clock rate attribute %.3f GHz\n", dev, sms, ghz);
  printf("dependent-issue latency = cycles per DFMA at ILP 1 with 1 warp per sub-partition:\n");
  run<1>(sms, 1, d_out, d_cyc, ghz);
  printf("throughput:\n");
  for (int w : {1, 2, 4, 8}) {
    run<1>(sms, w, d_out, d_cyc, ghz);
    run<2>(sms, w, d_out, d_cyc, ghz);
    run<4>(sms, w, d_out, d_cyc, ghz);
    run<8>(sms, w, d_out, d_cyc, ghz);
  }
  cudaFree(d_out);
  cudaFree(d_cyc);
  return cudaDeviceSynchronize() == cudaSuccess ? 0 : 1;
}
