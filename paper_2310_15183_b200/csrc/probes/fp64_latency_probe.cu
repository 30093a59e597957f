// fp64_latency_probe.cu — DFMA throughput against warps per SM sub-partition and independent chains per
// thread.  Stand-alone: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o fp64_latency_probe fp64_latency_probe.cu
#include <cstdio>
#include <cuda_runtime.h>
template <int ILP>
__global__ void k(long long iters, double a, double b, double *out) {
  double x[ILP];
#pragma unroll
  for (int i = 0; i < ILP; ++i) x[i] = threadIdx.x * 1e-9 + i;
  for (long long n = 0; n < iters; ++n) {
#pragma unroll
    for (int u = 0; u < 16; ++u)
#pragma unroll
      for (int i = 0; i < ILP; ++i) x[i] = fma(x[i], a, b);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < ILP; ++i) s += x[i];
  if (s == 12345.678) out[0] = s;
}
template <int ILP>
void run(int warps_per_smsp) {
  int blocks = 148 * warps_per_smsp;  // 128 threads = 4 warps = 1 warp per SMSP per block
  long long iters = 20000 / ILP;
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  double *d; cudaMalloc(&d, 8);
  k<ILP><<<blocks, 128>>>(10, 0.999, 1e-3, d);
  cudaEventRecord(e0);
  k<ILP><<<blocks, 128>>>(iters, 0.999, 1e-3, d);
  cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  double fma_total = (double)blocks * 128 * iters * 16 * ILP;
  double tf = 2 * fma_total / (ms * 1e-3) / 1e12;
  // cycles per warp-instruction per SMSP
  double cyc = ms * 1e-3 * 1.965e9 / ((double)iters * 16 * ILP * warps_per_smsp);
  printf("warps/SMSP %d ILP %d: %.2f TFLOP/s (%.1f%% of 37.2), %.2f cycles per warp-DFMA per SMSP\n", warps_per_smsp, ILP, tf, 100 * tf / 37.2, cyc);
}
int main() {
  for (int w : {1, 2, 3, 4, 6, 8}) { run<1>(w); run<2>(w); run<4>(w); run<8>(w); }
  return 0;
}
