// fp64_issue_mix_probe.cu — cost of non-FP64 instructions interleaved with DFMA:
// shows that the issue slot is held for both cycles of an FP64 instruction.  Stand-alone:
// nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o fp64_issue_mix_probe fp64_issue_mix_probe.cu
#include <cstdio>
#include <cuda_runtime.h>
__constant__ double kc[16] = {0.999, 1e-3, 0.998, 2e-3, 0.997, 3e-3, 0.996, 4e-3, 0.995, 5e-3, 0.994, 6e-3, 0.993, 7e-3, 0.992, 8e-3};
// MODE 0: DFMA regs; 1: DFMA with two constant-bank operands; 2: DMUL + DADD alternating; 3: DFMA + 1 FSEL-ish int op per DFMA
// 4: DFMA + 2 int ops per DFMA; 5: DFMA + LDS per 4 DFMA ; 6: DSETP+FSEL select (dmax) per DFMA
template <int MODE>
__global__ void k(long long iters, double a, double b, double *out, int sel) {
  __shared__ double sh[128];
  double x[8]; int y[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { x[i] = threadIdx.x * 1e-9 + i; y[i] = threadIdx.x + i; }
  sh[threadIdx.x] = a;
  for (long long n = 0; n < iters; ++n) {
#pragma unroll
    for (int u = 0; u < 8; ++u)
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        if (MODE == 0) x[i] = fma(x[i], a, b);
        if (MODE == 1) x[i] = fma(x[i], kc[2 * i], kc[2 * i + 1]);
        if (MODE == 2) x[i] = (u & 1) ? x[i] * a : x[i] + b;
        if (MODE == 3) { x[i] = fma(x[i], a, b); y[i] = (y[i] ^ sel) + (y[i] >> 3); }
        if (MODE == 4) { x[i] = fma(x[i], a, b); y[i] = (y[i] ^ sel) + (y[i] >> 3); y[i] = (y[i] & sel) | (y[i] << 2); }
        if (MODE == 5) { x[i] = fma(x[i], a, b); if ((i & 3) == 0) x[i] += sh[(threadIdx.x + y[i]) & 127]; }
        if (MODE == 6) { x[i] = fma(x[i], a, b); x[i] = x[i] > b ? x[i] : b; }
      }
  }
  double s = 0; int t = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) { s += x[i]; t += y[i]; }
  if (s == 12345.678 || t == 123456789) out[0] = s + t;
}
template <int MODE>
void run(int w) {
  int blocks = 148 * w; long long iters = 3000;
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  double *d; cudaMalloc(&d, 8);
  k<MODE><<<blocks, 128>>>(10, 0.999, 1e-3, d, 5);
  cudaEventRecord(e0);
  k<MODE><<<blocks, 128>>>(iters, 0.999, 1e-3, d, 5);
  cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  double cyc = ms * 1e-3 * 1.965e9 / ((double)iters * 64 * w);
  printf("mode %d warps/SMSP %d: %.2f cycles per loop-body item per SMSP\n", MODE, w, cyc);
}
int main() {
  for (int w : {3, 4}) { run<0>(w); run<1>(w); run<2>(w); run<3>(w); run<4>(w); run<5>(w); run<6>(w); }
}
