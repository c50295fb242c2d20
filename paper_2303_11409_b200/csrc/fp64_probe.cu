// fp64_probe.cu — measured FP64 throughput of this GPU (the denominator of the a3 / a2 roofline):
// register-resident chains of DFMA and of DMMA.8x8x4 (mma.sync.m8n8k4.f64), 8 independent accumulators per thread /
// warp, every SM filled.  Prints one JSON line {"dfma_tflops": ..., "dmma_tflops": ..., "sm_clock_mhz": ...}.
// Built by paper_2303_11409_b200.build next to libu1mps.so; bench.py runs it and reports the numbers beside the
// derived peak (148 SMs x 64 FMA/clk x 2 x clock).  Not part of the update path.
#include <cstdio>
#include <cuda_runtime.h>

__global__ void dfma_chain(double* out, int iters, double a, double b) {
  double x[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) x[i] = threadIdx.x * 1e-9 + i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = fma(x[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += x[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void dmma_chain(double* out, int iters, double a, double b) {
  double c[8][2];
#pragma unroll
  for (int i = 0; i < 8; ++i) { c[i][0] = threadIdx.x * 1e-9 + i; c[i][1] = 0.5 * i; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                   : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

int main() {
  int dev = 0, sms = 0, khz = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { printf("{\"error\": \"no CUDA device\"}\n"); return 1; }
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
  const int threads = 256, blocks = sms * 8, iters = 1 << 14;
  double* out;
  cudaMalloc(&out, sizeof(double) * threads * blocks);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  double res[2] = {0.0, 0.0};
  for (int k = 0; k < 2; ++k) {
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {   // first repetition warms up
      cudaEventRecord(e0);
      if (k == 0) dfma_chain<<<blocks, threads>>>(out, iters, 1.0000001, 1e-9);
      else dmma_chain<<<blocks, threads>>>(out, iters, 1e-3, 1e-3);
      cudaEventRecord(e1);
      cudaEventSynchronize(e1);
      float ms = 0.f;
      cudaEventElapsedTime(&ms, e0, e1);
      if (rep > 0 && ms < best) best = ms;
    }
    // flops: DFMA 2 per thread-instruction; DMMA 8x8x4 = 2 * 256 per warp-instruction
    const double per_iter = k == 0 ? 8.0 * 2.0 * threads * blocks : 8.0 * 512.0 * (threads / 32) * blocks;
    res[k] = per_iter * iters / (best * 1e-3) / 1e12;
  }
  if (cudaGetLastError() != cudaSuccess) { printf("{\"error\": \"CUDA error\"}\n"); return 1; }
  printf("{\"dfma_tflops\": %.3f, \"dmma_tflops\": %.3f, \"sms\": %d, \"sm_clock_mhz\": %.0f}\n", res[0], res[1], sms, khz / 1000.0);
  cudaFree(out);
  return 0;
}
