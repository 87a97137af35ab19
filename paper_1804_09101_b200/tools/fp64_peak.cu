// fp64_peak.cu — register-resident FP64 throughput microbenchmark for sm_100a (the derivative
// kernels report their fraction of an FP64 peak that is MEASURED here, not assumed).
//   mode 0: DFMA only (64 independent accumulators per warp-lane group, fma chains)
//   mode 1: DMMA only (mma.sync.aligned.m8n8k4.f64, 8 independent accumulator pairs)
//   mode 2: both interleaved in the same warp (are the two pipes independent?)
//   mode 3: half of the warps DFMA, half DMMA
// Build:  nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o fp64_peak fp64_peak.cu ; run: ./fp64_peak
#include <cuda_runtime.h>
#include <cstdio>

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <int MODE>
__global__ void __launch_bounds__(256) k_peak(double* out, int iters, double x) {
  double f[16], c[8][2];
  const double a = x + threadIdx.x * 1e-9, b = 1.0 - x;
#pragma unroll
  for (int i = 0; i < 16; ++i) f[i] = i * x;
#pragma unroll
  for (int i = 0; i < 8; ++i) c[i][0] = c[i][1] = i * x;
  const bool dm = (MODE == 1) || (MODE == 2) || (MODE == 3 && ((threadIdx.x >> 5) & 1));
  const bool df = (MODE == 0) || (MODE == 2) || (MODE == 3 && !((threadIdx.x >> 5) & 1));
  for (int it = 0; it < iters; ++it) {
    if (df) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int i = 0; i < 16; ++i) f[i] = fma(f[i], a, b);
    }
    if (dm) {
#pragma unroll
      for (int i = 0; i < 8; ++i) dmma(c[i][0], c[i][1], a, b);
    }
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += f[i];
#pragma unroll
  for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <int MODE>
double run(double* out, int sms, int ctas_per_sm, int iters, const char* name) {
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int grid = sms * ctas_per_sm;
  k_peak<MODE><<<grid, 256>>>(out, 16, 1e-3);
  cudaDeviceSynchronize();
  float best = 1e30f;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0);
    k_peak<MODE><<<grid, 256>>>(out, iters, 1e-3);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
  }
  // flop per thread-iteration: DFMA 64 fma = 128 flop per lane; DMMA 8 instr x 512 flop per warp = 128 flop per lane
  double per_lane = 0;
  if (MODE == 0 || MODE == 1) per_lane = 128; else if (MODE == 2) per_lane = 256; else per_lane = 128;
  const double flop = (double)grid * 256 * iters * per_lane;
  const double tf = flop / (best * 1e-3) / 1e12;
  printf("{\"mode\": \"%s\", \"ctas_per_sm\": %d, \"ms\": %.4f, \"tflops\": %.2f}\n", name, ctas_per_sm, best, tf);
  return tf;
}

int main() {
  int dev = 0, sms = 0; cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  double* out; cudaMalloc(&out, (size_t)sms * 8 * 256 * sizeof(double));
  const int iters = 20000;
  for (int c = 1; c <= 4; c *= 2) {
    run<0>(out, sms, c, iters, "dfma");
    run<1>(out, sms, c, iters, "dmma_m8n8k4");
    run<2>(out, sms, c, iters, "dfma+dmma same warp");
    run<3>(out, sms, c, iters, "dfma warps + dmma warps");
  }
  cudaFree(out);
  return 0;
}
