// FP64 peak probes: register-resident DFMA and DMMA (mma.sync m8n8k4 f64) issue loops.
// MEASURED_PEAKS.json carries only HBM and bf16 figures, so bench.py measures the FP64 roofline
// denominator with these (sustained over `seconds`), as SURVEY.md 8(d) requires.
#include <cuda_runtime.h>

#include "exx_internal.h"

namespace {

__global__ void __launch_bounds__(256) k_dfma(double* out, int iters, double a, double b) {
  double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6,
         x7 = x0 + 7;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
}

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(256) k_dmma(double* out, int iters, double a, double b) {
  double c[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) c[i] = threadIdx.x + i;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
#pragma unroll
      for (int t = 0; t < 8; ++t) dmma884(c[2 * t], c[2 * t + 1], a, b);
    }
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace

extern "C" exx_status exx_probe_fp64_peak(int kind, int device, double seconds, double* tflops) {
  if (!tflops || (kind != 0 && kind != 1) || !(seconds > 0.0) || seconds > 30.0) return EXX_ERR_INVALID_ARG;
  exx::DeviceScope dev_scope(device);  // the caller's current device is restored on return
  if (!dev_scope.ok()) return EXX_ERR_CUDA;
  int sms = 0;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) return EXX_ERR_CUDA;
  const int threads = 256, blocks = sms * 8;
  double* out = nullptr;
  if (cudaMalloc(&out, sizeof(double) * threads * blocks) != cudaSuccess) return EXX_ERR_ALLOC;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int iters = 4096;
  // flops per launch
  const double per_thread = kind == 0 ? 2.0 * 64.0 * iters           // 64 DFMA per iteration
                                      : 512.0 * 32.0 * iters / 32.0;  // 32 DMMA (512 flop) per warp-iteration
  const double flops = per_thread * threads * blocks;
  auto launch = [&]() {
    if (kind == 0) k_dfma<<<blocks, threads>>>(out, iters, 0.999999, 1e-9);
    else k_dmma<<<blocks, threads>>>(out, iters, 0.5, 0.25);
  };
  for (int w = 0; w < 3; ++w) launch();
  cudaDeviceSynchronize();
  double best_sustained = 0.0, elapsed = 0.0;
  int total = 0;
  cudaEventRecord(e0);
  while (elapsed < seconds * 1e3) {
    for (int r = 0; r < 8; ++r) launch();
    total += 8;
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    elapsed = ms;
  }
  best_sustained = flops * total / (elapsed * 1e-3) / 1e12;
  cudaError_t err = cudaGetLastError();
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(out);
  if (err != cudaSuccess) return EXX_ERR_CUDA;
  *tflops = best_sustained;
  return EXX_OK;
}
