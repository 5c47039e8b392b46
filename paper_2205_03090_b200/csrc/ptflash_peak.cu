// ptflash_peak.cu -- FP64 roofline probe (independent DFMA chains on every SM) and workspace sizing.
#include "ptflash_launch.h"
#include "ptflash_staged.cuh"

namespace ptf {

// 8 independent DFMA chains per thread, `iters` trips: 16 flops per thread per trip.
__global__ void __launch_bounds__(256) dfma_peak_kernel(int iters, double seed, double* sink) {
  double a0 = seed + threadIdx.x, a1 = a0 + 1.0, a2 = a0 + 2.0, a3 = a0 + 3.0, a4 = a0 + 4.0, a5 = a0 + 5.0, a6 = a0 + 6.0, a7 = a0 + 7.0;
  const double m = 0.999999, c = 1.0e-9;
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
      a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
  }
  const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
  if (s == 12345.678) sink[0] = s;  // never true; keeps the chains alive
}

int run_fp64_peak(int iters, double* flops_per_s, double* elapsed_ms, cudaStream_t st) {
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return -1;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
  double* sink = nullptr;
  if (cudaMalloc(&sink, sizeof(double)) != cudaSuccess) return -1;
  const int threads = 256, blocks = sms * 8;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  dfma_peak_kernel<<<blocks, threads, 0, st>>>(iters / 8 + 1, 1.0, sink);  // warm-up
  cudaEventRecord(e0, st);
  dfma_peak_kernel<<<blocks, threads, 0, st>>>(iters, 1.0, sink);
  cudaEventRecord(e1, st);
  int rc = 0;
  if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = -1;
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  if (rc) return rc;
  const double flops = (double)blocks * threads * (double)iters * 8.0 * 8.0 * 2.0;
  *flops_per_s = flops / (ms * 1.0e-3);
  *elapsed_ms = ms;
  return 0;
}

// Element-wise evaluation of one lean math routine of ptflash_math.cuh (diagnostic entry ptflash_math_probe).
__global__ void __launch_bounds__(256) math_probe_kernel(int fn, int64_t n, const double* __restrict__ x, double* __restrict__ y) {
  __shared__ double s_exp[PTF_EXP_TAB];
  exp_tab_init(s_exp);
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const double v = x[i];
    double r;
    switch (fn) {
      case 0: r = exp_fast(v); break;
      case 1: r = exp_tab(v, s_exp); break;
      case 2: r = log_fast(v); break;
      case 3: r = log1p_fast(v); break;
      case 4: r = rcp_fast(v); break;
      case 5: r = rsqrt_fast(v); break;
      case 6: r = sqrt_fast(v); break;
      case 7: r = div_fast(1.0, v); break;
      case 8: r = rcp_nr1(v); break;
      default: r = v; break;
    }
    y[i] = r;
  }
}

int run_math_probe(int fn, int64_t n, const double* x, double* y, cudaStream_t st) {
  if (n <= 0) return 0;
  const int64_t blocks = (n + 255) / 256;
  math_probe_kernel<<<(unsigned)(blocks < 4096 ? blocks : 4096), 256, 0, st>>>(fn, n, x, y);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

size_t staged_workspace_bytes(int nc, int64_t N) {
  return carve_workspace(nc, N, nullptr, nullptr);
}

}  // namespace ptf
