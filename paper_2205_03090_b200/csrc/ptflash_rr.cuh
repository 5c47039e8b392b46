// ptflash_rr.cuh -- batched Rachford-Rice solve with its derivative (ptflash_rachford_rice of include/ptflash.h).
//
// What the paper's initializer training calls for every sample: given z and an estimate of K, solve
// f_RR(theta, K) = sum_i (K_i - 1) z_i / (1 + (K_i - 1) theta) = 0 (eq. 7; App. C) and return
// d theta / d K by the implicit-function theorem (eq. 13) instead of differentiating through the iterations:
//     d theta / d K_i = -[d f / d theta]^-1 d f / d K_i,   d f / d K_i = z_i r_i^2,   d f / d theta = -sum_j (K_j - 1)^2 z_j r_j^2,
// with r_i = 1 / (1 + (K_i - 1) theta).  One thread per mixture, everything in registers; HBM bound (the solve is ~5 Newton
// steps of nc divisions against 8 (4 nc + 1) bytes of traffic per mixture).
#pragma once
#include "ptflash_fast.cuh"
#include "ptflash_staged.cuh"
#include "ptflash_launch.h"

namespace ptf {

template <int NC>
__global__ void __launch_bounds__(128) k_rr(const __grid_constant__ RrIo io) {
  const double nan = __longlong_as_double(0x7ff8000000000000LL);
  const int64_t N = io.N;
  PTF_GRID_STRIDE(n, N) {
    double z[NC], K[NC], x[NC], y[NC];
    double sz = 0.0;
    bool ok = true;
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      z[i] = io.z[(int64_t)i * N + n];
      const double lk = io.lnK[(int64_t)i * N + n];
      ok = ok && (z[i] >= 0.0) && (fabs(z[i]) <= 1.0e300) && (fabs(lk) <= 700.0);   // NaN fails every comparison
      K[i] = exp_fast(ok ? lk : 0.0);
      sz += z[i];
    }
    ok = ok && (sz > 0.0);
    const double isz = 1.0 / sz;
#pragma unroll
    for (int i = 0; i < NC; ++i) z[i] *= isz;
    double theta = -1.0e300;   // cold start
    ok = ok && rr_fast<NC>(K, z, theta, x, y);
    io.theta[n] = ok ? theta : nan;
    double r[NC], dfdth = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      const double km1 = (z[i] > 0.0) ? K[i] - 1.0 : 0.0;
      r[i] = 1.0 / fma(km1, theta, 1.0);
      dfdth = fma(-(km1 * r[i]) * (km1 * r[i]), z[i], dfdth);
    }
    const double inv = -1.0 / dfdth;
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      if (io.x) io.x[(int64_t)i * N + n] = ok ? x[i] : nan;
      if (io.y) io.y[(int64_t)i * N + n] = ok ? y[i] : nan;
      if (io.dth) io.dth[(int64_t)i * N + n] = ok ? z[i] * r[i] * r[i] * inv : nan;
    }
  }
}

template <int NC>
int launch_rr(const RrIo& io, cudaStream_t st) {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int threads = 128;
  const int64_t need = (io.N + threads - 1) / threads;
  const int64_t cap = (int64_t)sms * 16;
  k_rr<NC><<<(unsigned)(need < cap ? (need > 0 ? need : 1) : cap), threads, 0, st>>>(io);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace ptf
