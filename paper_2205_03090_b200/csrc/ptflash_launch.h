// ptflash_launch.h -- host-side interface between the C ABI (ptflash_api.cu) and the per-NC kernel
// translation units (ptflash_nc.cu compiled once per component count with -DPTF_NC=<k>).
#pragma once
#include <cuda_runtime.h>
#include "ptflash_device.cuh"

namespace ptf {

// Component constants for the largest system; narrowed to Sys<NC> by the launcher.
struct SysHost {
  int nc;
  double u[16], v[16], wb[16], lnpc[16], wil[16], tc[16];
  double omk[256];  // row-major nc x nc
  int kij_zero;
};

template <int NC>
inline Sys<NC> narrow(const SysHost& h) {
  Sys<NC> s;
  for (int i = 0; i < NC; ++i) {
    s.u[i] = h.u[i]; s.v[i] = h.v[i]; s.wb[i] = h.wb[i]; s.lnpc[i] = h.lnpc[i]; s.wil[i] = h.wil[i]; s.tc[i] = h.tc[i];
    for (int j = 0; j < NC; ++j) s.omk[i * NC + j] = h.omk[i * NC + j];
  }
  s.kij_zero = h.kij_zero;
  return s;
}

// Stage counters of the staged engine (first bytes of the workspace; mirrored to the host after each call).
struct StageCounters {
  long long n_invalid, n_case1, n_case2, n_case3, n_stab, n_stab_newton, n_split, n_split_newton, n_two_phase;
  long long n_restart;                         // skip-stability hints that failed and were re-flashed cold (C21)
  // the columns of the paper's profiler (Table 4) that are not queue lengths; [0] vapour-like, [1] liquid-like
  long long n_stab_tr[2], n_stab_capped[2];    // stability trials that went on to the trust-region stage / hit an iteration cap
  long long n_split_capped;                    // phase splits that hit an iteration cap
  long long max_probe, max_stab_ss[2], max_stab_tr[2], max_split_ss, max_split_tr;   // largest iteration counts per stage
  long long queue_overflow;                    // 1 if a work queue ended longer than its array (cannot happen by construction; checked after every call)
};

// Launchers return the number of kernels launched (>= 0) or -1 on error.
//   launch_mono_<NC>   engine 0: one run-to-completion kernel (workspace unused)
//   launch_staged_<NC> engine 1: staged persistent kernels with work queues in `workspace`
typedef int (*launch_fn)(const SysHost&, const Opt&, const Io&, void* workspace, cudaStream_t);
// arguments of the batched Rachford-Rice kernel (ptflash_rr.cuh)
struct RrIo {
  int64_t N;
  const double *lnK, *z;          // [nc][N]
  double *theta, *x, *y, *dth;    // [N], [nc][N] x 3 (x, y, dth optional)
};
typedef int (*launch_rr_fn)(const RrIo&, cudaStream_t);
size_t staged_workspace_bytes(int nc, int64_t N);
int run_fp64_peak(int iters, double* flops_per_s, double* elapsed_ms, cudaStream_t st);
int run_math_probe(int fn, int64_t n, const double* x, double* y, cudaStream_t st);

#define PTF_DECL(NC) int launch_mono_##NC(const SysHost&, const Opt&, const Io&, void*, cudaStream_t); \
  int launch_staged_##NC(const SysHost&, const Opt&, const Io&, void*, cudaStream_t); \
  int launch_rr_##NC(const RrIo&, cudaStream_t);
PTF_DECL(2) PTF_DECL(3) PTF_DECL(4) PTF_DECL(5) PTF_DECL(6) PTF_DECL(7) PTF_DECL(8) PTF_DECL(9)
PTF_DECL(10) PTF_DECL(11) PTF_DECL(12) PTF_DECL(13) PTF_DECL(14) PTF_DECL(15) PTF_DECL(16)
#undef PTF_DECL

}  // namespace ptf
