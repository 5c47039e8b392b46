// ptflash_nc.cu -- kernel instantiations for ONE component count; compiled once per NC with -DPTF_NC=<k>
// (nvcc -gencode arch=compute_100a,code=sm_100a), so the 15 variants build in parallel.
#include "ptflash_launch.h"
#include "ptflash_flash.cuh"
#include "ptflash_staged.cuh"
#include "ptflash_stage2.cuh"
#include "ptflash_rr.cuh"

#ifndef PTF_NC
#error "compile with -DPTF_NC=<2..16>"
#endif

#define PTF_CAT2(a, b) a##b
#define PTF_CAT(a, b) PTF_CAT2(a, b)

namespace ptf {

#ifdef PTF_STUB
// development build that left this component count out
int PTF_CAT(launch_mono_, PTF_NC)(const SysHost&, const Opt&, const Io&, void*, cudaStream_t) { return -1; }
int PTF_CAT(launch_staged_, PTF_NC)(const SysHost&, const Opt&, const Io&, void*, cudaStream_t) { return -1; }
int PTF_CAT(launch_rr_, PTF_NC)(const RrIo&, cudaStream_t) { return -1; }
}  // namespace ptf
#else

int PTF_CAT(launch_mono_, PTF_NC)(const SysHost& hs, const Opt& o, const Io& io, void*, cudaStream_t st) {
  constexpr int NC = PTF_NC;
  const Sys<NC> s = narrow<NC>(hs);
  const int threads = 128;
  const int64_t blocks = (io.N + threads - 1) / threads;
  flash_mono_kernel<NC><<<(unsigned)blocks, threads, 0, st>>>(s, o, io);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int PTF_CAT(launch_staged_, PTF_NC)(const SysHost& hs, const Opt& o, const Io& io, void* ws, cudaStream_t st) {
  // every component count (2..16) and both modes (trust-region Newton / pure successive substitution) run the
  // register-resident stage kernels; for nc >= 13 the Newton CTAs are limited by shared memory (one per SM at nc = 16)
  return launch_stage2<PTF_NC>(hs, o, io, ws, st);
}

int PTF_CAT(launch_rr_, PTF_NC)(const RrIo& io, cudaStream_t st) { return launch_rr<PTF_NC>(io, st); }

}  // namespace ptf
#endif
