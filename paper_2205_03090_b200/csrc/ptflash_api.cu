// ptflash_api.cu -- the C ABI of libptflash (include/ptflash.h): handle management, argument validation,
// workspace ownership, option table, host-buffer variant and the FP64 roofline probe.  No torch types,
// no CPU fallback: every numerical step runs in the kernels of ptflash_nc.cu.
#include <cmath>
#include <cstddef>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>

#include "../../include/ptflash.h"
#include "ptflash_launch.h"

namespace {

#define PTF_MAX_HOST_CHUNKS 8
#define PTF_HOST_DEPTH PTFLASH_HOST_DEPTH
thread_local std::string g_err;
void set_err(const std::string& s) { g_err = s; }
bool cuda_ok(cudaError_t e, const char* what) {
  if (e == cudaSuccess) return true;
  set_err(std::string(what) + ": " + cudaGetErrorString(e));
  return false;
}

const double kDefaultOpts[PTFLASH_NUM_OPTS] = {1e-10, 1e-12, 1e-7, 1e-8, 1e-6, 1e-9, 3, 9, 60, 9, 60, 1, 100000, 1, 0, 1e-6, 12, 1e-5, 0, 8, 0, 15, 0, 0};

}  // namespace

struct ptflash_handle_s {
  int device;
  ptf::SysHost sys;
  double opts[PTFLASH_NUM_OPTS];
  cudaStream_t last_stream;   // stream of the last FLASH call: what ptflash_get_stats / ptflash_get_stage_ms wait for
  bool used;
  cudaStream_t rr_stream;     // stream of the last ptflash_rachford_rice call (it has no counters: only ptflash_destroy waits for it)
  bool rr_used;
  // workspace of the staged engine (device) and its size
  void* ws;
  size_t ws_bytes;
  // staging buffers of ptflash_flash_host (device)
  void* stage;
  size_t stage_bytes;
  // host mirror of the stage counters of the last call
  ptf::StageCounters* counters_host;  // pinned
  int64_t last_N;
  int last_launches;
  // stage profiling (PTFLASH_OPT_STAGE_PROFILE): events recorded between the stage kernels of the last call
  cudaEvent_t events[PTF_MAX_STAGE_EVENTS];
  bool events_made;
  int n_events;
  // second stream + fork/join events of the staged engine (created on first use)
  cudaStream_t aux_stream, aux2_stream;
  cudaEvent_t ev_fork, ev_join, ev_c0, ev_c1, ev_cjoin, ev_probe;
  bool aux_made;
  int cta_cache[4];   // resident CTAs per SM of the persistent kernels on this handle's device (0 = not queried yet)
  // ptflash_flash_host pipeline: child handles (same component system, own workspace / streams / counters), one per chunk
  // in flight, each with a stream of its own on which its chunk's H2D copies, kernels and D2H copies are ordered
  ptflash_handle_s* child[PTF_MAX_HOST_CHUNKS];
  cudaStream_t child_stream[PTF_MAX_HOST_CHUNKS];
  cudaEvent_t child_done[PTF_MAX_HOST_CHUNKS];
  cudaEvent_t host_begin;
  int n_child;
  bool host_stats;       // the last call was a chunked ptflash_flash_host: statistics are the sum over the children
  int host_chunks_used;
  // ptflash_flash_host_async: PTFLASH_HOST_DEPTH batches in flight, each on a child handle with a stream of its own
  ptflash_handle_s* aslot[PTF_HOST_DEPTH];
  cudaStream_t astream[PTF_HOST_DEPTH];
  cudaEvent_t adone[PTF_HOST_DEPTH];
  int n_aslot;
  long long a_submitted;   // batches submitted so far
  int a_last;              // slot of the most recent batch (-1: the last call was not an async one)
};

namespace {

// Makes the handle's device current for the duration of a call and restores the caller's device afterwards
// (a handle is bound to the device that was current in ptflash_create).
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = (cudaSetDevice(dev) == cudaSuccess);
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

ptf::Opt make_opt(const double* o) {
  ptf::Opt r;
  r.tol_ss = o[PTFLASH_OPT_TOL_SS];
  r.tol_newton_g = o[PTFLASH_OPT_TOL_NEWTON_G];
  r.tol_newton_step = o[PTFLASH_OPT_TOL_NEWTON_STEP];
  r.tol_newton_step_stab = o[PTFLASH_OPT_TOL_NEWTON_STEP_STAB];
  r.probe_margin = o[PTFLASH_OPT_PROBE_MARGIN];
  r.trivial_tol = o[PTFLASH_OPT_TRIVIAL_TOL];
  r.triv_lo = std::exp(-r.trivial_tol);
  r.triv_hi = std::exp(r.trivial_tol);
  r.band = o[PTFLASH_OPT_BAND];
  r.probe_iters = (int)o[PTFLASH_OPT_PROBE_ITERS];
  r.stab_ss_iters = (int)o[PTFLASH_OPT_STAB_SS_ITERS];
  r.stab_tr_iters = (int)o[PTFLASH_OPT_STAB_TR_ITERS];
  r.split_ss_iters = (int)o[PTFLASH_OPT_SPLIT_SS_ITERS];
  r.split_tr_iters = (int)o[PTFLASH_OPT_SPLIT_TR_ITERS];
  r.use_newton = (int)o[PTFLASH_OPT_USE_NEWTON];
  r.ss_cap = (int)o[PTFLASH_OPT_SS_CAP];
  r.hint_ss_cap = (int)o[PTFLASH_OPT_HINT_SS_CAP];
  r.split_trivial_tol = o[PTFLASH_OPT_SPLIT_TRIVIAL_TOL];
  r.stability_only = (int)o[PTFLASH_OPT_STABILITY_ONLY];
  r.hint_eta_search = (int)o[PTFLASH_OPT_HINT_ETA_SEARCH];
  r.hint_tr_cap = (int)o[PTFLASH_OPT_HINT_TR_CAP];
  r.early_split_ss = (int)o[PTFLASH_OPT_EARLY_SPLIT_SS];
  r.prof_events = nullptr;
  r.prof_count = nullptr;
  r.aux_stream = r.ev_fork = r.ev_join = nullptr;
  r.aux2_stream = r.ev_c0 = r.ev_c1 = r.ev_cjoin = r.ev_probe = nullptr;
  r.cta_cache = nullptr;
  return r;
}

ptf::launch_rr_fn pick_rr(int nc) {
  using namespace ptf;
#define PTF_CASE(NC) case NC: return launch_rr_##NC;
  switch (nc) {
    PTF_CASE(2) PTF_CASE(3) PTF_CASE(4) PTF_CASE(5) PTF_CASE(6) PTF_CASE(7) PTF_CASE(8) PTF_CASE(9)
    PTF_CASE(10) PTF_CASE(11) PTF_CASE(12) PTF_CASE(13) PTF_CASE(14) PTF_CASE(15) PTF_CASE(16)
  }
#undef PTF_CASE
  return nullptr;
}

ptf::launch_fn pick_launcher(int nc, int engine) {
  using namespace ptf;
#define PTF_CASE(NC) case NC: return engine ? launch_staged_##NC : launch_mono_##NC;
  switch (nc) {
    PTF_CASE(2) PTF_CASE(3) PTF_CASE(4) PTF_CASE(5) PTF_CASE(6) PTF_CASE(7) PTF_CASE(8) PTF_CASE(9)
    PTF_CASE(10) PTF_CASE(11) PTF_CASE(12) PTF_CASE(13) PTF_CASE(14) PTF_CASE(15) PTF_CASE(16)
  }
#undef PTF_CASE
  return nullptr;
}

bool ensure(void** buf, size_t* have, size_t need, cudaStream_t st, const char* what) {
  if (*have >= need) return true;
  // growth: wait for work that may still use the old buffer, then reallocate
  if (!cuda_ok(cudaStreamSynchronize(st), "cudaStreamSynchronize")) return false;
  if (*buf) cudaFree(*buf);
  *buf = nullptr;
  *have = 0;
  if (!cuda_ok(cudaMalloc(buf, need), what)) return false;
  *have = need;
  return true;
}

// Strided copy of `rows` rows of `width` bytes: the component rows of one chunk's slice of an SoA array ([nc][N] on the host,
// [nc][Nc] on the device).  One cudaMemcpy2DAsync -- unless a pitch is beyond what the 2D copy accepts (cudaDevAttrMaxPitch,
// 2^31 - 1 bytes, i.e. host arrays of N >= 2^28 mixtures: "invalid pitch") or the caller asks for it
// (PTFLASH_OPT_HOST_ROW_COPIES): then one cudaMemcpyAsync per row, at most 16 of them.
bool copy_rows(void* dst, size_t dpitch, const void* src, size_t spitch, size_t width, int rows, cudaMemcpyKind kind,
               cudaStream_t st, size_t max_pitch, bool by_rows, const char* what) {
  if (!by_rows && dpitch <= max_pitch && spitch <= max_pitch)
    return cuda_ok(cudaMemcpy2DAsync(dst, dpitch, src, spitch, width, (size_t)rows, kind, st), what);
  for (int r = 0; r < rows; ++r)
    if (!cuda_ok(cudaMemcpyAsync((char*)dst + (size_t)r * dpitch, (const char*)src + (size_t)r * spitch, width, kind, st), what)) return false;
  return true;
}

// A child handle of the host-buffer calls: same component system, its own workspace and counters.  nullptr on failure.
ptflash_handle_s* make_child(const ptflash_handle_s* h) {
  ptflash_handle_s* k = new ptflash_handle_s();
  std::memset(k, 0, sizeof(*k));
  k->device = h->device;
  k->sys = h->sys;
  k->a_last = -1;
  if (!cuda_ok(cudaMallocHost((void**)&k->counters_host, sizeof(ptf::StageCounters)), "cudaMallocHost")) { delete k; return nullptr; }
  std::memset(k->counters_host, 0, sizeof(ptf::StageCounters));
  return k;
}

}  // namespace

extern "C" {

const char* ptflash_last_error(void) { return g_err.c_str(); }
const char* ptflash_version(void) { return "ptflash-b200 0.1 (sm_100a, fp64)"; }

ptflash_handle_t ptflash_create(int nc, const double* Tc, const double* Pc, const double* omega, const double* kij) {
  g_err.clear();
  if (nc < 2 || nc > PTFLASH_MAX_NC) { set_err("ptflash_create: nc must be in [2, 16]"); return nullptr; }
  if (!Tc || !Pc || !omega) { set_err("ptflash_create: null Tc/Pc/omega"); return nullptr; }
  for (int i = 0; i < nc; ++i) {
    if (!std::isfinite(Tc[i]) || !std::isfinite(Pc[i]) || !std::isfinite(omega[i]) || Tc[i] <= 0.0 || Pc[i] <= 0.0) {
      set_err("ptflash_create: Tc and Pc must be finite and positive, omega finite");
      return nullptr;
    }
  }
  if (kij) {
    for (int i = 0; i < nc; ++i) {
      if (kij[i * nc + i] != 0.0) { set_err("ptflash_create: kij diagonal must be zero"); return nullptr; }
      for (int j = 0; j < nc; ++j) {
        if (!std::isfinite(kij[i * nc + j]) || kij[i * nc + j] != kij[j * nc + i]) {
          set_err("ptflash_create: kij must be finite and symmetric");
          return nullptr;
        }
      }
    }
  }
  int dev = 0;
  if (!cuda_ok(cudaGetDevice(&dev), "cudaGetDevice")) return nullptr;
  ptflash_handle_s* h = new ptflash_handle_s();
  std::memset(h, 0, sizeof(*h));
  h->device = dev;
  ptf::SysHost& s = h->sys;
  s.nc = nc;
  s.kij_zero = 1;
  for (int i = 0; i < nc; ++i) {
    // A.2d-g PAPER.md:420-427 folded into per-component constants (see ptflash_device.cuh)
    const double m = 0.480 + 1.574 * omega[i] - 0.176 * omega[i] * omega[i];
    const double k = std::sqrt(0.42748 / Pc[i]);
    s.u[i] = k * Tc[i] * (1.0 + m);
    s.v[i] = k * std::sqrt(Tc[i]) * m;
    s.wb[i] = 0.08664 * Tc[i] / Pc[i];
    s.lnpc[i] = std::log(Pc[i]);
    s.wil[i] = 5.373 * (1.0 + omega[i]);  // eq. 6
    s.tc[i] = Tc[i];
    for (int j = 0; j < nc; ++j) {
      const double kk = kij ? kij[i * nc + j] : 0.0;
      s.omk[i * nc + j] = 1.0 - kk;
      if (kk != 0.0) s.kij_zero = 0;
    }
  }
  std::memcpy(h->opts, kDefaultOpts, sizeof(kDefaultOpts));
  h->a_last = -1;
  if (!cuda_ok(cudaMallocHost((void**)&h->counters_host, sizeof(ptf::StageCounters)), "cudaMallocHost")) { delete h; return nullptr; }
  std::memset(h->counters_host, 0, sizeof(ptf::StageCounters));
  return h;
}

int ptflash_destroy(ptflash_handle_t h) {
  if (!h) return PTFLASH_OK;
  int rc = PTFLASH_OK;
  DeviceGuard guard(h->device);
  if (h->used && !cuda_ok(cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize")) rc = PTFLASH_ECUDA;
  if (h->rr_used && !cuda_ok(cudaStreamSynchronize(h->rr_stream), "cudaStreamSynchronize")) rc = PTFLASH_ECUDA;
  if (h->ws) cudaFree(h->ws);
  if (h->stage) cudaFree(h->stage);
  if (h->counters_host) cudaFreeHost(h->counters_host);
  if (h->events_made)
    for (int i = 0; i < PTF_MAX_STAGE_EVENTS; ++i) cudaEventDestroy(h->events[i]);
  if (h->aux_made) {
    cudaStreamDestroy(h->aux_stream); cudaStreamDestroy(h->aux2_stream);
    cudaEventDestroy(h->ev_fork); cudaEventDestroy(h->ev_join);
    cudaEventDestroy(h->ev_c0); cudaEventDestroy(h->ev_c1); cudaEventDestroy(h->ev_cjoin); cudaEventDestroy(h->ev_probe);
  }
  for (int c = 0; c < h->n_child; ++c) {
    cudaStreamSynchronize(h->child_stream[c]);
    ptflash_destroy(h->child[c]);
    cudaStreamDestroy(h->child_stream[c]);
    cudaEventDestroy(h->child_done[c]);
  }
  if (h->n_child) cudaEventDestroy(h->host_begin);
  for (int c = 0; c < h->n_aslot; ++c) {
    cudaStreamSynchronize(h->astream[c]);
    ptflash_destroy(h->aslot[c]);
    cudaStreamDestroy(h->astream[c]);
    cudaEventDestroy(h->adone[c]);
  }
  delete h;
  return rc;
}

int ptflash_set_option(ptflash_handle_t h, int key, double value) {
  if (!h || key < 0 || key >= PTFLASH_NUM_OPTS || !std::isfinite(value)) { set_err("ptflash_set_option: bad handle/key/value"); return PTFLASH_EINVAL; }
  bool ok = true;
  switch (key) {
    case PTFLASH_OPT_TOL_SS: case PTFLASH_OPT_TOL_NEWTON_G: case PTFLASH_OPT_TOL_NEWTON_STEP: case PTFLASH_OPT_TOL_NEWTON_STEP_STAB:
    case PTFLASH_OPT_TRIVIAL_TOL: case PTFLASH_OPT_SPLIT_TRIVIAL_TOL:
      ok = value > 0.0 && value < 1.0; break;                      // tolerances
    case PTFLASH_OPT_PROBE_MARGIN: case PTFLASH_OPT_BAND:
      ok = value >= 0.0 && value < 1.0; break;
    case PTFLASH_OPT_PROBE_ITERS: case PTFLASH_OPT_STAB_SS_ITERS: case PTFLASH_OPT_STAB_TR_ITERS: case PTFLASH_OPT_SPLIT_SS_ITERS:
    case PTFLASH_OPT_SPLIT_TR_ITERS: case PTFLASH_OPT_SS_CAP: case PTFLASH_OPT_HINT_SS_CAP: case PTFLASH_OPT_HINT_TR_CAP:
      ok = value >= 0.0 && value <= 1.0e9 && value == std::floor(value); break;   // iteration counts
    case PTFLASH_OPT_USE_NEWTON: case PTFLASH_OPT_ENGINE: case PTFLASH_OPT_STAGE_PROFILE: case PTFLASH_OPT_STABILITY_ONLY:
    case PTFLASH_OPT_HINT_ETA_SEARCH: case PTFLASH_OPT_EARLY_SPLIT_SS: case PTFLASH_OPT_HOST_ROW_COPIES:
      ok = value == 0.0 || value == 1.0; break;                   // switches
    case PTFLASH_OPT_HOST_CHUNKS:
      ok = value >= 1.0 && value <= (double)PTF_MAX_HOST_CHUNKS && value == std::floor(value); break;
    default: break;
  }
  if (!ok) { set_err("ptflash_set_option: value out of range for this option"); return PTFLASH_EINVAL; }
  h->opts[key] = value;
  return PTFLASH_OK;
}
int ptflash_get_option(ptflash_handle_t h, int key, double* value) {
  if (!h || !value || key < 0 || key >= PTFLASH_NUM_OPTS) { set_err("ptflash_get_option: bad handle/key"); return PTFLASH_EINVAL; }
  *value = h->opts[key];
  return PTFLASH_OK;
}

int ptflash_flash_ex(ptflash_handle_t h, const ptflash_io_t* io, void* stream) {
  g_err.clear();
  if (!h || !io) { set_err("ptflash_flash: null handle or io"); return PTFLASH_EINVAL; }
  if (io->N < 0) { set_err("ptflash_flash: N < 0"); return PTFLASH_EINVAL; }
  if (io->N == 0) return PTFLASH_OK;
  // the stage queues hold mixture ids (and 2 n + start for the stability trials) as 32-bit integers
  if (io->N > PTFLASH_MAX_N) { set_err("ptflash_flash: N exceeds PTFLASH_MAX_N (2^30 - 1); split the batch"); return PTFLASH_EINVAL; }
  if (!io->z || !io->P || !io->T || !io->out_beta || !io->out_x || !io->out_y || !io->out_phase) {
    set_err("ptflash_flash: null required pointer");
    return PTFLASH_EINVAL;
  }
  DeviceGuard guard(h->device);
  cudaStream_t st = (cudaStream_t)stream;
  const int engine = (int)h->opts[PTFLASH_OPT_ENGINE];
  ptf::launch_fn fn = pick_launcher(h->sys.nc, engine);
  if (!fn) { set_err("ptflash_flash: no kernel for this nc"); return PTFLASH_EINVAL; }
  ptf::Io d;
  d.N = io->N;
  d.z = io->z; d.P = io->P; d.T = io->T;
  d.lnK0 = io->lnK0;
  d.flags = io->lnK0 ? io->flags : nullptr;
  d.beta = io->out_beta; d.x = io->out_x; d.y = io->out_y;
  d.phase = io->out_phase; d.iters = io->out_iters;
  d.tpd_min = io->out_tpd_min; d.lnK = io->out_lnK; d.status = io->out_status; d.stab_iters = io->out_stab_iters;
  d.dbeta_dK = io->out_dbeta_dK;
  if (engine) {
    const size_t need = ptf::staged_workspace_bytes(h->sys.nc, io->N);
    if (!ensure(&h->ws, &h->ws_bytes, need, st, "cudaMalloc(workspace)")) return PTFLASH_ECUDA;
  }
  ptf::Opt o = make_opt(h->opts);
  o.cta_cache = h->cta_cache;
  h->n_events = 0;
  if ((int)h->opts[PTFLASH_OPT_STAGE_PROFILE] && engine) {
    if (!h->events_made) {
      for (int i = 0; i < PTF_MAX_STAGE_EVENTS; ++i)
        if (!cuda_ok(cudaEventCreate(&h->events[i]), "cudaEventCreate")) return PTFLASH_ECUDA;
      h->events_made = true;
    }
    o.prof_events = h->events;
    o.prof_count = &h->n_events;
  } else if (engine) {
    if (!h->aux_made) {
      if (!cuda_ok(cudaStreamCreateWithFlags(&h->aux_stream, cudaStreamNonBlocking), "cudaStreamCreate")) return PTFLASH_ECUDA;
      if (!cuda_ok(cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming), "cudaEventCreate")) return PTFLASH_ECUDA;
      if (!cuda_ok(cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming), "cudaEventCreate")) return PTFLASH_ECUDA;
      // the crawler stream has the highest priority: its few CTAs must be placed BEFORE the persistent Newton CTAs of the
      // split fill every SM, else a crawler's serial chain (hundreds of iterations) starts only when those retire
      int pr_least = 0, pr_greatest = 0;
      cudaDeviceGetStreamPriorityRange(&pr_least, &pr_greatest);
      if (!cuda_ok(cudaStreamCreateWithPriority(&h->aux2_stream, cudaStreamNonBlocking, pr_greatest), "cudaStreamCreate")) return PTFLASH_ECUDA;
      if (!cuda_ok(cudaEventCreateWithFlags(&h->ev_c0, cudaEventDisableTiming), "cudaEventCreate")) return PTFLASH_ECUDA;
      if (!cuda_ok(cudaEventCreateWithFlags(&h->ev_c1, cudaEventDisableTiming), "cudaEventCreate")) return PTFLASH_ECUDA;
      if (!cuda_ok(cudaEventCreateWithFlags(&h->ev_cjoin, cudaEventDisableTiming), "cudaEventCreate")) return PTFLASH_ECUDA;
      if (!cuda_ok(cudaEventCreateWithFlags(&h->ev_probe, cudaEventDisableTiming), "cudaEventCreate")) return PTFLASH_ECUDA;
      h->aux_made = true;
    }
    o.aux_stream = h->aux_stream; o.ev_fork = h->ev_fork; o.ev_join = h->ev_join;
    o.aux2_stream = h->aux2_stream; o.ev_c0 = h->ev_c0; o.ev_c1 = h->ev_c1; o.ev_cjoin = h->ev_cjoin; o.ev_probe = h->ev_probe;
  }
  const int launches = fn(h->sys, o, d, h->ws, st);
  if (launches < 0) { cuda_ok(cudaGetLastError(), "kernel launch"); if (g_err.empty()) set_err("kernel launch failed"); return PTFLASH_ECUDA; }
  if (engine) {
    // stage counters -> pinned host mirror (read by ptflash_get_stats after a synchronise)
    if (!cuda_ok(cudaMemcpyAsync(h->counters_host, h->ws, sizeof(ptf::StageCounters), cudaMemcpyDeviceToHost, st), "cudaMemcpyAsync(counters)"))
      return PTFLASH_ECUDA;
  }
  h->last_stream = st;
  h->used = true;
  h->last_N = io->N;
  h->last_launches = launches;
  h->host_stats = false;
  h->a_last = -1;
  return PTFLASH_OK;
}

int ptflash_flash(ptflash_handle_t h, int64_t N, const double* z, const double* P, const double* T, double* out_beta,
                  double* out_x, double* out_y, int32_t* out_phase, int32_t* out_iters, void* stream) {
  ptflash_io_t io;
  std::memset(&io, 0, sizeof(io));
  io.N = N; io.z = z; io.P = P; io.T = T;
  io.out_beta = out_beta; io.out_x = out_x; io.out_y = out_y; io.out_phase = out_phase; io.out_iters = out_iters;
  return ptflash_flash_ex(h, &io, stream);
}

// Host-buffer variant.  The batch is cut into chunks of consecutive mixtures; chunk c is handled by child handle c on a
// stream of its own: H2D copies of its slices of z, P, T (the SoA slices are strided: copy_rows) -> the flash kernels
// -> D2H copies of its results.  Streams of different chunks overlap, so the PCIe transfers of one chunk hide under the
// kernels of the others (PCIe is full duplex: H2D and D2H use different copy engines).  The device buffers are chunk-local
// SoA ([nc][Nc]), so each chunk is an ordinary ptflash_flash call.
int ptflash_flash_host(ptflash_handle_t h, int64_t N, const double* z, const double* P, const double* T, double* out_beta,
                       double* out_x, double* out_y, int32_t* out_phase, int32_t* out_iters, void* stream) {
  g_err.clear();
  if (!h) { set_err("ptflash_flash_host: null handle"); return PTFLASH_EINVAL; }
  if (N < 0) { set_err("ptflash_flash_host: N < 0"); return PTFLASH_EINVAL; }
  if (N == 0) return PTFLASH_OK;
  if (N > PTFLASH_MAX_N) { set_err("ptflash_flash_host: N exceeds PTFLASH_MAX_N (2^30 - 1); split the batch"); return PTFLASH_EINVAL; }
  if (!z || !P || !T || !out_beta || !out_x || !out_y || !out_phase) { set_err("ptflash_flash_host: null required pointer"); return PTFLASH_EINVAL; }
  DeviceGuard guard(h->device);
  cudaStream_t st = (cudaStream_t)stream;
  const int nc = h->sys.nc;
  // chunks: at most PTFLASH_OPT_HOST_CHUNKS, none smaller than 32768 mixtures (below that a call is latency bound)
  int chunks = (int)h->opts[PTFLASH_OPT_HOST_CHUNKS];
  while (chunks > 1 && N / chunks < 32768) --chunks;
  while (h->n_child < chunks) {
    // a slot counts (n_child) only once its handle, stream and events all exist; a failure on the way releases what was made
    const int c = h->n_child;
    ptflash_handle_s* k = make_child(h);
    if (!k) return PTFLASH_ECUDA;
    if (!cuda_ok(cudaStreamCreateWithFlags(&h->child_stream[c], cudaStreamNonBlocking), "cudaStreamCreate")) { ptflash_destroy(k); return PTFLASH_ECUDA; }
    if (!cuda_ok(cudaEventCreateWithFlags(&h->child_done[c], cudaEventDisableTiming), "cudaEventCreate")) {
      cudaStreamDestroy(h->child_stream[c]); ptflash_destroy(k); return PTFLASH_ECUDA;
    }
    if (c == 0 && !cuda_ok(cudaEventCreateWithFlags(&h->host_begin, cudaEventDisableTiming), "cudaEventCreate")) {
      cudaEventDestroy(h->child_done[c]); cudaStreamDestroy(h->child_stream[c]); ptflash_destroy(k); return PTFLASH_ECUDA;
    }
    h->child[c] = k;
    h->n_child = c + 1;
  }
  // work queued on the caller's stream before this call completes before any chunk starts
  if (!cuda_ok(cudaEventRecord(h->host_begin, st), "cudaEventRecord")) return PTFLASH_ECUDA;
  const int64_t per = ((N + chunks - 1) / chunks + 31) & ~(int64_t)31;
  const size_t hp = (size_t)N * sizeof(double);   // pitch of the host SoA arrays
  int max_pitch_attr = 0x7fffffff;
  cudaDeviceGetAttribute(&max_pitch_attr, cudaDevAttrMaxPitch, h->device);
  const size_t max_pitch = (size_t)max_pitch_attr;
  const bool by_rows = (int)h->opts[PTFLASH_OPT_HOST_ROW_COPIES] != 0;
  int launches = 0;
  for (int c = 0; c < chunks; ++c) {
    const int64_t n0 = (int64_t)c * per;
    const int64_t nn = (n0 + per <= N ? per : N - n0);
    if (nn <= 0) { chunks = c; break; }
    ptflash_handle_s* k = h->child[c];
    std::memcpy(k->opts, h->opts, sizeof(k->opts));
    cudaStream_t cs = h->child_stream[c];
    const size_t nd = (size_t)nn, dp = nd * sizeof(double);
    const size_t need = nd * (size_t)(nc + 2 + 1 + 2 * nc) * sizeof(double) + 2 * nd * sizeof(int32_t);
    if (!ensure(&k->stage, &k->stage_bytes, need, cs, "cudaMalloc(staging)")) return PTFLASH_ECUDA;
    double* dz = (double*)k->stage;
    double* dP = dz + nd * nc;
    double* dT = dP + nd;
    double* dbeta = dT + nd;
    double* dx = dbeta + nd;
    double* dy = dx + nd * nc;
    int32_t* dphase = (int32_t*)(dy + nd * nc);
    int32_t* diters = dphase + nd;
    if (!cuda_ok(cudaStreamWaitEvent(cs, h->host_begin, 0), "cudaStreamWaitEvent")) return PTFLASH_ECUDA;
    if (!copy_rows(dz, dp, z + n0, hp, dp, nc, cudaMemcpyHostToDevice, cs, max_pitch, by_rows, "H2D z")) return PTFLASH_ECUDA;
    if (!cuda_ok(cudaMemcpyAsync(dP, P + n0, dp, cudaMemcpyHostToDevice, cs), "H2D P")) return PTFLASH_ECUDA;
    if (!cuda_ok(cudaMemcpyAsync(dT, T + n0, dp, cudaMemcpyHostToDevice, cs), "H2D T")) return PTFLASH_ECUDA;
    const int rc = ptflash_flash(k, nn, dz, dP, dT, dbeta, dx, dy, dphase, out_iters ? diters : nullptr, cs);
    if (rc != PTFLASH_OK) return rc;
    launches += k->last_launches;
    if (!cuda_ok(cudaMemcpyAsync(out_beta + n0, dbeta, dp, cudaMemcpyDeviceToHost, cs), "D2H beta")) return PTFLASH_ECUDA;
    if (!copy_rows(out_x + n0, hp, dx, dp, dp, nc, cudaMemcpyDeviceToHost, cs, max_pitch, by_rows, "D2H x")) return PTFLASH_ECUDA;
    if (!copy_rows(out_y + n0, hp, dy, dp, dp, nc, cudaMemcpyDeviceToHost, cs, max_pitch, by_rows, "D2H y")) return PTFLASH_ECUDA;
    if (!cuda_ok(cudaMemcpyAsync(out_phase + n0, dphase, nd * sizeof(int32_t), cudaMemcpyDeviceToHost, cs), "D2H phase")) return PTFLASH_ECUDA;
    if (out_iters && !cuda_ok(cudaMemcpyAsync(out_iters + n0, diters, nd * sizeof(int32_t), cudaMemcpyDeviceToHost, cs), "D2H iters")) return PTFLASH_ECUDA;
    if (!cuda_ok(cudaEventRecord(h->child_done[c], cs), "cudaEventRecord")) return PTFLASH_ECUDA;
    if (!cuda_ok(cudaStreamWaitEvent(st, h->child_done[c], 0), "cudaStreamWaitEvent")) return PTFLASH_ECUDA;   // join
  }
  if (!cuda_ok(cudaStreamSynchronize(st), "cudaStreamSynchronize")) return PTFLASH_ECUDA;
  h->last_stream = st;
  h->used = true;
  h->last_N = N;
  h->last_launches = launches;
  h->host_stats = true;
  h->host_chunks_used = chunks;
  h->a_last = -1;
  return PTFLASH_OK;
}

// Pipelined host-buffer variant: batch k's H2D copies, kernels and D2H copies are ordered on the stream of slot k mod DEPTH;
// the slots' streams overlap, so the copies of one batch run under the kernels of its neighbours (PCIe is full duplex).
int ptflash_flash_host_async(ptflash_handle_t h, int64_t N, const double* z, const double* P, const double* T, double* out_beta,
                             double* out_x, double* out_y, int32_t* out_phase, int32_t* out_iters) {
  g_err.clear();
  if (!h) { set_err("ptflash_flash_host_async: null handle"); return PTFLASH_EINVAL; }
  if (N < 0) { set_err("ptflash_flash_host_async: N < 0"); return PTFLASH_EINVAL; }
  if (N == 0) return PTFLASH_OK;
  if (N > PTFLASH_MAX_N) { set_err("ptflash_flash_host_async: N exceeds PTFLASH_MAX_N (2^30 - 1); split the batch"); return PTFLASH_EINVAL; }
  if (!z || !P || !T || !out_beta || !out_x || !out_y || !out_phase) { set_err("ptflash_flash_host_async: null required pointer"); return PTFLASH_EINVAL; }
  DeviceGuard guard(h->device);
  const int nc = h->sys.nc;
  const int slot = (int)(h->a_submitted % PTF_HOST_DEPTH);
  while (h->n_aslot <= slot) {
    const int c = h->n_aslot;
    ptflash_handle_s* k = make_child(h);
    if (!k) return PTFLASH_ECUDA;
    if (!cuda_ok(cudaStreamCreateWithFlags(&h->astream[c], cudaStreamNonBlocking), "cudaStreamCreate")) { ptflash_destroy(k); return PTFLASH_ECUDA; }
    if (!cuda_ok(cudaEventCreateWithFlags(&h->adone[c], cudaEventDisableTiming), "cudaEventCreate")) {
      cudaStreamDestroy(h->astream[c]); ptflash_destroy(k); return PTFLASH_ECUDA;
    }
    h->aslot[c] = k;
    h->n_aslot = c + 1;
  }
  ptflash_handle_s* k = h->aslot[slot];
  cudaStream_t cs = h->astream[slot];
  // the slot's previous batch (DEPTH submissions ago) must have left its staging buffers
  if (h->a_submitted >= PTF_HOST_DEPTH && !cuda_ok(cudaEventSynchronize(h->adone[slot]), "cudaEventSynchronize")) return PTFLASH_ECUDA;
  std::memcpy(k->opts, h->opts, sizeof(k->opts));
  const size_t nd = (size_t)N;
  const size_t need = nd * (size_t)(nc + 2 + 1 + 2 * nc) * sizeof(double) + 2 * nd * sizeof(int32_t);
  if (!ensure(&k->stage, &k->stage_bytes, need, cs, "cudaMalloc(staging)")) return PTFLASH_ECUDA;
  double* dz = (double*)k->stage;
  double* dP = dz + nd * nc;
  double* dT = dP + nd;
  double* dbeta = dT + nd;
  double* dx = dbeta + nd;
  double* dy = dx + nd * nc;
  int32_t* dphase = (int32_t*)(dy + nd * nc);
  int32_t* diters = dphase + nd;
  if (!cuda_ok(cudaMemcpyAsync(dz, z, nd * nc * sizeof(double), cudaMemcpyHostToDevice, cs), "H2D z")) return PTFLASH_ECUDA;
  if (!cuda_ok(cudaMemcpyAsync(dP, P, nd * sizeof(double), cudaMemcpyHostToDevice, cs), "H2D P")) return PTFLASH_ECUDA;
  if (!cuda_ok(cudaMemcpyAsync(dT, T, nd * sizeof(double), cudaMemcpyHostToDevice, cs), "H2D T")) return PTFLASH_ECUDA;
  const int rc = ptflash_flash(k, N, dz, dP, dT, dbeta, dx, dy, dphase, out_iters ? diters : nullptr, cs);
  if (rc != PTFLASH_OK) return rc;
  if (!cuda_ok(cudaMemcpyAsync(out_beta, dbeta, nd * sizeof(double), cudaMemcpyDeviceToHost, cs), "D2H beta")) return PTFLASH_ECUDA;
  if (!cuda_ok(cudaMemcpyAsync(out_x, dx, nd * nc * sizeof(double), cudaMemcpyDeviceToHost, cs), "D2H x")) return PTFLASH_ECUDA;
  if (!cuda_ok(cudaMemcpyAsync(out_y, dy, nd * nc * sizeof(double), cudaMemcpyDeviceToHost, cs), "D2H y")) return PTFLASH_ECUDA;
  if (!cuda_ok(cudaMemcpyAsync(out_phase, dphase, nd * sizeof(int32_t), cudaMemcpyDeviceToHost, cs), "D2H phase")) return PTFLASH_ECUDA;
  if (out_iters && !cuda_ok(cudaMemcpyAsync(out_iters, diters, nd * sizeof(int32_t), cudaMemcpyDeviceToHost, cs), "D2H iters")) return PTFLASH_ECUDA;
  if (!cuda_ok(cudaEventRecord(h->adone[slot], cs), "cudaEventRecord")) return PTFLASH_ECUDA;
  h->a_submitted++;
  h->a_last = slot;
  h->used = true;
  h->last_stream = cs;
  h->last_N = N;
  h->last_launches = k->last_launches;
  h->host_stats = false;
  return PTFLASH_OK;
}

int ptflash_host_wait(ptflash_handle_t h) {
  g_err.clear();
  if (!h) { set_err("ptflash_host_wait: null handle"); return PTFLASH_EINVAL; }
  DeviceGuard guard(h->device);
  for (int c = 0; c < h->n_aslot; ++c)
    if (!cuda_ok(cudaStreamSynchronize(h->astream[c]), "cudaStreamSynchronize")) return PTFLASH_ECUDA;
  return PTFLASH_OK;
}

int ptflash_rachford_rice(ptflash_handle_t h, int64_t N, const double* lnK, const double* z, double* out_theta,
                          double* out_x, double* out_y, double* out_dtheta_dK, void* stream) {
  g_err.clear();
  if (!h) { set_err("ptflash_rachford_rice: null handle"); return PTFLASH_EINVAL; }
  if (N < 0) { set_err("ptflash_rachford_rice: N < 0"); return PTFLASH_EINVAL; }
  if (N == 0) return PTFLASH_OK;
  if (!lnK || !z || !out_theta) { set_err("ptflash_rachford_rice: null required pointer"); return PTFLASH_EINVAL; }
  ptf::launch_rr_fn fn = pick_rr(h->sys.nc);
  if (!fn) { set_err("ptflash_rachford_rice: no kernel for this nc"); return PTFLASH_EINVAL; }
  DeviceGuard guard(h->device);
  ptf::RrIo io;
  io.N = N; io.lnK = lnK; io.z = z; io.theta = out_theta; io.x = out_x; io.y = out_y; io.dth = out_dtheta_dK;
  if (fn(io, (cudaStream_t)stream) < 0) { cuda_ok(cudaGetLastError(), "rachford-rice kernel"); if (g_err.empty()) set_err("kernel launch failed"); return PTFLASH_ECUDA; }
  // not last_stream: the statistics and stage times of the last flash stay tied to the stream that flash ran on
  h->rr_stream = (cudaStream_t)stream;
  h->rr_used = true;
  return PTFLASH_OK;
}

int ptflash_get_stats(ptflash_handle_t h, ptflash_stats_t* out) {
  if (!h || !out) { set_err("ptflash_get_stats: null argument"); return PTFLASH_EINVAL; }
  std::memset(out, 0, sizeof(*out));
  if (!h->used) return PTFLASH_OK;
  DeviceGuard guard(h->device);
  if (!cuda_ok(cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize")) return PTFLASH_ECUDA;
  ptf::StageCounters sum;
  if (h->host_stats) {
    // chunked host call: sums (and maxima) over the chunks' child handles, all complete after the synchronise above
    std::memset(&sum, 0, sizeof(sum));
    for (int k = 0; k < h->host_chunks_used; ++k) {
      const long long* a = (const long long*)h->child[k]->counters_host;
      long long* b = (long long*)&sum;
      const size_t n_add = offsetof(ptf::StageCounters, max_probe) / sizeof(long long), n_all = sizeof(sum) / sizeof(long long);
      for (size_t i = 0; i < n_all; ++i) b[i] = (i < n_add) ? b[i] + a[i] : (a[i] > b[i] ? a[i] : b[i]);
    }
  } else if (h->a_last >= 0) {
    sum = *h->aslot[h->a_last]->counters_host;   // the most recent pipelined batch
  } else {
    sum = *h->counters_host;
  }
  const ptf::StageCounters& c = sum;
  if (c.queue_overflow) { set_err("ptflash_get_stats: an internal work queue overflowed in the last call (results are not trustworthy); please report"); return PTFLASH_ECUDA; }
  out->n_total = h->last_N;
  out->kernel_launches = h->last_launches;
  if ((int)h->opts[PTFLASH_OPT_ENGINE]) {
    out->n_invalid = c.n_invalid;
    out->n_probe_case1 = c.n_case1;
    out->n_probe_case2 = c.n_case2;
    out->n_probe_case3 = c.n_case3;
    out->n_stability = c.n_stab;
    out->n_stab_newton = c.n_stab_newton;
    out->n_split = c.n_split;
    out->n_split_newton = c.n_split_newton;
    out->n_two_phase = c.n_two_phase;
    for (int k = 0; k < 2; ++k) {
      out->n_stab_tr[k] = c.n_stab_tr[k];
      out->n_stab_capped[k] = c.n_stab_capped[k];
      // trials that went on to the trust-region stage did all stab_ss_iters SS iterations (counted off the hot path)
      out->max_stab_ss_iters[k] = (int32_t)c.max_stab_ss[k];
      if (c.n_stab_tr[k] > 0 && out->max_stab_ss_iters[k] < (int32_t)h->opts[PTFLASH_OPT_STAB_SS_ITERS])
        out->max_stab_ss_iters[k] = (int32_t)h->opts[PTFLASH_OPT_STAB_SS_ITERS];
      out->max_stab_tr_iters[k] = (int32_t)c.max_stab_tr[k];
    }
    out->n_split_capped = c.n_split_capped;
    out->n_warm_restarts = c.n_restart;
    out->max_probe_iters = (int32_t)c.max_probe;
    out->max_split_ss_iters = (int32_t)c.max_split_ss;
    out->max_split_tr_iters = (int32_t)c.max_split_tr;
  }
  return PTFLASH_OK;
}

int ptflash_get_stage_ms(ptflash_handle_t h, float* ms, int cap) {
  if (!h || !ms || cap < 0) { set_err("ptflash_get_stage_ms: bad argument"); return PTFLASH_EINVAL; }
  if (!h->used || h->n_events < 2) return 0;
  DeviceGuard guard(h->device);
  if (!cuda_ok(cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize")) return PTFLASH_ECUDA;
  int n = 0;
  for (int i = 0; i + 1 < h->n_events && n < cap; ++i, ++n)
    if (!cuda_ok(cudaEventElapsedTime(&ms[n], h->events[i], h->events[i + 1]), "cudaEventElapsedTime")) return PTFLASH_ECUDA;
  return n;
}

int ptflash_fp64_peak(int iters, double* flops_per_s, double* elapsed_ms, void* stream) {
  g_err.clear();
  if (iters <= 0 || !flops_per_s) { set_err("ptflash_fp64_peak: bad arguments"); return PTFLASH_EINVAL; }
  double fl = 0.0, ms = 0.0;
  if (ptf::run_fp64_peak(iters, &fl, &ms, (cudaStream_t)stream) != 0) { cuda_ok(cudaGetLastError(), "fp64 peak kernel"); return PTFLASH_ECUDA; }
  *flops_per_s = fl;
  if (elapsed_ms) *elapsed_ms = ms;
  return PTFLASH_OK;
}

int ptflash_math_probe(int fn, int64_t n, const double* x, double* y, void* stream) {
  g_err.clear();
  if (fn < 0 || fn >= PTFLASH_NUM_MATH_FN || n < 0 || (n > 0 && (!x || !y))) { set_err("ptflash_math_probe: bad arguments"); return PTFLASH_EINVAL; }
  if (ptf::run_math_probe(fn, n, x, y, (cudaStream_t)stream) != 0) { cuda_ok(cudaGetLastError(), "math probe kernel"); return PTFLASH_ECUDA; }
  return PTFLASH_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// ptflash_flash_static: the staged flash on a workspace that is part of the library's device image, for callers that
// must not allocate (see include/ptflash.h for who they are).  Nothing above this line is used differently by it: it
// borrows the option defaults, make_opt and pick_launcher, and launches the same stage kernels as ptflash_flash_ex.
// ---------------------------------------------------------------------------------------------------------------------
namespace {

// The workspace itself.  A __device__ array at file scope: the CUDA runtime places one copy in the memory of every GPU
// that loads this translation unit's device code and keeps it there until the process ends, so using it costs no
// allocation call -- and nobody can give it back.  256-byte alignment is what carve_workspace assumes of its base.
static __device__ __align__(256) unsigned char g_static_ws[PTFLASH_STATIC_SCRATCH_BYTES];

// CAUTION for whoever edits this file: in HOST code the identifier g_static_ws is only the runtime's host-side stand-in
// for the array.  Its host address is not a device address; handing &g_static_ws[0] to a kernel or to cudaMemsetAsync
// makes the kernel fault (or, on a system where the GPU can reach host memory, scribble over the wrong bytes without
// any error).  The device address has to be asked for, per device, with cudaGetSymbolAddress while that device is
// current; static_workspace() below is the only place that does so and the only way the rest of the file gets the pointer.
constexpr int kStaticMaxDevices = 64;
struct StaticDevice {
  void* ws;            // device address of g_static_ws on this device; nullptr = not asked for yet
  int cta[17][2][4];   // resident-CTA counts of the persistent kernels per (nc, kij all zero): launch_stage2's cache (0 = not queried)
};
StaticDevice g_static_dev[kStaticMaxDevices];   // zero-initialised
std::mutex g_static_mu;                         // guards g_static_dev; held for the (host-side) duration of a call

// Device address of the static workspace on the CURRENT device `dev`, looked up on the first call there.  Caller holds g_static_mu.
void* static_workspace(int dev) {
  StaticDevice& sd = g_static_dev[dev];
  if (sd.ws == nullptr) {
    void* p = nullptr;
    if (!cuda_ok(cudaGetSymbolAddress(&p, g_static_ws), "ptflash_flash_static: cudaGetSymbolAddress(workspace)")) return nullptr;
    if (p == nullptr || ((uintptr_t)p & 255u) != 0) { set_err("ptflash_flash_static: the runtime returned an unusable workspace address"); return nullptr; }
    sd.ws = p;
  }
  return sd.ws;
}

// The component system of a handle-free call: the checks and the constant folding (A.2d-g PAPER.md:420-427, eq. 6
// PAPER.md:74) that ptflash_create applies once per handle, applied per call.
bool static_system(int nc, const double* Tc, const double* Pc, const double* omega, const double* kij, ptf::SysHost* out) {
  if (nc < 2 || nc > PTFLASH_MAX_NC) { set_err("ptflash_flash_static: nc must be in [2, 16]"); return false; }
  if (!Tc || !Pc || !omega) { set_err("ptflash_flash_static: null Tc/Pc/omega"); return false; }
  ptf::SysHost& s = *out;
  std::memset(&s, 0, sizeof(s));
  s.nc = nc;
  s.kij_zero = 1;
  for (int i = 0; i < nc; ++i) {
    if (!std::isfinite(Tc[i]) || !std::isfinite(Pc[i]) || !std::isfinite(omega[i]) || Tc[i] <= 0.0 || Pc[i] <= 0.0) {
      set_err("ptflash_flash_static: Tc and Pc must be finite and positive, omega finite");
      return false;
    }
    const double m = 0.480 + 1.574 * omega[i] - 0.176 * omega[i] * omega[i];
    const double k = std::sqrt(0.42748 / Pc[i]);
    s.u[i] = k * Tc[i] * (1.0 + m);
    s.v[i] = k * std::sqrt(Tc[i]) * m;
    s.wb[i] = 0.08664 * Tc[i] / Pc[i];
    s.lnpc[i] = std::log(Pc[i]);
    s.wil[i] = 5.373 * (1.0 + omega[i]);
    s.tc[i] = Tc[i];
    for (int j = 0; j < nc; ++j) {
      const double kk = kij ? kij[i * nc + j] : 0.0;
      if (!std::isfinite(kk) || (kij && kk != kij[j * nc + i]) || (i == j && kk != 0.0)) {
        set_err("ptflash_flash_static: kij must be finite and symmetric with a zero diagonal");
        return false;
      }
      s.omk[i * nc + j] = 1.0 - kk;
      if (kk != 0.0) s.kij_zero = 0;
    }
  }
  return true;
}

}  // namespace

extern "C" int ptflash_flash_static(int nc, const double* Tc, const double* Pc, const double* omega, const double* kij,
                                    int64_t N, const double* z, const double* P, const double* T, double* out_beta,
                                    double* out_x, double* out_y, int32_t* out_phase, int32_t* out_iters, void* stream) {
  g_err.clear();
  ptf::SysHost sys;
  if (!static_system(nc, Tc, Pc, omega, kij, &sys)) return PTFLASH_EINVAL;
  if (N < 0) { set_err("ptflash_flash_static: N < 0"); return PTFLASH_EINVAL; }
  if (N == 0) return PTFLASH_OK;
  const size_t need = N <= PTFLASH_STATIC_MAX_N ? ptf::staged_workspace_bytes(nc, N) : 0;
  if (N > PTFLASH_STATIC_MAX_N || need > (size_t)PTFLASH_STATIC_SCRATCH_BYTES) {
    // the second condition cannot hold for nc <= 16 and N <= PTFLASH_STATIC_MAX_N; it keeps the two constants honest
    set_err("ptflash_flash_static: N = " + std::to_string((long long)N) + " exceeds PTFLASH_STATIC_MAX_N = " +
            std::to_string(PTFLASH_STATIC_MAX_N) + " (the static workspace is " + std::to_string(PTFLASH_STATIC_SCRATCH_BYTES >> 20) +
            " MiB and cannot grow): cut the batch into pieces of at most that many mixtures, or use ptflash_flash");
    return PTFLASH_EINVAL;
  }
  if (!z || !P || !T || !out_beta || !out_x || !out_y || !out_phase) { set_err("ptflash_flash_static: null required pointer"); return PTFLASH_EINVAL; }
  ptf::launch_fn fn = pick_launcher(nc, 1);
  if (!fn) { set_err("ptflash_flash_static: no kernel for this nc"); return PTFLASH_EINVAL; }
  int dev = 0;
  if (!cuda_ok(cudaGetDevice(&dev), "cudaGetDevice")) return PTFLASH_ECUDA;
  if (dev < 0 || dev >= kStaticMaxDevices) { set_err("ptflash_flash_static: device ordinal beyond the 64 this entry point keeps state for"); return PTFLASH_EINVAL; }
  std::lock_guard<std::mutex> lock(g_static_mu);
  void* ws = static_workspace(dev);
  if (!ws) return PTFLASH_ECUDA;
  ptf::Io d;
  std::memset(&d, 0, sizeof(d));
  d.N = N;
  d.z = z; d.P = P; d.T = T;
  d.beta = out_beta; d.x = out_x; d.y = out_y;
  d.phase = out_phase; d.iters = out_iters;
  // default options; no profiling events and no auxiliary streams, so launch_stage2 orders every stage kernel on `stream`.
  // Its first action is a cudaMemsetAsync of the stage counters and queue lengths at the head of `ws`: the only part of the
  // workspace that has to start at zero, and the array still holds the previous call's values.
  ptf::Opt o = make_opt(kDefaultOpts);
  o.cta_cache = g_static_dev[dev].cta[nc][sys.kij_zero ? 1 : 0];
  const int launches = fn(sys, o, d, ws, (cudaStream_t)stream);
  if (launches < 0) { cuda_ok(cudaGetLastError(), "ptflash_flash_static: kernel launch"); if (g_err.empty()) set_err("ptflash_flash_static: kernel launch failed"); return PTFLASH_ECUDA; }
  return PTFLASH_OK;
}
