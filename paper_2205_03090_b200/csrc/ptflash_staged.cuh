// ptflash_staged.cuh -- engine 1: the flash as a sequence of stage kernels connected by work queues in HBM.
//
// The paper vectorises every stage over the surviving samples and compacts with a boolean mask after EVERY
// iteration, with the host in the loop (synchronizer, eq. 10, Alg. 1; barriers
// at the entry of stability and split).  Here a mixture's iterate stays in registers for a whole
// stage; only the per-stage hand-over (ids + O(nc) doubles) goes through HBM, and the queues are built on the
// device with warp-aggregated atomics (ballot + popc prefix), so the host never waits:
//
//   K1a init        all N: validate, normalise, ln z, d = ln z + lnphi(z), first Rachford-Rice window test
//                   -> q_probe | q_stab (probe case 1) | q_split (caller said "unstable")
//   K1b probe       q_probe: 3 phase-split SS iterations + Delta G/tpd test (section 2.2.3)
//                   -> q_stab (cases 1, 2) | q_split (case 3)
//   K2  stab_ss     2 x q_stab (one work item per start): <= 9 SS iterations (eq. 5) -> done | q_stab_newton
//   K3  stab_newton q_stab_newton: trust-region Newton (B.1-B.3)
//   K4  stab_decide q_stab: label + K seed -> single-phase store | q_split
//   K5  split_ss    q_split: <= 9 SS iterations (Fig. 1) -> store | q_split_newton
//   K6  split_newton q_split_newton: trust-region Newton on G (B.4-B.5) -> store
//
// Every kernel is persistent-style: a fixed grid sized from the SM count walks its queue with a grid-stride
// loop, reading the queue length from device memory.
#pragma once
#include "ptflash_flash.cuh"
#include "ptflash_launch.h"
#include "ptflash_math.cuh"
#include "ptflash_fast.cuh"

namespace ptf {

// The phase split has two queue sets: part 0 = mixtures the probe (or the caller) sent straight to the split, part 1 =
// mixtures the stability analysis found unstable (Q_*_B).  Engine 1 runs part 0 on a second stream, concurrently with
// the stability kernels.
enum : int { Q_PROBE = 0, Q_STAB = 1, Q_STAB_NEWTON = 2, Q_SPLIT = 3, Q_SPLIT_NEWTON = 4, Q_TICKET_STAB = 5, Q_TICKET_SPLIT = 6, Q_RETRY = 7,
              Q_SPLIT_B = 8, Q_SPLIT_NEWTON_B = 9, Q_TICKET_SPLIT_B = 10,
              Q_STAB_NEWTON_E = 11 /* fast engine: trials expected to be short, stored from the END of q_stab_newton */,
              Q_SPLIT_NEWTON_E = 12, Q_SPLIT_NEWTON_BE = 13 /* the same for the two split queues */,
              // part 2 of the phase split ("crawlers"): splits whose successive substitution is still outside 0 < theta < 1 when the
              // switch to the Newton stage is due (reading C13: the SS goes on until theta is inside).  They are rare and can
              // take hundreds of iterations, so they leave the SS kernel and finish on a stream of their own.
              Q_SPLIT_C = 14, Q_SPLIT_NEWTON_C = 15, Q_TICKET_SPLIT_C = 16, Q_SPLIT_NEWTON_CE = 17,
              Q_SPLIT_D = 18, Q_SPLIT_NEWTON_D = 19, Q_TICKET_SPLIT_D = 20, Q_SPLIT_NEWTON_DE = 21 /* part 3: the crawlers of part 1 */, Q_COUNT = 22 };
// queue ids / arrays of split part 0 (probe-found), 1 (stability-found), 2 / 3 (the crawlers of part 0 / 1)
__host__ __device__ __forceinline__ int qid_split(int part) { return part == 0 ? Q_SPLIT : part == 1 ? Q_SPLIT_B : part == 2 ? Q_SPLIT_C : Q_SPLIT_D; }
__host__ __device__ __forceinline__ int qid_split_newton(int part) { return part == 0 ? Q_SPLIT_NEWTON : part == 1 ? Q_SPLIT_NEWTON_B : part == 2 ? Q_SPLIT_NEWTON_C : Q_SPLIT_NEWTON_D; }
__host__ __device__ __forceinline__ int qid_split_newton_e(int part) { return part == 0 ? Q_SPLIT_NEWTON_E : part == 1 ? Q_SPLIT_NEWTON_BE : part == 2 ? Q_SPLIT_NEWTON_CE : Q_SPLIT_NEWTON_DE; }
__host__ __device__ __forceinline__ int qid_ticket_split(int part) { return part == 0 ? Q_TICKET_SPLIT : part == 1 ? Q_TICKET_SPLIT_B : part == 2 ? Q_TICKET_SPLIT_C : Q_TICKET_SPLIT_D; }
enum : int { TF_CONVERGED = 1, TF_EXACT = 2, TF_CAPPED = 4, TF_BETA = 8, TF_ITER_SHIFT = 8 + 0 };

struct Work;
struct Work {
  StageCounters* ctr;
  int* qcount;  // [Q_COUNT]
  int *q_probe, *q_stab, *q_stab_newton, *q_split, *q_split_newton, *q_retry, *q_split_b, *q_split_newton_b;
  int *q_split_c, *q_split_newton_c, *q_split_d, *q_split_newton_d;   // crawlers (split parts 2, 3)
  int* ssk;          // [N] SS iterations done when a crawler left k2_split_ss
  double* crawl;     // [2][N] its theta and last SS residual
  int decide_part;  // queue set k_stab_decide feeds (0 / 1)
  int pass;  // 0: first pass; 1: re-flash of mixtures whose skip-stability hint failed (ST_WARM_RESTART)
  double *lnz, *d, *lnK;   // [NC][N]
  double* zn;              // [NC][N] normalised feed z / sum z (written once by k_init)
  double* lnW;             // [2][NC][N]
  double *tm, *sumW;       // [2][N]
  double *Zfeed, *tpdmin;  // [N]
  double *Zw, *Zxy;        // [2][N] cubic roots handed from an SS stage to its Newton stage (warm starts)
  int* tflags;             // [2][N]
  int *status, *iters, *stabit;  // [N]
  int* actmask;            // [N] bit i set <=> z_i > 0
};

__device__ __forceinline__ int* q_split_of(const Work& w, int part) { return part == 0 ? w.q_split : part == 1 ? w.q_split_b : part == 2 ? w.q_split_c : w.q_split_d; }
__device__ __forceinline__ int* q_split_newton_of(const Work& w, int part) { return part == 0 ? w.q_split_newton : part == 1 ? w.q_split_newton_b : part == 2 ? w.q_split_newton_c : w.q_split_newton_d; }

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

// Carves the workspace; with base == nullptr only the size is computed.
// Queue capacities.  A queue entry is a mixture id (a trial id 2 n + start in q_stab_newton), and an id is appended by the
// one thread that handled that mixture (trial) in the stage before, at most once per queue:
//   k_init            sends every mixture to exactly one of q_probe / q_stab / q_split                       -> each <= N
//   k_requeue_failed_hints  moves q_retry (hinted mixtures, which k_init had put in q_split, never in q_probe)
//                     behind q_probe and empties q_split                                                     -> q_probe <= N
//   k2_probe          sends every mixture of q_probe to q_stab or q_split (distinct from those already there) -> each <= N
//   k2_stab_ss        appends each of the 2 |q_stab| trials at most once to q_stab_newton, hard ones from the
//                     front, easy ones from the back of the same array                                       -> front + back <= 2 N
//   k_stab_decide     appends a mixture of q_stab at most once to q_split_b                                  -> <= N
//   k2_split_ss(p)    sends every mixture of split queue p to the front or the back of q_split_newton(p), or
//                     (p = 0, 1 only) to the crawler queue q_split(p + 2)                                    -> front + back <= N, crawlers <= N
//   a failed hint     is appended once to q_retry                                                            -> <= N
// So no append can pass the end of its array.  The queue_push routines do not clamp (the index would cost every append);
// k_requeue_failed_hints and k_finalize_counters compare the final lengths with these bounds instead -- a check after the
// fact that raises StageCounters::queue_overflow if the argument above is ever broken by a change to the kernels.
inline size_t carve_workspace(int nc, int64_t N, char* base, Work* w) {
  size_t off = 0;
  auto take = [&](size_t bytes) { char* p = base ? base + off : nullptr; off += align256(bytes); return p; };
  const size_t n = (size_t)N, c = (size_t)nc;
  char* p;
  p = take(sizeof(StageCounters)); if (w) w->ctr = (StageCounters*)p;
  p = take(Q_COUNT * sizeof(int)); if (w) w->qcount = (int*)p;
  p = take(n * 4); if (w) w->q_probe = (int*)p;
  p = take(n * 4); if (w) w->q_stab = (int*)p;
  p = take(2 * n * 4); if (w) w->q_stab_newton = (int*)p;
  p = take(n * 4); if (w) w->q_split = (int*)p;
  p = take(n * 4); if (w) w->q_split_newton = (int*)p;
  p = take(n * 4); if (w) w->q_retry = (int*)p;
  p = take(n * 4); if (w) w->q_split_b = (int*)p;
  p = take(n * 4); if (w) w->q_split_newton_b = (int*)p;
  p = take(n * 4); if (w) w->q_split_c = (int*)p;
  p = take(n * 4); if (w) w->q_split_newton_c = (int*)p;
  p = take(n * 4); if (w) w->q_split_d = (int*)p;
  p = take(n * 4); if (w) w->q_split_newton_d = (int*)p;
  p = take(n * 4); if (w) w->ssk = (int*)p;
  p = take(2 * n * 8); if (w) w->crawl = (double*)p;
  if (w) { w->pass = 0; w->decide_part = 0; }
  p = take(c * n * 8); if (w) w->lnz = (double*)p;
  p = take(c * n * 8); if (w) w->d = (double*)p;
  p = take(c * n * 8); if (w) w->lnK = (double*)p;
  p = take(c * n * 8); if (w) w->zn = (double*)p;
  p = take(2 * c * n * 8); if (w) w->lnW = (double*)p;
  p = take(2 * n * 8); if (w) w->tm = (double*)p;
  p = take(2 * n * 8); if (w) w->sumW = (double*)p;
  p = take(n * 8); if (w) w->Zfeed = (double*)p;
  p = take(n * 8); if (w) w->tpdmin = (double*)p;
  p = take(2 * n * 8); if (w) w->Zw = (double*)p;
  p = take(2 * n * 8); if (w) w->Zxy = (double*)p;
  p = take(2 * n * 4); if (w) w->tflags = (int*)p;
  p = take(n * 4); if (w) w->status = (int*)p;
  p = take(n * 4); if (w) w->iters = (int*)p;
  p = take(n * 4); if (w) w->stabit = (int*)p;
  p = take(n * 4); if (w) w->actmask = (int*)p;
  return off;
}

// Warp-aggregated append: lanes with pred == true get consecutive slots of the queue (ballot + prefix popc).
__device__ __forceinline__ void queue_push(bool pred, int* __restrict__ count, int* __restrict__ queue, int value) {
  const unsigned active = __activemask();
  const unsigned mask = __ballot_sync(active, pred);
  if (mask == 0u) return;
  const int lane = threadIdx.x & 31;
  const int leader = __ffs(mask) - 1;
  int base = 0;
  if (lane == leader) base = atomicAdd(count, __popc(mask));
  base = __shfl_sync(active, base, leader);
  if (pred) queue[base + __popc(mask & ((1u << lane) - 1u))] = value;
}

// the same, filling the array downwards from `last` (two queues can share one array, one from each end)
__device__ __forceinline__ void queue_push_back(bool pred, int* __restrict__ count, int* __restrict__ last, int value) {
  const unsigned active = __activemask();
  const unsigned mask = __ballot_sync(active, pred);
  if (mask == 0u) return;
  const int lane = threadIdx.x & 31;
  const int leader = __ffs(mask) - 1;
  int base = 0;
  if (lane == leader) base = atomicAdd(count, __popc(mask));
  base = __shfl_sync(active, base, leader);
  if (pred) last[-(int64_t)(base + __popc(mask & ((1u << lane) - 1u)))] = value;
}

__device__ __forceinline__ void count_add(bool pred, long long* ctr) {
  const unsigned active = __activemask();
  const unsigned mask = __ballot_sync(active, pred);
  if (mask && (int)(threadIdx.x & 31) == __ffs(mask) - 1) atomicAdd((unsigned long long*)ctr, (unsigned long long)__popc(mask));
}

// Table 4's "max number of iterations" rows and the per-start counts: the thread keeps its own maximum / count in a register and the warp
// publishes once, after its loop (all lanes converged), so the hot loop carries a compare instead of an atomic.
__device__ __forceinline__ void flush_max(int v, long long* ctr) {
  const int m = __reduce_max_sync(0xffffffffu, v);
  if (m > 0 && (threadIdx.x & 31) == 0) atomicMax((unsigned long long*)ctr, (unsigned long long)m);
}
__device__ __forceinline__ void flush_add(int v, long long* ctr) {
  const int m = __reduce_add_sync(0xffffffffu, v);
  if (m > 0 && (threadIdx.x & 31) == 0) atomicAdd((unsigned long long*)ctr, (unsigned long long)m);
}

#define PTF_GRID_STRIDE(idx, total) \
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < (total); idx += (int64_t)gridDim.x * blockDim.x)

// ---- K1a ------------------------------------------------------------------------------------------
#ifndef PTF_INIT_MINB
#define PTF_INIT_MINB 4
#endif
template <int NC>
__global__ void __launch_bounds__(128, PTF_INIT_MINB) k_init(const __grid_constant__ Sys<NC> S, const __grid_constant__ Opt o,
                                              const __grid_constant__ Io io, const __grid_constant__ Work w) {
  const int64_t Npad = (io.N + 31) & ~(int64_t)31;  // whole warps stay together for the ballots
  PTF_GRID_STRIDE(idx, Npad) {
    const bool in = idx < io.N;
    const int n = (int)idx;
    MixCtx<NC> m;
    double P = 1.0, T = 1.0, Zf = 0.0;
    bool valid = false;
    if (in) {
      valid = load_feed<NC>(io, n, m.z, P, T);
      if (!valid) store_invalid<NC>(io, n);
    }
    count_add(in && !valid, &w.ctr->n_invalid);
    int dest = -1;  // 0 probe, 1 stab, 2 split
    if (valid) {
      {
        // ln z, per-(P,T) setup and d = ln z + lnphi(z) with the lean math (cold cubic: no previous root)
#pragma unroll
        for (int i = 0; i < NC; ++i) m.lnz[i] = log_fast_m(m.z[i], m.z[i] > 0.0);
        eos_setup<NC>(S, P, T, m.sa, m.bi);
        double lp[NC], Sv[NC];
        Eos e;
        e.Z = 0.0;
        lnphi_fast<NC, false>(S, m.sa, m.bi, m.z, lp, Sv, e);
        Zf = e.Z;
#pragma unroll
        for (int i = 0; i < NC; ++i) m.d[i] = m.lnz[i] + lp[i];
      }
      int status = 0, fl = 0;
      double lnKs[NC];
      const bool have0 = start_lnK<NC>(S, io, n, P, T, lnKs, fl, status);
#pragma unroll
      for (int i = 0; i < NC; ++i) {
        w.lnz[(int64_t)i * io.N + n] = m.lnz[i];
        w.d[(int64_t)i * io.N + n] = m.d[i];
        w.zn[(int64_t)i * io.N + n] = m.z[i];
      }
      w.Zfeed[n] = Zf;
      w.Zxy[n] = 0.0;
      w.Zxy[io.N + n] = 0.0;
      w.status[n] = status;
      w.iters[n] = 0;
      {
        int am = 0;
#pragma unroll
        for (int i = 0; i < NC; ++i) am |= (m.z[i] > 0.0) ? (1 << i) : 0;
        w.actmask[n] = am;
      }
      if (have0 && (fl & 1)) {
        dest = 2;
        w.status[n] = status | ST_INTERNAL_SKIPPED;
#pragma unroll
        for (int i = 0; i < NC; ++i) w.lnK[(int64_t)i * io.N + n] = lnKs[i];
        w.tpdmin[n] = __longlong_as_double(0x7ff8000000000000LL);
      } else if (o.probe_iters == 0) {
        dest = 1;
      } else {
        // first Rachford-Rice of the probe: theta in (0,1) <=> f(0) > 0 and f(1) < 0
        dest = rr_root_inside01<NC>(m.z, lnKs) ? 0 : 1;
      }
    }
    // stabit doubles as the "goes through the stability analysis" mark (-1) that k_stab_decide walks the batch by
    if (in) w.stabit[n] = (dest == 1) ? -1 : 0;
    count_add(dest == 1, &w.ctr->n_case1);
    queue_push(dest == 0, &w.qcount[Q_PROBE], w.q_probe, n);
    queue_push(dest == 1, &w.qcount[Q_STAB], w.q_stab, n);
    queue_push(dest == 2, &w.qcount[Q_SPLIT], w.q_split, n);
  }
}

// Result of one stability trial for k_stab_decide (cf. stab_finish of ptflash_flash.cuh, which engine 0 uses with ln W in
// hand).  v = beta (TF_BETA: the trial was finished by the Newton stage) or ln W (it ended inside k2_stab_ss; m.lnz loaded).
template <int NC>
__device__ __forceinline__ void decide_trial(const Opt& o, const MixCtx<NC>& m, const double (&v)[NC], int flags, double tm,
                                             double sumW, StabRes& res) {
  bool triv = true;
  if (flags & TF_BETA) {
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      const double W = 0.25 * v[i] * v[i];
      if (m.z[i] > 0.0) triv = triv && (W > m.z[i] * o.triv_lo) && (W < m.z[i] * o.triv_hi);
    }
  } else {
    double d = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i)
      if (m.z[i] > 0.0) d = fmax(d, fabs(v[i] - m.lnz[i]));
    triv = d < o.trivial_tol;
  }
  res.trivial = triv;
  res.iters = flags >> TF_ITER_SHIFT;
  res.capped = (flags & TF_CAPPED) != 0;
  if (triv) { res.tm = 0.0; res.tpd = 0.0; }
  else {
    res.tm = (flags & TF_EXACT) ? (1.0 - sumW) : tm;
    res.tpd = -log(1.0 - res.tm);  // tm is second-order accurate; tpd = -ln sum W = -ln(1 - tm) at a stationary point
  }
}
// Label from the two finished trials (readings C9, C10): the part of stab_decide that needs no composition
__device__ __forceinline__ bool stab_label(const Opt& o, const StabRes& sv, const StabRes& sl, double& tpd_min, int& status) {
  if (sv.capped || sl.capped) status |= ST_STAB_CAP;
  tpd_min = 0.0;
  bool any = false;
  if (!sv.trivial) { tpd_min = sv.tpd; any = true; }
  if (!sl.trivial) { tpd_min = any ? fmin(tpd_min, sl.tpd) : sl.tpd; any = true; }
  if (tpd_min != 0.0 && fabs(tpd_min) < o.band) status |= ST_BAND;
  return tpd_min < 0.0;
}

// ---- K4 -------------------------------------------------------------------------------------------
#ifndef PTF_DECIDE_MINB
#define PTF_DECIDE_MINB 4
#endif
template <int NC>
__global__ void __launch_bounds__(128, PTF_DECIDE_MINB) k_stab_decide(const __grid_constant__ Sys<NC> S, const __grid_constant__ Opt o,
                                                     const __grid_constant__ Io io, const __grid_constant__ Work w) {
  // The kernel is bound by memory traffic, so it walks the batch in mixture order (full, coalesced sectors) and skips the
  // mixtures that did not go through the stability analysis, instead of gathering through q_stab (whose order follows the
  // CTA scheduling of k_init / k2_probe: 3.3 x the necessary DRAM traffic).
  const int64_t N = io.N;
  const int64_t pad = (N + 31) & ~(int64_t)31;
  int my_tr = 0;   // trials that came back from the trust-region stage: vapour-like in the low, liquid-like in the high half
  PTF_GRID_STRIDE(idx, pad) {
    const int n = (int)idx;
    const bool in = idx < N && w.stabit[n] == -1;
    bool unstable = false;
    if (in) {
      // A trial finished by the Newton stage comes back as beta = 2 sqrt(W) (B.1a).  Its trivial-solution test (reading C7)
      // max_i |ln W_i - ln z_i| < trivial_tol is taken as triv_lo < W_i / z_i < triv_hi with W_i = (beta_i / 2)^2: no
      // logarithm and no ln z; both are needed only for the K seed of an unstable mixture (2 % of them on config 3) and for
      // the few trials that ended inside k2_stab_ss, which come back as ln W.
      MixCtx<NC> m;
      double P, T;
      load_feed<NC>(io, n, m.z, P, T);
      const int fv = w.tflags[n], fl_ = w.tflags[N + n];
      my_tr += ((fv & TF_BETA) ? 1 : 0) + ((fl_ & TF_BETA) ? 65536 : 0);
      double bv[NC], bl[NC];   // beta or ln W, as stored
#pragma unroll
      for (int i = 0; i < NC; ++i) { bv[i] = w.lnW[(int64_t)i * N + n]; bl[i] = w.lnW[((int64_t)NC + i) * N + n]; }
      const bool need_lnz = !(fv & TF_BETA) || !(fl_ & TF_BETA);
      if (need_lnz) {
#pragma unroll
        for (int i = 0; i < NC; ++i) m.lnz[i] = w.lnz[(int64_t)i * N + n];
      }
      StabRes rv, rl;
      decide_trial<NC>(o, m, bv, fv, w.tm[n], w.sumW[n], rv);
      decide_trial<NC>(o, m, bl, fl_, w.tm[N + n], w.sumW[N + n], rl);
      double lnK[NC], tpd_min = 0.0;
      int status = w.status[n];
      unstable = stab_label(o, rv, rl, tpd_min, status);
      if (unstable) {
        // K seed (reading C10): K = z / W^L if tm^L < tm^V, else W^V / z
        const bool liq = rl.tm < rv.tm;
        const int fs = liq ? fl_ : fv;
#pragma unroll
        for (int i = 0; i < NC; ++i) {
          double lw = liq ? bl[i] : bv[i];
          if (fs & TF_BETA) lw = 2.0 * log_fast_m(0.5 * lw, m.z[i] > 0.0);   // ln W = 2 ln(beta / 2)
          const double lz = need_lnz ? m.lnz[i] : w.lnz[(int64_t)i * N + n];
          lnK[i] = liq ? lz - lw : lw - lz;
        }
      }
      const int stab_iters = rv.iters + rl.iters;
      if (unstable) {
#pragma unroll
        for (int i = 0; i < NC; ++i) w.lnK[(int64_t)i * N + n] = lnK[i];
        w.tpdmin[n] = tpd_min;
        w.status[n] = status;
        w.stabit[n] = stab_iters;
      } else {
        store_result<NC>(io, n, false, 0.0, m.z, m.z, m.z, lnK, w.Zfeed[n], w.iters[n], status & ~ST_INTERNAL_SKIPPED, tpd_min, stab_iters, false);
      }
    }
    queue_push(unstable, &w.qcount[w.decide_part ? Q_SPLIT_B : Q_SPLIT], w.decide_part ? w.q_split_b : w.q_split, n);
  }
  flush_add(my_tr & 0xffff, &w.ctr->n_stab_tr[0]);
  flush_add(my_tr >> 16, &w.ctr->n_stab_tr[1]);
}

// ---- K5 / K6 --------------------------------------------------------------------------------------
// Final store of a mixture that went through the split -- or, if its skip-stability hint did not lead to two phases,
// hand it to the second pass (hint dropped, full cold flash; reported as ST_WARM_RESTART).
template <int NC>
__device__ __forceinline__ void finish_common(const Io& io, const Work& w, int n, const double (&z)[NC], bool two, double theta,
                                              int st_iters, int st_status, const double (&x)[NC], const double (&y)[NC],
                                              const double (&lnK)[NC], bool swap) {
  const int ws = w.status[n];
  const bool retry = (w.pass == 0) && (ws & ST_INTERNAL_SKIPPED) && !two;
  if (retry) {
    w.status[n] = (ws & ST_LNK0_REJECTED) | ST_WARM_RESTART;
    w.iters[n] += st_iters;
  } else {
    int status = (ws | st_status) & ~ST_INTERNAL_SKIPPED;
    if (!two) status |= ST_SPLIT_FAILED;
    store_result<NC>(io, n, two, theta, z, x, y, lnK, w.Zfeed[n], w.iters[n] + st_iters, status, w.tpdmin[n], w.stabit[n], swap);
  }
  count_add(two, &w.ctr->n_two_phase);
  queue_push(retry, &w.qcount[Q_RETRY], w.q_retry, n);
}

// ---- stability-only mode --------------------------------------------------------------------------
// PTFLASH_OPT_STABILITY_ONLY: the mixtures queued for the phase split (probe case 3, the caller's
// "unstable" flag, or the stability verdict) are labelled instead of split; the stable ones were stored by k_stab_decide.
template <int NC>
__global__ void __launch_bounds__(128) k_label_only(const __grid_constant__ Io io, const __grid_constant__ Work w) {
  const int64_t N = io.N;
#pragma unroll 1
  for (int part = 0; part < 2; ++part) {
    const int* const q = part ? w.q_split_b : w.q_split;
    const int64_t cnt = w.qcount[part ? Q_SPLIT_B : Q_SPLIT];
    PTF_GRID_STRIDE(idx, cnt) {
      const int n = q[idx];
      double z[NC], lnK[NC];
#pragma unroll
      for (int i = 0; i < NC; ++i) { z[i] = w.zn[(int64_t)i * N + n]; lnK[i] = w.lnK[(int64_t)i * N + n]; }
      store_unstable_label<NC>(io, n, z, lnK, w.iters[n], w.status[n] & ~ST_INTERNAL_SKIPPED, w.tpdmin[n], w.stabit[n]);
    }
  }
}

// counters that are simply queue lengths (accumulated over the passes)
static __global__ void k_finalize_counters(const __grid_constant__ Work w, const long long N) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    // every queue holds at most N ids (the stability Newton queue 2 N, filled from both ends): argued above carve_workspace,
    // compared here with the final lengths (after the fact: an overflow has already written past its array) and reported by
    // ptflash_get_stats
    bool bad = w.qcount[Q_PROBE] > N || w.qcount[Q_STAB] > N || w.qcount[Q_RETRY] > N ||
               (long long)w.qcount[Q_STAB_NEWTON] + w.qcount[Q_STAB_NEWTON_E] > 2 * N;
#pragma unroll 1
    for (int part = 0; part < 4; ++part)
      bad = bad || w.qcount[qid_split(part)] > N || (long long)w.qcount[qid_split_newton(part)] + w.qcount[qid_split_newton_e(part)] > N;
    if (bad) w.ctr->queue_overflow = 1;
    w.ctr->n_stab += w.qcount[Q_STAB];
    w.ctr->n_stab_newton += w.qcount[Q_STAB_NEWTON] + w.qcount[Q_STAB_NEWTON_E];
    w.ctr->n_split += w.qcount[Q_SPLIT] + w.qcount[Q_SPLIT_B];
    w.ctr->n_split_newton += w.qcount[Q_SPLIT_NEWTON] + w.qcount[Q_SPLIT_NEWTON_B] + w.qcount[Q_SPLIT_NEWTON_E] + w.qcount[Q_SPLIT_NEWTON_BE] +
                             w.qcount[Q_SPLIT_NEWTON_C] + w.qcount[Q_SPLIT_NEWTON_CE] + w.qcount[Q_SPLIT_NEWTON_D] + w.qcount[Q_SPLIT_NEWTON_DE];
  }
}

// Warm-start calls of the fast engine: the splits entered through a skip-stability hint run FIRST; the hints that failed
// (Q_RETRY, reading C21) then join the probe queue of the mixtures without a hint, so the whole call stays one pass.
// The split queues and tickets restart from zero for the probe- and stability-found splits that follow.
static __global__ void k_requeue_failed_hints(const __grid_constant__ Work w, const long long N) {
  int cnt = w.qcount[Q_RETRY];
  const int base = w.qcount[Q_PROBE];
  // the queue lengths of the hinted pass are about to be reset: compare them with their capacities first (the same check
  // as k_finalize_counters makes for the rest of the call), and never copy past the end of q_probe
  const bool bad = cnt > N || base > N || (long long)base + cnt > N || w.qcount[Q_SPLIT] > N ||
                   (long long)w.qcount[Q_SPLIT_NEWTON] + w.qcount[Q_SPLIT_NEWTON_E] > N;
  if (bad) cnt = 0;
  for (int i = threadIdx.x; i < cnt; i += blockDim.x) w.q_probe[base + i] = w.q_retry[i];
  __syncthreads();
  if (threadIdx.x == 0) {
    if (bad) w.ctr->queue_overflow = 1;
    w.ctr->n_restart += cnt;
    w.ctr->n_split += w.qcount[Q_SPLIT];
    w.ctr->n_split_newton += w.qcount[Q_SPLIT_NEWTON] + w.qcount[Q_SPLIT_NEWTON_E];
    w.qcount[Q_PROBE] = base + cnt;
    w.qcount[Q_RETRY] = 0;
    w.qcount[Q_SPLIT] = 0; w.qcount[Q_SPLIT_NEWTON] = 0; w.qcount[Q_SPLIT_NEWTON_E] = 0; w.qcount[Q_TICKET_SPLIT] = 0;
  }
}

}  // namespace ptf
