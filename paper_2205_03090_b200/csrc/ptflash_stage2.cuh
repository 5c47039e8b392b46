// ptflash_stage2.cuh -- optimised stage kernels of engine 1 (see ptflash_staged.cuh for the pipeline).
//
//   k2_probe / k2_stab_ss / k2_split_ss   one work item per thread, iterate in registers, warm-started cubic and
//                                         Rachford-Rice, everything inlined (no per-mixture struct in local memory)
//   k3_stab_newton / k3_split_newton      (ptflash_newton.cuh) persistent warps with LANE REFILL: every lane owns one
//                                         work item; one loop trip = one trust-region iteration (one lnphi evaluation
//                                         per phase + one row-wise Cholesky); a lane whose item finishes stores it and
//                                         pulls the next item from a global ticket (warp ballot + popc prefix), so
//                                         early finishers do not stall their warp (north_star subsystem 4; the
//                                         paper's per-iteration mask-and-compact, eq. 10).
#pragma once
#include "ptflash_fast.cuh"
#include "ptflash_staged.cuh"

namespace ptf {

template <int NC>
__device__ __forceinline__ void load_zn(const Io& io, const Work& w, int n, double (&z)[NC]) {
#pragma unroll
  for (int i = 0; i < NC; ++i) z[i] = __ldg(&w.zn[(int64_t)i * io.N + n]);   // normalised once by k_init
}

// ---- K1b: probe -----------------------------------------------------------------------------------
#ifndef PTF_SPLIT_MINB
#define PTF_SPLIT_MINB 3
#endif
template <int NC, bool KIJ0>
__global__ void __launch_bounds__(128, PTF_SPLIT_MINB) k2_probe(const __grid_constant__ Sys<NC> S, const __grid_constant__ Opt o,
                                                                const __grid_constant__ Io io, const __grid_constant__ Work w) {
  __shared__ double s_exp[PTF_EXP_TAB];
  exp_tab_init(s_exp);
  const int64_t cnt = w.qcount[Q_PROBE];
  const int64_t pad = (cnt + 31) & ~(int64_t)31;
  int my_max = 0;
  PTF_GRID_STRIDE(idx, pad) {
    const bool in = idx < cnt;
    int pcase = 0, n = 0, iters = 0;
    if (in) {
      n = w.q_probe[idx];
      double z[NC], lnK[NC], x[NC], y[NC], lpx[NC], lpy[NC];
      const double P = io.P[n], T = io.T[n];
      PT3<NC> q;
      { const double iT = rcp_fast(T); q.sT = sqrt_fast(T); q.spt = sqrt_fast(P) * iT; q.pt = P * iT; }
      load_zn<NC>(io, w, n, z);
      int status = w.status[n] & ST_WARM_RESTART, fl = 0;
      start_lnK<NC>(S, io, n, P, T, lnK, fl, status);
      double theta = -1.0e300, Zx = 0.0, Zy = 0.0;
      pcase = 2;
#pragma unroll 1
      for (int it = 0; it < o.probe_iters; ++it) {
        {
          double K[NC];
#pragma unroll
          for (int i = 0; i < NC; ++i) K[i] = exp_tab(lnK[i], s_exp);
          if (!rr_fast<NC>(K, z, theta, x, y) || !(theta > 0.0) || !(theta < 1.0)) { pcase = 1; break; }
        }
        Eos e;
        double Sv[NC];
        e.Z = Zx;
        lnphi_pt<NC, KIJ0>(S, q, x, lpx, Sv, e);
        Zx = e.Z;
        e.Z = Zy;
        lnphi_pt<NC, KIJ0>(S, q, y, lpy, Sv, e);
        Zy = e.Z;
#pragma unroll
        for (int i = 0; i < NC; ++i)
          if (z[i] > 0.0) lnK[i] = lpx[i] - lpy[i];
        iters++;
      }
      double tpd_min = 0.0;
      if (pcase == 2 && o.probe_iters > 0) {
        double tx = 0.0, ty = 0.0;
#pragma unroll
        for (int i = 0; i < NC; ++i) {
          const double di = __ldg(&w.d[(int64_t)i * io.N + n]);
          // z_i = 0: x_i = y_i = 0 and the term is 0 * (ln 1 + ..) = 0, without a branch around the logarithms
          tx = fma(x[i], log_fast_m(x[i], x[i] > 0.0) + lpx[i] - di, tx);
          ty = fma(y[i], log_fast_m(y[i], y[i] > 0.0) + lpy[i] - di, ty);
        }
        const double dG = (1.0 - theta) * tx + theta * ty;
        const double mn = dmin(dG, dmin(tx, ty));
        if (mn < -o.probe_margin) { tpd_min = mn; pcase = 3; }
      }
      w.iters[n] += iters;
      if (pcase == 3) {
#pragma unroll
        for (int i = 0; i < NC; ++i) w.lnK[(int64_t)i * io.N + n] = lnK[i];
        w.tpdmin[n] = tpd_min;
        w.Zxy[n] = Zx;
        w.Zxy[io.N + n] = Zy;
      } else {
        w.stabit[n] = -1;   // goes through the stability analysis (k_stab_decide walks the batch by this mark)
      }
    }
    count_add(pcase == 1, &w.ctr->n_case1);
    count_add(pcase == 2, &w.ctr->n_case2);
    count_add(pcase == 3, &w.ctr->n_case3);
    my_max = max(my_max, iters);
    queue_push(pcase == 1 || pcase == 2, &w.qcount[Q_STAB], w.q_stab, n);
    queue_push(pcase == 3, &w.qcount[Q_SPLIT], w.q_split, n);
  }
  flush_max(my_max, &w.ctr->max_probe);
}

// ---- K2: stability SS -----------------------------------------------------------------------------
// Register-lean: the only per-component state kept in registers across iterations is ln W; d sits in shared memory
// (one conflict-free column per thread) and sqrt(A_i), B_i are rebuilt from three scalars, so four CTAs of 128 threads
// fit per SM.  Branch-free over the components: a component with z_i = 0 is carried at ln W_i = LNW_ZERO (W_i underflows
// to ~1e-308 and drops out of every sum) and masked out of the residual with selects, so that the ten exponentials
// of an iteration are one straight-line block the scheduler can interleave (with `act ? exp(..) : 0` the compiler
// emitted ten branch-around blocks, i.e. ten serial Horner chains).
#ifndef PTF_SS_MINB
#define PTF_SS_MINB 4
#endif
constexpr double LNW_ZERO = -1000.0;
// Longest-processing-time-first order of the Newton stage: a trial that is still further than this from the trivial solution
// (max_i |ln W_i - ln z_i|) after the SS iterations is queued at the front.  On config 3 that is 13 % of the trials and it
// contains every trial that needs >= 8 trust-region iterations (87 % of those with >= 5): started first, they no longer
// form the tail of the persistent kernel.
constexpr double STAB_HARD_DIST = 0.3;
template <int NC, bool KIJ0>
__global__ void __launch_bounds__(128, PTF_SS_MINB) k2_stab_ss(const __grid_constant__ Sys<NC> S, const __grid_constant__ Opt o,
                                                               const __grid_constant__ Io io, const __grid_constant__ Work w) {
  __shared__ double s_d[NC * 128];
  __shared__ double s_lz[NC * 128];
  __shared__ double s_exp[PTF_EXP_TAB];
  exp_tab_init(s_exp);
  double* const sd = s_d + threadIdx.x;
  double* const slz = s_lz + threadIdx.x;
  const int64_t cnt = 2 * (int64_t)w.qcount[Q_STAB];
  const int64_t pad = (cnt + 31) & ~(int64_t)31;
  const int64_t N = io.N;
  PTF_GRID_STRIDE(idx, pad) {
    const bool in = idx < cnt;
    bool need_newton = false, capped = false, hard = false;
    int item = 0, iters = 0;
    if (in) {
      const int n = w.q_stab[idx >> 1];
      const int sidx = (int)(idx & 1);  // 0 vapour-like, 1 liquid-like
      item = (n << 1) | sidx;
      double lnW[NC], W[NC], lp[NC], Sv[NC];
      const double P = io.P[n], T = io.T[n];
      PT3<NC> q;
      { const double iT = rcp_fast(T); q.sT = sqrt_fast(T); q.spt = sqrt_fast(P) * iT; q.pt = P * iT; }
      const unsigned act = (unsigned)w.actmask[n];
      {
        int status = w.status[n] & ST_WARM_RESTART, fl = 0;
        double lnKs[NC];
        start_lnK<NC>(S, io, n, P, T, lnKs, fl, status);
        const double side = sidx ? -1.0 : 1.0;
#pragma unroll
        for (int i = 0; i < NC; ++i) {
          const double lz = w.lnz[(int64_t)i * N + n];
          slz[i * 128] = lz;
          lnW[i] = ((act >> i) & 1u) ? fma(side, lnKs[i], lz) : LNW_ZERO;
          sd[i * 128] = __ldg(&w.d[(int64_t)i * N + n]);
        }
      }
      Eos e;
      e.Z = 0.0;
      const int ss_max = o.use_newton ? o.stab_ss_iters : o.ss_cap;
      bool converged = false;
      double tm = 0.0, sumW = 1.0;
#pragma unroll 1
      for (int k = 0; k <= ss_max; ++k) {
        // evaluate the residual r = ln W + lnphi(w) - d at the current iterate
        double sw0 = 0.0, sw1 = 0.0;
#pragma unroll
        for (int i = 0; i < NC; ++i) { W[i] = exp_tab(lnW[i], s_exp); if (i & 1) sw1 += W[i]; else sw0 += W[i]; }
        sumW = sw0 + sw1;
        {
          const double inv = rcp_fast(sumW);
          double wn[NC];
#pragma unroll
          for (int i = 0; i < NC; ++i) wn[i] = W[i] * inv;
          lnphi_pt<NC, KIJ0>(S, q, wn, lp, Sv, e);
        }
        bool conv = true;
        double tm0 = 1.0, tm1 = 0.0;
#pragma unroll
        for (int i = 0; i < NC; ++i) {
          // lp <- d - lnphi (the next iterate of eq. 5); r = ln W - (d - lnphi)
          lp[i] = sd[i * 128] - lp[i];
          const double r = lnW[i] - lp[i];
          conv = conv && (!((act >> i) & 1u) || fabs(r) < o.tol_ss);
          if (i & 1) tm1 = fma(W[i], r - 1.0, tm1); else tm0 = fma(W[i], r - 1.0, tm0);   // a z_i = 0 component adds ~1e-305
        }
        tm = tm0 + tm1;
        if (conv) { converged = true; break; }
        if (k == ss_max) { capped = !o.use_newton; break; }   // the last pass only evaluates (pure-SS mode reports the cap)
#pragma unroll
        for (int i = 0; i < NC; ++i) lnW[i] = ((act >> i) & 1u) ? lp[i] : LNW_ZERO;  // eq. 5
        iters++;
        if (k == ss_max - 1 && o.use_newton) break;   // hand-over to the Newton stage after ss_max updates: no further evaluation needed here
      }
      need_newton = !converged && o.use_newton;
      {
        double dist = 0.0;
#pragma unroll
        for (int i = 0; i < NC; ++i) dist = dmax(dist, ((act >> i) & 1u) ? fabs(lnW[i] - slz[i * 128]) : 0.0);
        hard = dist > STAB_HARD_DIST;
      }
#pragma unroll
      for (int i = 0; i < NC; ++i) {
        const bool a = (act >> i) & 1u;
        const double hb = 2.0 * exp_fast(0.5 * lnW[i]);   // Newton works in beta = 2 sqrt(W) (B.1a)
        w.lnW[((int64_t)sidx * NC + i) * N + n] = a ? (need_newton ? hb : lnW[i]) : 0.0;
      }
      w.tm[(int64_t)sidx * N + n] = tm;
      w.sumW[(int64_t)sidx * N + n] = sumW;
      w.tflags[(int64_t)sidx * N + n] = (converged ? TF_CONVERGED : 0) | (capped ? TF_CAPPED : 0) | (iters << TF_ITER_SHIFT);
      if (need_newton) w.Zw[(int64_t)sidx * N + n] = e.Z;
    }
    // Table-4 counters off the hot path: only a trial that ENDS here (converged within the SS cap, or capped in pure-SS
    // mode: 0.7 % of the trials of config 3) touches a counter; the trials that go on are counted per start by k_stab_decide,
    // and their SS iteration count is the cap itself (ptflash_get_stats folds that in)
    if (in && !need_newton) {
      atomicMax((unsigned long long*)&w.ctr->max_stab_ss[item & 1], (unsigned long long)iters);
      if (capped) atomicAdd((unsigned long long*)&w.ctr->n_stab_capped[item & 1], 1ull);
    }
    // hard trials from the front of the array, the others from its end (the Newton stage takes the front first)
    queue_push(need_newton && hard, &w.qcount[Q_STAB_NEWTON], w.q_stab_newton, item);
    queue_push_back(need_newton && !hard, &w.qcount[Q_STAB_NEWTON_E], w.q_stab_newton + 2 * N - 1, item);
  }
}

// ---- lane refill ----------------------------------------------------------------------------------
// Lanes with want == true take consecutive tickets; returns the ticket (>= total means the queue is exhausted).
__device__ __forceinline__ int64_t take_ticket(bool want, int* __restrict__ ticket) {
  const unsigned mask = __ballot_sync(0xffffffffu, want);
  if (mask == 0u) return -1;
  const int lane = threadIdx.x & 31;
  const int leader = __ffs(mask) - 1;
  int base = 0;
  if (lane == leader) base = atomicAdd(ticket, __popc(mask));
  base = __shfl_sync(0xffffffffu, base, leader);
  return want ? (int64_t)base + __popc(mask & ((1u << lane) - 1u)) : -1;
}

// Trust-region bookkeeping shared by the two Newton kernels: the eta sequence of tr_subproblem() as a
// resumable state machine, so the (large, fully unrolled) build-factor-solve body appears once in the code.
struct EtaSearch {
  double eta, eta_lo, eta_hi, eta0;
  int phase, k;   // phase 0: eta = 0; 1: growing (x8); 2: geometric bisection; 3: done; 4: failed
  __device__ __forceinline__ void start(double e0) { eta = 0.0; eta_lo = 0.0; eta_hi = 0.0; eta0 = e0; phase = 0; k = 0; }
  // feed the outcome of the attempt at `eta`; returns true if `s` of this attempt should be kept
  __device__ __forceinline__ bool feed(bool good, double sn, double Delta, double& kept_sn) {
    bool keep = false;
    if (phase == 0) {
      if (good) { keep = true; kept_sn = sn; phase = 3; }
      else { phase = 1; eta = eta0; k = 0; }
    } else if (phase == 1) {
      if (good) { keep = true; kept_sn = sn; eta_hi = eta; phase = 2; k = 0; }
      else { eta_lo = eta; eta *= 8.0; if (++k >= 60) phase = 4; }
    } else if (phase == 2) {
      if (good) { keep = true; kept_sn = sn; eta_hi = eta; } else eta_lo = eta;
      ++k;
    }
    if (phase == 2) {
      if (kept_sn >= 0.5 * Delta || (eta_lo > 0.0 && eta_hi / eta_lo < 1.5) || k >= 12) phase = 3;
      else eta = (eta_lo > 0.0) ? sqrt_fast(eta_lo * eta_hi) : eta_hi * 0.125;
    }
    return keep;
  }
};

// Longest-processing-time-first order of the split Newton stage: a split whose last SS step contracted by less than this
// factor is queued at the front.  On config 3 that is 4.5 % of the Newton items and every one that needs >= 6 iterations.
constexpr double SPLIT_SLOW_RATE = 0.8;

// ---- K5: phase-split SS ---------------------------------------------------------------------------
template <int NC>
__device__ __forceinline__ void store_split(const Io& io, const Work& w, int n, const double (&z)[NC], bool converged,
                                            bool failed, double theta, int st_iters, int st_status, const double (&x)[NC],
                                            const double (&y)[NC], const double (&lnK)[NC], double Zx, double Zy) {
  const bool two = !failed && converged && theta > 0.0 && theta < 1.0;
  finish_common<NC>(io, w, n, z, two, theta, st_iters, st_status, x, y, lnK, two && (Zy < Zx));   // phase identity by Z (C23)
}

template <int NC, bool KIJ0>
__global__ void __launch_bounds__(128, PTF_SPLIT_MINB) k2_split_ss(const __grid_constant__ Sys<NC> S, const __grid_constant__ Opt o,
                                                                   const __grid_constant__ Io io, const __grid_constant__ Work w,
                                                                   const int part, const int crawl_out) {
  __shared__ double s_exp[PTF_EXP_TAB];
  exp_tab_init(s_exp);
  // part 0 / 1: the splits found by the probe / by the stability analysis, from their K seed.  part 2 / 3: the crawlers they
  // left behind (crawl_out != 0): still outside 0 < theta < 1 when the switch to the Newton stage was due; they resume here,
  // on a stream of their own, with their iterate, iteration count, last residual and theta -- a few mixtures per million
  // that take hundreds of iterations next to a bubble or dew point (reading C13) and would otherwise hold the whole SS
  // stage (paper's 9-component workload: 1.8 ms instead of 0.5 ms).
  const bool resume = part >= 2;
  const int* const q_in = q_split_of(w, part);
  const int64_t cnt = w.qcount[qid_split(part)];
  const int64_t pad = (cnt + 31) & ~(int64_t)31;
  const int64_t N = io.N;
  int my_max = 0;
  PTF_GRID_STRIDE(idx, pad) {
    const bool in = idx < cnt;
    bool go_newton = false, slow = false, crawl = false;
    int n = 0, k = 0, status = 0;
    if (in) {
      n = q_in[idx];
      double z[NC], lnK[NC], x[NC], y[NC], lpx[NC], lpy[NC];
      const double P = io.P[n], T = io.T[n];
      PT3<NC> q;
      { const double iT = rcp_fast(T); q.sT = sqrt_fast(T); q.spt = sqrt_fast(P) * iT; q.pt = P * iT; }
      load_zn<NC>(io, w, n, z);
#pragma unroll
      for (int i = 0; i < NC; ++i) lnK[i] = w.lnK[(int64_t)i * N + n];
      double theta = -1.0e300, r_prev = -1.0;
      if (resume) { k = w.ssk[n]; theta = w.crawl[n]; r_prev = w.crawl[N + n]; }
      const bool hinted = (w.pass == 0) && (w.status[n] & ST_INTERNAL_SKIPPED);
      double Zx = w.Zxy[n], Zy = w.Zxy[N + n];   // roots of the stage that produced lnK (0: none)
      bool converged = false, failed = false, final_rr = false;
      // One copy of exp + Rachford-Rice + the two lnphi evaluations: the Rachford-Rice that makes x, y consistent with
      // the converged lnK is the top of one more trip (final_rr).
#pragma unroll 1
      while (true) {
        double mk = 0.0;
#pragma unroll
        for (int i = 0; i < NC; ++i)
          if (z[i] > 0.0) mk = dmax(mk, fabs(lnK[i]));
        if (mk < o.split_trivial_tol) { failed = true; break; }   // trivial collapse (C22)
        {
          double K[NC];
#pragma unroll
          for (int i = 0; i < NC; ++i) K[i] = exp_tab(lnK[i], s_exp);
          if (!rr_fast<NC>(K, z, theta, x, y)) { failed = true; break; }
        }
        if (final_rr) { converged = true; break; }
        if (o.use_newton && k >= o.split_ss_iters && theta > 0.0 && theta < 1.0) { go_newton = true; break; }
        if (k >= o.ss_cap) { status |= ST_SPLIT_CAP; break; }
        if (crawl_out && o.use_newton && k >= o.split_ss_iters) { crawl = true; break; }   // -> part 2
        // A skip-stability hint (C21) whose successive substitution has not brought theta into (0,1) after hint_ss_cap
        // iterations is dropped here (-> cold re-flash) instead of crawling towards the SS cap: next to the
        // phase boundary such a mixture can take 1e5 iterations (40 ms for the whole call) to fail.
        if (hinted && k >= o.hint_ss_cap && !(theta > 0.0 && theta < 1.0)) { failed = true; break; }
        {
          Eos e;
          double Sv[NC];
          e.Z = Zx;
          lnphi_pt<NC, KIJ0>(S, q, x, lpx, Sv, e);
          Zx = e.Z;
          e.Z = Zy;
          lnphi_pt<NC, KIJ0>(S, q, y, lpy, Sv, e);
          Zy = e.Z;
        }
        double rk = 0.0;
#pragma unroll
        for (int i = 0; i < NC; ++i)
          if (z[i] > 0.0) { const double nk = lpx[i] - lpy[i]; rk = dmax(rk, fabs(nk - lnK[i])); lnK[i] = nk; }
        ++k;
        slow = r_prev > 0.0 && rk > SPLIT_SLOW_RATE * r_prev;
        if (rk < 1.0e-14) final_rr = true;
        else if (r_prev > 0.0 && rk < o.tol_ss) {
          const double rho = rk * rcp_fast(r_prev);   // linear-convergence error estimate eps = r rho / (1 - rho)
          if (rho < 1.0 && rk * rho < o.tol_ss * (1.0 - rho)) final_rr = true;
        }
        r_prev = rk;
      }
      if (crawl) {
        // state of the iteration, resumed by the launch for part 2 (lnK as it stands; the Rachford-Rice is repeated there)
#pragma unroll
        for (int i = 0; i < NC; ++i) w.lnK[(int64_t)i * N + n] = lnK[i];
        w.ssk[n] = k;
        w.crawl[n] = theta;
        w.crawl[N + n] = r_prev;
        w.Zxy[n] = Zx;
        w.Zxy[N + n] = Zy;
      } else if (go_newton) {
        // hand-over in the Newton variables: n^V_i = theta y_i (B.4)
        // ... of the MINORITY phase: for theta > 1/2 the roles of the two phases are exchanged (n^L = (1 - theta) x is
        // handed over as "n^V"), so that the majority composition (z - n)/(1 - sum n) is formed without cancellation; G
        // and its stationary point are the same, and the final store restores the phase identity by Z (C23).
        const bool mirror = theta > 0.5;
#pragma unroll
        for (int i = 0; i < NC; ++i) w.lnK[(int64_t)i * N + n] = dmin(mirror ? (1.0 - theta) * x[i] : theta * y[i], z[i]);
        w.iters[n] += k;
        w.status[n] |= status;
        w.Zxy[n] = mirror ? Zy : Zx;
        w.Zxy[N + n] = mirror ? Zx : Zy;
      } else {
        store_split<NC>(io, w, n, z, converged, failed, theta, k, status, x, y, lnK, Zx, Zy);
      }
    }
    my_max = max(my_max, k);
    count_add((status & ST_SPLIT_CAP) != 0, &w.ctr->n_split_capped);   // rare: no atomic unless a lane hit the cap
    // longest first: splits whose successive substitution was still contracting slowly (near-critical mixtures) are queued at
    // the front of the array, the others from its end (the Newton stage takes the front first)
    queue_push(go_newton && slow, &w.qcount[qid_split_newton(part)], q_split_newton_of(w, part), n);
    queue_push_back(go_newton && !slow, &w.qcount[qid_split_newton_e(part)], q_split_newton_of(w, part) + N - 1, n);
    queue_push(crawl, &w.qcount[qid_split(part + 2)], q_split_of(w, part + 2), n);
  }
  flush_max(my_max, &w.ctr->max_split_ss);
}

}  // namespace ptf
#include "ptflash_newton.cuh"
namespace ptf {

template <int NC, bool KIJ0>
int launch_stage2_impl(const Sys<NC>& s, const Opt& o, const Io& io, const Work& w_in, int sms, cudaStream_t st) {
  const int threads = 128;
  auto grid_for = [&](int64_t items) {
    const int64_t need = (items + threads - 1) / threads;
    const int64_t cap = (int64_t)sms * 16;
    return (unsigned)(need < cap ? (need > 0 ? need : 1) : cap);
  };
  const unsigned gN = grid_for(io.N), g2N = grid_for(2 * io.N);
  Work w = w_in;
  // persistent refill kernels: as many CTAs per SM as registers and shared memory allow (queried once per instantiation)
  const size_t stab_bytes = (size_t)stabn_smem_doubles<NC>() * NEWTON_THREADS * sizeof(double);
  const size_t split_bytes = (size_t)splitn_smem_doubles<NC>() * NEWTON_THREADS * sizeof(double);
  // (queried once per handle, i.e. per device and component system: the shared-memory attribute of a kernel is device
  // state; setting it again from another handle on the same device is idempotent)
  int local_cache[2] = {0, 0};
  int* const cache = o.cta_cache ? o.cta_cache : local_cache;
  if (cache[0] == 0 || cache[1] == 0) {
    if (cudaFuncSetAttribute(k3_stab_newton<NC, KIJ0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)stab_bytes) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(k3_split_newton<NC, KIJ0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)split_bytes) != cudaSuccess) return -1;
    int a = 0, b = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, k3_stab_newton<NC, KIJ0>, NEWTON_THREADS, stab_bytes) != cudaSuccess) return -1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, k3_split_newton<NC, KIJ0>, NEWTON_THREADS, split_bytes) != cudaSuccess) return -1;
    if (a < 1 || b < 1) return -1;   // the kernel does not fit an SM: report instead of launching an empty grid
    cache[0] = a;
    cache[1] = b;
  }
  const int stab_cta = cache[0], split_cta = cache[1];
  // optional stage profiling: one event before the first kernel and one after every stage kernel
  cudaEvent_t* ev = (cudaEvent_t*)o.prof_events;
  int nev = 0;
  auto mark = [&]() { if (ev && nev < PTF_MAX_STAGE_EVENTS) cudaEventRecord(ev[nev++], st); };
  mark();
  k_init<NC><<<gN, threads, 0, st>>>(s, o, io, w);
  mark();
  int launches = 1;
  // Fork after the stability stages.  The phase split has two parts: (0) the mixtures the probe (or the caller's flag)
  // declared unstable -- most of them, well conditioned -- and (1) the few the stability analysis found unstable: close
  // to the phase boundary, where single mixtures take ~100 trust-region trips, so that part 1 alone ends in a long tail
  // with a handful of busy lanes (0.24 ms of a 3.2 ms call on config 3, profiles/r02g_kernels.md).  Part 1 runs on the caller's stream, part 0 on the
  // handle's second stream at the same time, so the tail of one is covered by the bulk of the other.  (Running part 0
  // earlier, concurrently with the stability kernels, gains little: those fill the register file on their own.)
  // With stage profiling on, everything stays on the caller's stream so that the event-to-event times are per stage.
  cudaStream_t aux = (cudaStream_t)o.aux_stream;
  const bool fork = aux != nullptr && ev == nullptr;
  w.decide_part = 1;
  // Warm-start call (caller flags): the hinted splits run first; the hints that fail (reading C21) are appended to the probe
  // queue and take the cold path together with the mixtures that came without a hint -- one pass, no second sweep
  // (in stability-only mode a hint is a verdict, not a split: nothing to run).
  if (io.flags && io.lnK0 && !o.stability_only) {
    k2_split_ss<NC, KIJ0><<<gN, threads, 0, st>>>(s, o, io, w, 0, 0);
    mark();
    k3_split_newton<NC, KIJ0><<<(unsigned)(sms * split_cta), NEWTON_THREADS, split_bytes, st>>>(s, o, io, w, 0);
    mark();
    k_requeue_failed_hints<<<1, 1024, 0, st>>>(w, (long long)io.N);
    mark();
    launches += 3;
  }
  w.pass = 0;
  k2_probe<NC, KIJ0><<<gN, threads, 0, st>>>(s, o, io, w);
  mark();
  // the crawlers (parts 2, 3) are few: a small grid for their SS, one Newton CTA per SM
  const unsigned gC = grid_for(io.N < 65536 ? io.N : 65536);
  const bool early = fork && !o.stability_only && o.early_split_ss;
  cudaStream_t aux2 = (cudaStream_t)o.aux2_stream;
  if (early) {
    // PTFLASH_OPT_EARLY_SPLIT_SS: the SS stage of the probe-found splits (part 0) starts right after the probe, next to the
    // stability analysis of the other mixtures, and hands its crawlers to the third stream at once: a crawler is a serial chain
    // of hundreds of iterations (~3 us each) that nothing shortens, so it has to start early to end under the rest of the call.
    // (The Newton stage of part 0 still waits for k_stab_decide: its persistent CTAs would hold half of the register file
    // while the stability kernels need it.)
    cudaEventRecord((cudaEvent_t)o.ev_probe, st);
    cudaStreamWaitEvent(aux, (cudaEvent_t)o.ev_probe, 0);
    k2_split_ss<NC, KIJ0><<<gN, threads, 0, aux>>>(s, o, io, w, 0, 1);
    cudaEventRecord((cudaEvent_t)o.ev_c0, aux);
    cudaStreamWaitEvent(aux2, (cudaEvent_t)o.ev_c0, 0);
    k2_split_ss<NC, KIJ0><<<gC, threads, 0, aux2>>>(s, o, io, w, 2, 0);
    k3_split_newton<NC, KIJ0><<<(unsigned)sms, NEWTON_THREADS, split_bytes, aux2>>>(s, o, io, w, 2);
  }
  k2_stab_ss<NC, KIJ0><<<g2N, threads, 0, st>>>(s, o, io, w);
  mark();
  k3_stab_newton<NC, KIJ0><<<(unsigned)(sms * stab_cta), NEWTON_THREADS, stab_bytes, st>>>(s, o, io, w);
  mark();
  k_stab_decide<NC><<<gN, threads, 0, st>>>(s, o, io, w);
  mark();
  if (o.stability_only) {
    k_label_only<NC><<<gN, threads, 0, st>>>(io, w);
    mark();
    k_finalize_counters<<<1, 32, 0, st>>>(w, (long long)io.N);
    mark();
    launches += 6;
  } else {
    if (fork) {
      cudaEventRecord((cudaEvent_t)o.ev_fork, st);
      cudaStreamWaitEvent(aux, (cudaEvent_t)o.ev_fork, 0);
      // part 1 first: its hard items should start as early as possible, every one on a lane of its own if they fit
      // (one CTA per SM: 19 k lanes on B200, and room for part 0 next to it)
      k2_split_ss<NC, KIJ0><<<gN, threads, 0, st>>>(s, o, io, w, 1, 1);
      cudaEventRecord((cudaEvent_t)o.ev_c1, st);
      k3_split_newton<NC, KIJ0><<<(unsigned)sms, NEWTON_THREADS, split_bytes, st>>>(s, o, io, w, 1);
      if (!early) {
        k2_split_ss<NC, KIJ0><<<gN, threads, 0, aux>>>(s, o, io, w, 0, 1);
        cudaEventRecord((cudaEvent_t)o.ev_c0, aux);
        cudaStreamWaitEvent(aux2, (cudaEvent_t)o.ev_c0, 0);
        k2_split_ss<NC, KIJ0><<<gC, threads, 0, aux2>>>(s, o, io, w, 2, 0);
        k3_split_newton<NC, KIJ0><<<(unsigned)sms, NEWTON_THREADS, split_bytes, aux2>>>(s, o, io, w, 2);
      }
      k3_split_newton<NC, KIJ0><<<(unsigned)(sms * split_cta), NEWTON_THREADS, split_bytes, aux>>>(s, o, io, w, 0);
      cudaEventRecord((cudaEvent_t)o.ev_join, aux);
      // the crawlers of part 1 follow those of part 0 on the third stream
      cudaStreamWaitEvent(aux2, (cudaEvent_t)o.ev_c1, 0);
      k2_split_ss<NC, KIJ0><<<gC, threads, 0, aux2>>>(s, o, io, w, 3, 0);
      k3_split_newton<NC, KIJ0><<<(unsigned)sms, NEWTON_THREADS, split_bytes, aux2>>>(s, o, io, w, 3);
      cudaEventRecord((cudaEvent_t)o.ev_cjoin, aux2);
      cudaStreamWaitEvent(st, (cudaEvent_t)o.ev_join, 0);    // join
      cudaStreamWaitEvent(st, (cudaEvent_t)o.ev_cjoin, 0);
    } else {
      k2_split_ss<NC, KIJ0><<<gN, threads, 0, st>>>(s, o, io, w, 0, 1);
      k2_split_ss<NC, KIJ0><<<gN, threads, 0, st>>>(s, o, io, w, 1, 1);
      k2_split_ss<NC, KIJ0><<<gC, threads, 0, st>>>(s, o, io, w, 2, 0);
      k2_split_ss<NC, KIJ0><<<gC, threads, 0, st>>>(s, o, io, w, 3, 0);
      mark();
      k3_split_newton<NC, KIJ0><<<(unsigned)(sms * split_cta), NEWTON_THREADS, split_bytes, st>>>(s, o, io, w, 0);
      k3_split_newton<NC, KIJ0><<<(unsigned)(sms * split_cta), NEWTON_THREADS, split_bytes, st>>>(s, o, io, w, 1);
      k3_split_newton<NC, KIJ0><<<(unsigned)sms, NEWTON_THREADS, split_bytes, st>>>(s, o, io, w, 2);
      k3_split_newton<NC, KIJ0><<<(unsigned)sms, NEWTON_THREADS, split_bytes, st>>>(s, o, io, w, 3);
    }
    k_finalize_counters<<<1, 32, 0, st>>>(w, (long long)io.N);
    mark();
    launches += 13;
  }
  if (o.prof_count) *o.prof_count = nev;
  return cudaGetLastError() == cudaSuccess ? launches : -1;
}

// engine 1 entry
template <int NC>
int launch_stage2(const SysHost& hs, const Opt& o, const Io& io, void* workspace, cudaStream_t st) {
  const Sys<NC> s = narrow<NC>(hs);
  Work w;
  carve_workspace(NC, io.N, (char*)workspace, &w);
  if (cudaMemsetAsync(workspace, 0, align256(sizeof(StageCounters)) + align256(Q_COUNT * sizeof(int)), st) != cudaSuccess) return -1;
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  return hs.kij_zero ? launch_stage2_impl<NC, true>(s, o, io, w, sms, st) : launch_stage2_impl<NC, false>(s, o, io, w, sms, st);
}

}  // namespace ptf
