// ptflash_stage2.cuh -- optimised stage kernels of engine 1 (see ptflash_staged.cuh for the pipeline).
//
//   k2_probe / k2_stab_ss / k2_split_ss   one work item per thread, iterate in registers, warm-started cubic and
//                                         Rachford-Rice, everything inlined (no per-mixture struct in local memory)
//   k2_stab_newton / k2_split_newton      persistent warps with LANE REFILL: every lane owns one work item; one loop
//                                         trip = one trust-region iteration (one lnphi evaluation per phase + one
//                                         packed in-register Cholesky); a lane whose item finishes stores it and
//                                         pulls the next item from a global ticket (warp ballot + popc prefix), so
//                                         early finishers do not stall their warp (north_star subsystem 4; the
//                                         paper's per-iteration mask-and-compact, eq. 10).
#pragma once
#include "ptflash_fast.cuh"
#include "ptflash_staged.cuh"

namespace ptf {

// per-(P,T) arrays + active mask of mixture n (already validated and normalised by k_init)
template <int NC>
__device__ __forceinline__ void load_pt(const Sys<NC>& S, const Io& io, int n, double (&sa)[NC], double (&bi)[NC], double& P,
                                        double& T) {
  P = io.P[n];
  T = io.T[n];
  eos_setup<NC>(S, P, T, sa, bi);
}

template <int NC>
__device__ __forceinline__ void load_zn(const Io& io, const Work& w, int n, double (&z)[NC]) {
#pragma unroll
  for (int i = 0; i < NC; ++i) z[i] = __ldg(&w.zn[(int64_t)i * io.N + n]);   // normalised once by k_init
}

// one successive-substitution iteration of the phase split (Fig. 1): K = exp(lnK), RR, lnphi(x), lnphi(y),
// lnK <- lnphi(x) - lnphi(y).  Returns false if Rachford-Rice has no window.  rk = max |d lnK|.
template <int NC, bool KIJ0>
__device__ __forceinline__ bool split_iteration(const Sys<NC>& S, const double (&sa)[NC], const double (&bi)[NC],
                                                const double (&z)[NC], double (&lnK)[NC], double& theta, double (&x)[NC],
                                                double (&y)[NC], double (&lpx)[NC], double (&lpy)[NC], double& Zx, double& Zy,
                                                double& rk, bool update) {
  double K[NC], Sv[NC];
#pragma unroll
  for (int i = 0; i < NC; ++i) K[i] = exp_fast(lnK[i]);
  if (!rr_fast<NC>(K, z, theta, x, y)) return false;
  if (!update) return true;
  Eos e;
  e.Z = Zx;
  lnphi_fast<NC, KIJ0>(S, sa, bi, x, lpx, Sv, e);
  Zx = e.Z;
  e.Z = Zy;
  lnphi_fast<NC, KIJ0>(S, sa, bi, y, lpy, Sv, e);
  Zy = e.Z;
  rk = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i)
    if (z[i] > 0.0) { const double nk = lpx[i] - lpy[i]; rk = fmax(rk, fabs(nk - lnK[i])); lnK[i] = nk; }
  return true;
}

// ---- K1b: probe -----------------------------------------------------------------------------------
#ifndef PTF_SPLIT_MINB
#define PTF_SPLIT_MINB 3
#endif
template <int NC, bool KIJ0>
__global__ void __launch_bounds__(128, PTF_SPLIT_MINB) k2_probe(const __grid_constant__ Sys<NC> S, const __grid_constant__ Opt o,
                                                                const __grid_constant__ Io io, const __grid_constant__ Work w) {
  const int64_t cnt = w.qcount[Q_PROBE];
  const int64_t pad = (cnt + 31) & ~(int64_t)31;
  PTF_GRID_STRIDE(idx, pad) {
    const bool in = idx < cnt;
    int pcase = 0, n = 0;
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
      int iters = 0;
      pcase = 2;
#pragma unroll 1
      for (int it = 0; it < o.probe_iters; ++it) {
        {
          double K[NC];
#pragma unroll
          for (int i = 0; i < NC; ++i) K[i] = exp_fast(lnK[i]);
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
          if (x[i] > 0.0) tx = fma(x[i], log_fast(x[i]) + lpx[i] - di, tx);
          if (y[i] > 0.0) ty = fma(y[i], log_fast(y[i]) + lpy[i] - di, ty);
        }
        const double dG = (1.0 - theta) * tx + theta * ty;
        const double mn = fmin(dG, fmin(tx, ty));
        if (mn < -o.probe_margin) { tpd_min = mn; pcase = 3; }
      }
      w.iters[n] += iters;
      if (pcase == 3) {
#pragma unroll
        for (int i = 0; i < NC; ++i) w.lnK[(int64_t)i * io.N + n] = lnK[i];
        w.tpdmin[n] = tpd_min;
        w.Zxy[n] = Zx;
        w.Zxy[io.N + n] = Zy;
      }
    }
    count_add(pcase == 1, &w.ctr->n_case1);
    count_add(pcase == 2, &w.ctr->n_case2);
    count_add(pcase == 3, &w.ctr->n_case3);
    queue_push(pcase == 1 || pcase == 2, &w.qcount[Q_STAB], w.q_stab, n);
    queue_push(pcase == 3, &w.qcount[Q_SPLIT], w.q_split, n);
  }
}

// ---- K2: stability SS -----------------------------------------------------------------------------
// Register-lean: the only per-component state kept across iterations is ln W; d is re-read from the workspace
// (L1/L2 resident) and sqrt(A_i), B_i are rebuilt from three scalars, so four CTAs of 128 threads fit per SM.
#ifndef PTF_SS_MINB
#define PTF_SS_MINB 4
#endif
template <int NC, bool KIJ0>
__global__ void __launch_bounds__(128, PTF_SS_MINB) k2_stab_ss(const __grid_constant__ Sys<NC> S, const __grid_constant__ Opt o,
                                                               const __grid_constant__ Io io, const __grid_constant__ Work w) {
  const int64_t cnt = 2 * (int64_t)w.qcount[Q_STAB];
  const int64_t pad = (cnt + 31) & ~(int64_t)31;
  const int64_t N = io.N;
  PTF_GRID_STRIDE(idx, pad) {
    const bool in = idx < cnt;
    bool need_newton = false;
    int item = 0;
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
        for (int i = 0; i < NC; ++i) lnW[i] = ((act >> i) & 1u) ? fma(side, lnKs[i], w.lnz[(int64_t)i * N + n]) : 0.0;
      }
      Eos e;
      e.Z = 0.0;
      const int ss_max = o.use_newton ? o.stab_ss_iters : o.ss_cap;
      bool converged = false, capped = false;
      int iters = 0;
      double tm = 0.0, sumW = 1.0;
#pragma unroll 1
      for (int k = 0; k <= ss_max; ++k) {
        // evaluate the residual r = ln W + lnphi(w) - d at the current iterate
        sumW = 0.0;
#pragma unroll
        for (int i = 0; i < NC; ++i) { W[i] = ((act >> i) & 1u) ? exp_fast(lnW[i]) : 0.0; sumW += W[i]; }
        {
          const double inv = rcp_fast(sumW);
          double wn[NC];
#pragma unroll
          for (int i = 0; i < NC; ++i) wn[i] = W[i] * inv;
          lnphi_pt<NC, KIJ0>(S, q, wn, lp, Sv, e);
        }
        double rmax = 0.0;
        tm = 1.0;
#pragma unroll
        for (int i = 0; i < NC; ++i) {
          // lp <- d - lnphi (the next iterate of eq. 5); r = ln W - (d - lnphi)
          lp[i] = __ldg(&w.d[(int64_t)i * N + n]) - lp[i];
          const double r = ((act >> i) & 1u) ? lnW[i] - lp[i] : 0.0;
          rmax = fmax(rmax, fabs(r));
          tm = fma(W[i], r - 1.0, tm);
        }
        if (rmax < o.tol_ss) { converged = true; break; }
        if (k == ss_max) { capped = !o.use_newton; break; }   // the last pass only evaluates (pure-SS mode reports the cap)
        if (k == ss_max - 1 && o.use_newton) {
          // hand-over to the Newton stage after ss_max updates: no further evaluation needed here
#pragma unroll
          for (int i = 0; i < NC; ++i)
            if ((act >> i) & 1u) lnW[i] = lp[i];
          iters++;
          break;
        }
#pragma unroll
        for (int i = 0; i < NC; ++i)
          if ((act >> i) & 1u) lnW[i] = lp[i];  // eq. 5
        iters++;
      }
      need_newton = !converged && o.use_newton;
#pragma unroll
      for (int i = 0; i < NC; ++i)
        w.lnW[((int64_t)sidx * NC + i) * N + n] =
            need_newton ? (((act >> i) & 1u) ? 2.0 * exp_fast(0.5 * lnW[i]) : 0.0) : lnW[i];   // Newton works in beta = 2 sqrt(W) (B.1a)
      w.tm[(int64_t)sidx * N + n] = tm;
      w.sumW[(int64_t)sidx * N + n] = sumW;
      w.tflags[(int64_t)sidx * N + n] = (converged ? TF_CONVERGED : 0) | (capped ? TF_CAPPED : 0) | (iters << TF_ITER_SHIFT);
      if (need_newton) w.Zw[(int64_t)sidx * N + n] = e.Z;
    }
    queue_push(need_newton, &w.qcount[Q_STAB_NEWTON], w.q_stab_newton, item);
  }
}

#ifndef PTF_TRI_SMEM
#define PTF_TRI_SMEM 1   // packed Newton matrices in shared memory (440 B per thread at nc = 10) instead of registers
#endif
#ifndef PTF_NEWTON_MINB
#define PTF_NEWTON_MINB 3
#endif
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

// ---- K3: stability trust-region Newton (B.1-B.3), persistent warps with lane refill --------------
template <int NC, bool KIJ0>
__global__ void __launch_bounds__(128, PTF_NEWTON_MINB) k2_stab_newton(const __grid_constant__ Sys<NC> S, const __grid_constant__ Opt o,
                                                      const __grid_constant__ Io io, const __grid_constant__ Work w) {
  constexpr int NT = NC * (NC + 1) / 2;
  constexpr unsigned FULL = 0xffffffffu;
  const int64_t N = io.N;
  const int total = w.qcount[Q_STAB_NEWTON];
  int* ticket = &w.qcount[Q_TICKET_STAB];
  // ---- lane state ----
  bool busy = false, exhausted = false, first = true, reeval = false, searching = false, exact = false;
  int n = 0, sidx = 0, iters = 0, tr_it = 0;
  unsigned act = 0u;
  double spt = 0.0, sT = 0.0, pt = 0.0;   // sqrt(P)/T, sqrt(T), P/T: sqrt(A_i), B_i are rebuilt from constants
  double beta[NC], s[NC];                 // accepted point (beta = 2 sqrt(W), B.1a) and pending / best-so-far step
  double tm = 0.0, rmax_acc = 0.0, pred = 0.0, Delta = 1.0, Delta_cap = 8.0, snorm = 0.0, Zw = 0.0, kept_sn = 0.0;
  EtaSearch es;
  es.start(1.0e-3);
#pragma unroll
  for (int i = 0; i < NC; ++i) { beta[i] = 0.0; s[i] = 0.0; }

#pragma unroll 1
  while (true) {
    // ---- refill idle lanes from the ticket ----
    if (__any_sync(FULL, !busy && !exhausted)) {
      const int64_t tk = take_ticket(!busy && !exhausted, ticket);
      if (tk >= 0) {
        if (tk < total) {
          const int item = w.q_stab_newton[tk];
          n = item >> 1;
          sidx = item & 1;
          const double P = io.P[n], T = io.T[n];
          { const double iT = rcp_fast(T); sT = sqrt_fast(T); spt = sqrt_fast(P) * iT; pt = P * iT; }
          act = (unsigned)w.actmask[n];
#pragma unroll
          for (int i = 0; i < NC; ++i) {
            beta[i] = w.lnW[((int64_t)sidx * NC + i) * N + n];   // k2_stab_ss left beta = 2 sqrt(W) here
            s[i] = 0.0;
          }
          iters = w.tflags[(int64_t)sidx * N + n] >> TF_ITER_SHIFT;
          tr_it = 0;
          first = true;
          reeval = false;
          searching = false;
          Zw = w.Zw[(int64_t)sidx * N + n];
          busy = true;
        } else {
          exhausted = true;
        }
      }
    }
    if (!__any_sync(FULL, busy)) break;

    // The trip below is written WITHOUT early `continue`s and with explicit __syncwarp() joins: the factorisation
    // block must be entered once per trip by all searching lanes together (a divergent entry makes the warp run
    // the ~1500-instruction block twice with half the lanes each).
    double sa[NC], bi[NC], W[NC], lp[NC], Sv[NC], r[NC];
    double sumW = 0.0;
    Eos e;
    e.Z = Zw;
    bool finish = false, fin_conv = false, fin_exact = false, fin_cap = false;
    if (busy) {
    // ---- evaluate tm and its gradient: at the trial point beta + s, or at beta while an eta search is pending ----
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      sa[i] = spt * fabs(fma(-S.v[i], sT, S.u[i]));
      bi[i] = pt * S.wb[i];
      const double h = 0.5 * (searching ? beta[i] : beta[i] + s[i]);
      W[i] = h * h;                                              // B.1d
      r[i] = ((act >> i) & 1u) ? 2.0 * log_fast(h) : 0.0;        // ln W_i
      sumW += W[i];
    }
    {
      const double inv = rcp_fast(sumW);
      double wn[NC];
#pragma unroll
      for (int i = 0; i < NC; ++i) wn[i] = W[i] * inv;
      lnphi_fast<NC, KIJ0>(S, sa, bi, wn, lp, Sv, e);
    }
    Zw = e.Z;
    double rmax = 0.0, tm_new = 1.0;
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      r[i] = ((act >> i) & 1u) ? r[i] + lp[i] - w.d[(int64_t)i * N + n] : 0.0;
      rmax = fmax(rmax, fabs(r[i]));
      tm_new = fma(W[i], r[i] - 1.0, tm_new);
    }
    if (!searching) {
      // ---- accept / reject the pending step (B.3) ----
      bool accepted = true;
      if (first) {
        double bn = 0.0;
#pragma unroll
        for (int i = 0; i < NC; ++i) bn = fma(beta[i], beta[i], bn);
        Delta = fmax(1.0, 0.5 * sqrt_fast(bn));
        Delta_cap = 8.0 * Delta;
      } else if (!reeval) {
        const double act_red = tm_new - tm;
        accepted = (act_red < 0.0) || (rmax < rmax_acc);
        if (accepted) {
          if (fabs(pred) > 1.0e-13) {
            const double ratio = fabs(act_red * rcp_fast(pred));
            if (ratio <= 0.25) Delta *= 0.5;
            else if (ratio >= 0.75) Delta = fmin(2.0 * Delta, Delta_cap);
          }
        } else {
          Delta = 0.5 * fmin(Delta, snorm);
          reeval = true;   // next trip re-evaluates at the accepted point (s = 0) and continues from there
        }
      }
      if (!accepted) {
#pragma unroll
        for (int i = 0; i < NC; ++i) s[i] = 0.0;
      } else {
#pragma unroll
        for (int i = 0; i < NC; ++i) { beta[i] += s[i]; s[i] = 0.0; }
        tm = tm_new;
        rmax_acc = rmax;
        first = false;
        reeval = false;
        // ---- convergence / cap, else start the eta search of a new trust-region iteration ----
        if (rmax < o.tol_newton_g) { finish = true; fin_conv = true; }
        else if (tr_it >= o.stab_tr_iters) { finish = true; fin_cap = true; }
        else {
          tr_it++;
          iters++;
          es.start(1.0e-3);
          kept_sn = 0.0;
          searching = true;
        }
      }
    }
    }  // busy
    __syncwarp();
    if (busy && searching) {
      // ---- ONE attempt of the restricted-step sub-problem at es.eta (B.1b): build H + eta I, factor, solve ----
      const MCoef mc = mcoef(e);
      const double isq = rsqrt_fast(sumW);
      double g[NC], st[NC];
#pragma unroll
      for (int i = 0; i < NC; ++i) g[i] = 0.5 * beta[i] * r[i];   // B.2a
#if PTF_TRI_SMEM
      extern __shared__ double ptf_smem[];
      TriSmem<128> Lm{ptf_smem + threadIdx.x};
#else
      double Lm[NT];
#endif
#pragma unroll
      for (int j = 0; j < NC; ++j) {
        const double ej = bi[j] * mc.invB;
        double pj, cj, Dqj;
        mcol(mc, ej - 1.0, Sv[j] - mc.A, pj, cj, Dqj);
        const double hj = 0.5 * beta[j] * isq;
#pragma unroll
        for (int i = j; i < NC; ++i) {
          const double ei = bi[i] * mc.invB;
          const double ui = fma(2.0, Sv[i], -mc.A * ei);
          const double Aij = (KIJ0 ? 1.0 : S.omk[i * NC + j]) * sa[i] * sa[j];
          const double Mij = fma(ei, pj, cj) - fma(Dqj, ui, mc.q2 * (Aij - Sv[i]));
          const double hi_ = 0.5 * beta[i] * isq;
          double hij = hi_ * hj * Mij;                                   // B.2b
          if (i == j) hij += 1.0 + 0.5 * r[i] + es.eta;
          Lm[tri(i, j)] = hij;
        }
      }
      bool good = chol_packed<NC>(Lm, g, st);
      double sn = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i) {
        sn = fma(st[i], st[i], sn);
        if (((act >> i) & 1u) && !(beta[i] + st[i] > 0.0)) good = false;
      }
      sn = sqrt_fast(sn);
      good = good && (sn <= Delta);
      const double eta_used = es.eta;
      if (es.feed(good, sn, Delta, kept_sn)) {
#pragma unroll
        for (int i = 0; i < NC; ++i) s[i] = st[i];
        snorm = sn;
        double sg = 0.0;   // predicted reduction s.g + s.H.s/2 with H s = -g - eta s
#pragma unroll
        for (int i = 0; i < NC; ++i) sg = fma(s[i], g[i], sg);
        pred = 0.5 * sg - 0.5 * eta_used * sn * sn;
        exact = (eta_used == 0.0);
      }
      if (es.phase == 4) { finish = true; fin_cap = true; searching = false; }
      else if (es.phase == 3) {
        searching = false;
        double smax = 0.0;
#pragma unroll
        for (int i = 0; i < NC; ++i) smax = fmax(smax, fabs(s[i]));
        if (exact && smax < o.tol_newton_step) {
          // quadratic-convergence finish: apply the full Newton step and stop
          finish = true;
          fin_conv = true;
          fin_exact = true;
          sumW = 0.0;
#pragma unroll
          for (int i = 0; i < NC; ++i) {
            beta[i] += s[i];
            const double h = 0.5 * beta[i];
            sumW = fma(h, h, sumW);
          }
        }
      }
    }
    __syncwarp();
    if (finish) {
      // beta is stored; k_stab_decide turns it into ln W = 2 ln(beta/2) with all lanes active (TF_BETA)
#pragma unroll
      for (int i = 0; i < NC; ++i) w.lnW[((int64_t)sidx * NC + i) * N + n] = beta[i];
      w.tm[(int64_t)sidx * N + n] = tm;
      w.sumW[(int64_t)sidx * N + n] = sumW;
      w.tflags[(int64_t)sidx * N + n] = (fin_conv ? TF_CONVERGED : 0) | (fin_exact ? TF_EXACT : 0) |
                                        (fin_cap ? TF_CAPPED : 0) | TF_BETA | (iters << TF_ITER_SHIFT);
      busy = false;
    }
  }
}

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
                                                                   const __grid_constant__ Io io, const __grid_constant__ Work w) {
  const int64_t cnt = w.qcount[Q_SPLIT];
  const int64_t pad = (cnt + 31) & ~(int64_t)31;
  const int64_t N = io.N;
  PTF_GRID_STRIDE(idx, pad) {
    const bool in = idx < cnt;
    bool go_newton = false;
    int n = 0;
    if (in) {
      n = w.q_split[idx];
      double z[NC], lnK[NC], x[NC], y[NC], lpx[NC], lpy[NC];
      const double P = io.P[n], T = io.T[n];
      PT3<NC> q;
      { const double iT = rcp_fast(T); q.sT = sqrt_fast(T); q.spt = sqrt_fast(P) * iT; q.pt = P * iT; }
      load_zn<NC>(io, w, n, z);
#pragma unroll
      for (int i = 0; i < NC; ++i) lnK[i] = w.lnK[(int64_t)i * N + n];
      double theta = -1.0e300, r_prev = -1.0;
      double Zx = w.Zxy[n], Zy = w.Zxy[N + n];   // roots of the stage that produced lnK (0: none)
      bool converged = false, failed = false, final_rr = false;
      int k = 0, status = 0;
      // One copy of exp + Rachford-Rice + the two lnphi evaluations: the Rachford-Rice that makes x, y consistent with
      // the converged lnK is the top of one more trip (final_rr).
#pragma unroll 1
      while (true) {
        double mk = 0.0;
#pragma unroll
        for (int i = 0; i < NC; ++i)
          if (z[i] > 0.0) mk = fmax(mk, fabs(lnK[i]));
        if (mk < 1.0e-9) { failed = true; break; }   // trivial collapse
        {
          double K[NC];
#pragma unroll
          for (int i = 0; i < NC; ++i) K[i] = exp_fast(lnK[i]);
          if (!rr_fast<NC>(K, z, theta, x, y)) { failed = true; break; }
        }
        if (final_rr) { converged = true; break; }
        if (o.use_newton && k >= o.split_ss_iters && theta > 0.0 && theta < 1.0) { go_newton = true; break; }
        if (k >= o.ss_cap) { status |= ST_SPLIT_CAP; break; }
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
          if (z[i] > 0.0) { const double nk = lpx[i] - lpy[i]; rk = fmax(rk, fabs(nk - lnK[i])); lnK[i] = nk; }
        ++k;
        if (rk < 1.0e-14) final_rr = true;
        else if (r_prev > 0.0 && rk < o.tol_ss) {
          const double rho = rk * rcp_fast(r_prev);   // linear-convergence error estimate eps = r rho / (1 - rho)
          if (rho < 1.0 && rk * rho < o.tol_ss * (1.0 - rho)) final_rr = true;
        }
        r_prev = rk;
      }
      if (go_newton) {
        // hand-over in the Newton variables: n^V_i = theta y_i (B.4)
        // ... of the MINORITY phase: for theta > 1/2 the roles of the two phases are exchanged (n^L = (1 - theta) x is
        // handed over as "n^V"), so that the majority composition (z - n)/(1 - sum n) is formed without cancellation; G
        // and its stationary point are the same, and the final store restores the phase identity by Z (C23).
        const bool mirror = theta > 0.5;
#pragma unroll
        for (int i = 0; i < NC; ++i) w.lnK[(int64_t)i * N + n] = fmin(mirror ? (1.0 - theta) * x[i] : theta * y[i], z[i]);
        w.iters[n] += k;
        w.status[n] |= status;
        w.Zxy[n] = mirror ? Zy : Zx;
        w.Zxy[N + n] = mirror ? Zx : Zy;
      } else {
        store_split<NC>(io, w, n, z, converged, failed, theta, k, status, x, y, lnK, Zx, Zy);
      }
    }
    queue_push(go_newton, &w.qcount[Q_SPLIT_NEWTON], w.q_split_newton, n);
  }
}

// ---- K6: phase-split trust-region Newton on G (B.4-B.5), persistent warps with lane refill --------
template <int NC, bool KIJ0>
__global__ void __launch_bounds__(128, PTF_NEWTON_MINB) k2_split_newton(const __grid_constant__ Sys<NC> S, const __grid_constant__ Opt o,
                                                       const __grid_constant__ Io io, const __grid_constant__ Work w) {
  constexpr int NT = NC * (NC + 1) / 2;
  constexpr unsigned FULL = 0xffffffffu;
  const int64_t N = io.N;
  const int total = w.qcount[Q_SPLIT_NEWTON];
  int* ticket = &w.qcount[Q_TICKET_SPLIT];
  bool busy = false, exhausted = false, first = true, reeval = false, searching = false, exact = false;
  int n = 0, tr_it = 0, status = 0;
  unsigned act = 0u;
  double spt = 0.0, sT = 0.0, pt = 0.0;
  double nV[NC], s[NC];   // accepted vapour mole numbers (B.4) and pending / best-so-far step
  double G = 0.0, gmax_acc = 0.0, pred = 0.0, Delta = 0.25, snorm = 0.0, Zx = 0.0, Zy = 0.0, kept_sn = 0.0;
  EtaSearch es;
  es.start(1.0);
#pragma unroll
  for (int i = 0; i < NC; ++i) { nV[i] = 0.0; s[i] = 0.0; }

#pragma unroll 1
  while (true) {
    if (__any_sync(FULL, !busy && !exhausted)) {
      const int64_t tk = take_ticket(!busy && !exhausted, ticket);
      if (tk >= 0) {
        if (tk < total) {
          n = w.q_split_newton[tk];
          const double P = io.P[n], T = io.T[n];
          { const double iT = rcp_fast(T); sT = sqrt_fast(T); spt = sqrt_fast(P) * iT; pt = P * iT; }
          act = (unsigned)w.actmask[n];
          // k2_split_ss left n^V = theta y of its last Rachford-Rice here
#pragma unroll
          for (int i = 0; i < NC; ++i) { nV[i] = w.lnK[(int64_t)i * N + n]; s[i] = 0.0; }
          tr_it = 0;
          status = 0;
          first = true;
          reeval = false;
          searching = false;
          Delta = 0.25;
          Zx = w.Zxy[n];
          Zy = w.Zxy[N + n];
          busy = true;
        } else {
          exhausted = true;
        }
      }
    }
    if (!__any_sync(FULL, busy)) break;

    double sa[NC], bi[NC], z[NC], x[NC], y[NC], lp[NC], Sx[NC], Sy[NC], gt[NC];
    double theta = 0.0;
    Eos ex, ey;
    bool finish = false, fin_conv = false;
    if (busy) {
    // ---- evaluate G (eq. 8) and its gradient (B.5a): at n^V + s, or at n^V while an eta search is pending ----
    load_zn<NC>(io, w, n, z);
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      sa[i] = spt * fabs(fma(-S.v[i], sT, S.u[i]));
      bi[i] = pt * S.wb[i];
      const double v = searching ? nV[i] : nV[i] + s[i];
      y[i] = v;
      theta += v;
    }
    {
      const double it = rcp_fast(theta), il = rcp_fast(1.0 - theta);
#pragma unroll
      for (int i = 0; i < NC; ++i) { const double v = y[i]; y[i] = v * it; x[i] = (z[i] - v) * il; }
    }
    ex.Z = Zx;
    lnphi_call<NC, KIJ0>(S, sa, bi, x, lp, Sx, ex);
    Zx = ex.Z;
    double G_new = 0.0, gmax = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      double fx = 0.0;
      if ((act >> i) & 1u) { fx = log_fast(x[i]) + lp[i]; G_new = fma(x[i] * (1.0 - theta), fx, G_new); }
      gt[i] = -fx;
    }
    ey.Z = Zy;
    lnphi_call<NC, KIJ0>(S, sa, bi, y, lp, Sy, ey);
    Zy = ey.Z;
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      if ((act >> i) & 1u) { const double fy = log_fast(y[i]) + lp[i]; G_new = fma(y[i] * theta, fy, G_new); gt[i] += fy; }
      gmax = fmax(gmax, fabs(gt[i]));
    }
    if (!searching) {
      // ---- accept / reject ----
      bool accepted = true;
      if (!first && !reeval) {
        const double act_red = G_new - G;
        accepted = (act_red < 0.0) || (gmax < gmax_acc);
        if (accepted) {
          if (fabs(pred) > 1.0e-13) {
            const double ratio = fabs(act_red * rcp_fast(pred));
            if (ratio <= 0.25) Delta *= 0.5;
            else if (ratio >= 0.75) Delta = fmin(2.0 * Delta, 1.0);
          }
        } else {
          Delta = 0.5 * fmin(Delta, snorm);
          reeval = true;
        }
      }
      if (!accepted) {
#pragma unroll
        for (int i = 0; i < NC; ++i) s[i] = 0.0;
      } else {
#pragma unroll
        for (int i = 0; i < NC; ++i) { nV[i] += s[i]; s[i] = 0.0; }
        G = G_new;
        gmax_acc = gmax;
        first = false;
        reeval = false;
        if (gmax < o.tol_newton_g) { finish = true; fin_conv = true; }
        else if (tr_it >= o.split_tr_iters) { finish = true; status |= ST_SPLIT_CAP; }
        else {
          tr_it++;
          es.start(1.0e-3 * rcp_fast(theta * (1.0 - theta)));
          kept_sn = 0.0;
          searching = true;
        }
      }
    }
    }  // busy
    __syncwarp();
    if (busy && searching) {
      // ---- ONE attempt of the restricted-step sub-problem at es.eta (B.4a) ----
      const MCoef mx = mcoef(ex), my = mcoef(ey);
      const double tt = theta * (1.0 - theta), itt = rcp_fast(tt);
      const double wx = theta * itt, wy = (1.0 - theta) * itt;   // weights of M(x), M(y) in B.5b
      double D[NC], st[NC];
#pragma unroll
      for (int i = 0; i < NC; ++i) D[i] = ((act >> i) & 1u) ? z[i] * rcp_fast(x[i] * y[i]) : 1.0;
#if PTF_TRI_SMEM
      extern __shared__ double ptf_smem[];
      TriSmem<128> Lm{ptf_smem + threadIdx.x};
#else
      double Lm[NT];
#endif
#pragma unroll
      for (int j = 0; j < NC; ++j) {
        const double exj = bi[j] * mx.invB, eyj = bi[j] * my.invB;
        double pxj, cxj, Dqxj, pyj, cyj, Dqyj;
        mcol(mx, exj - 1.0, Sx[j] - mx.A, pxj, cxj, Dqxj);
        mcol(my, eyj - 1.0, Sy[j] - my.A, pyj, cyj, Dqyj);
        const bool aj = (act >> j) & 1u;
#pragma unroll
        for (int i = j; i < NC; ++i) {
          const bool ai = (act >> i) & 1u;
          const double exi = bi[i] * mx.invB, eyi = bi[i] * my.invB;
          const double uxi = fma(2.0, Sx[i], -mx.A * exi), uyi = fma(2.0, Sy[i], -my.A * eyi);
          const double Aij = (KIJ0 ? 1.0 : S.omk[i * NC + j]) * sa[i] * sa[j];
          const double Mx = fma(exi, pxj, cxj) - fma(Dqxj, uxi, mx.q2 * (Aij - Sx[i]));
          const double My = fma(eyi, pyj, cyj) - fma(Dqyj, uyi, my.q2 * (Aij - Sy[i]));
          double hij = fma(wx, Mx, wy * My) - itt;                                  // B.5b
          if (i == j) hij += D[i] * (itt + es.eta);                                // + eta D (B.4a)
          if (!(ai && aj)) hij = (i == j) ? 1.0 : 0.0;
          Lm[tri(i, j)] = hij;
        }
      }
      bool good = chol_packed<NC>(Lm, gt, st);
      double sn = 0.0, sds = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i) {
        sn = fma(st[i], st[i], sn);
        sds = fma(st[i] * st[i], D[i], sds);
        if ((act >> i) & 1u) {
          const double nv = nV[i] + st[i];
          if (!(nv > 0.0) || !(nv < z[i])) good = false;
        }
      }
      sn = sqrt_fast(sn);
      good = good && (sn <= Delta);
      const double eta_used = es.eta;
      if (es.feed(good, sn, Delta, kept_sn)) {
#pragma unroll
        for (int i = 0; i < NC; ++i) s[i] = st[i];
        snorm = sn;
        double sg = 0.0;
#pragma unroll
        for (int i = 0; i < NC; ++i) sg = fma(s[i], gt[i], sg);
        pred = 0.5 * sg - 0.5 * eta_used * sds;
        exact = (eta_used == 0.0);
      }
      if (es.phase == 4) { finish = true; status |= ST_SPLIT_CAP; searching = false; }
      else if (es.phase == 3) {
        searching = false;
        double smax = 0.0;
#pragma unroll
        for (int i = 0; i < NC; ++i) smax = fmax(smax, fabs(s[i]));
        if (exact && smax < o.tol_newton_step) {
          finish = true;
          fin_conv = true;
          theta = 0.0;
#pragma unroll
          for (int i = 0; i < NC; ++i) { nV[i] += s[i]; theta += nV[i]; }
          const double it = rcp_fast(theta), il = rcp_fast(1.0 - theta);
#pragma unroll
          for (int i = 0; i < NC; ++i) { y[i] = nV[i] * it; x[i] = (z[i] - nV[i]) * il; }
        }
      }
    }
    __syncwarp();
    if (finish) {
      double lnK[NC];
      // trivial collapse x = y (max |ln K| < 1e-9): |y/x - 1| is the same test to first order and needs no logarithm
      double mkn = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i)
        if ((act >> i) & 1u) mkn = fmax(mkn, fabs(y[i] - x[i]) * rcp_fast(x[i]));
      const bool trivial = mkn < 1.0e-9;
      if (io.lnK) {
#pragma unroll
        for (int i = 0; i < NC; ++i) lnK[i] = ((act >> i) & 1u) ? log_fast(y[i]) - log_fast(x[i]) : 0.0;
      } else {
#pragma unroll
        for (int i = 0; i < NC; ++i) lnK[i] = 0.0;
      }
      store_split<NC>(io, w, n, z, fin_conv, trivial, theta, tr_it, status, x, y, lnK, Zx, Zy);
      busy = false;
    }
  }
}

}  // namespace ptf
#include "ptflash_newton.cuh"
namespace ptf {

#ifndef PTF_NEWTON_V3
#define PTF_NEWTON_V3 1   // 1: matrix-free rows + shared-memory Cholesky (ptflash_newton.cuh); 0: register-resident k2_* kernels
#endif

template <int NC, bool KIJ0>
int launch_stage2_impl(const Sys<NC>& s, const Opt& o, const Io& io, const Work& w_in, int sms, cudaStream_t st) {
  const int threads = 128;
  auto grid_for = [&](int64_t items) {
    const int64_t need = (items + threads - 1) / threads;
    const int64_t cap = (int64_t)sms * 16;
    return (unsigned)(need < cap ? (need > 0 ? need : 1) : cap);
  };
  const unsigned gN = grid_for(io.N), g2N = grid_for(2 * io.N);
  const unsigned gP = (unsigned)(sms * PTF_NEWTON_MINB);   // persistent refill kernels: a few CTAs per SM pull tickets
  Work w = w_in;
  const size_t tri_bytes = PTF_TRI_SMEM ? (size_t)(NC * (NC + 1) / 2) * threads * sizeof(double) : 0;
  if (tri_bytes > 48 * 1024) {
    cudaFuncSetAttribute(k2_stab_newton<NC, KIJ0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tri_bytes);
    cudaFuncSetAttribute(k2_split_newton<NC, KIJ0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tri_bytes);
  }
#if PTF_NEWTON_V3
  // persistent refill kernels: as many CTAs per SM as registers and shared memory allow (queried once per instantiation)
  const size_t stab_bytes = (size_t)stabn_smem_doubles<NC>() * NEWTON_THREADS * sizeof(double);
  const size_t split_bytes = (size_t)splitn_smem_doubles<NC>() * NEWTON_THREADS * sizeof(double);
  static int stab_cta = 0, split_cta = 0;
  if (stab_cta == 0) {
    cudaFuncSetAttribute(k3_stab_newton<NC, KIJ0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)stab_bytes);
    cudaFuncSetAttribute(k3_split_newton<NC, KIJ0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)split_bytes);
    int a = 0, b = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, k3_stab_newton<NC, KIJ0>, NEWTON_THREADS, stab_bytes);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, k3_split_newton<NC, KIJ0>, NEWTON_THREADS, split_bytes);
    stab_cta = a > 0 ? a : 1;
    split_cta = b > 0 ? b : 1;
  }
#endif
  // optional stage profiling: one event before the first kernel and one after every stage kernel
  cudaEvent_t* ev = (cudaEvent_t*)o.prof_events;
  int nev = 0;
  auto mark = [&]() { if (ev && nev < PTF_MAX_STAGE_EVENTS) cudaEventRecord(ev[nev++], st); };
  mark();
  k_init<NC><<<gN, threads, 0, st>>>(s, o, io, w);
  mark();
  int launches = 1;
  const int passes = (io.flags && io.lnK0) ? 2 : 1;   // pass 1: cold re-flash of mixtures whose skip-stability hint failed
  for (int pass = 0; pass < passes; ++pass) {
    w.pass = pass;
    if (pass) { k_begin_pass2<<<1, 1024, 0, st>>>(w); ++launches; }
    k2_probe<NC, KIJ0><<<gN, threads, 0, st>>>(s, o, io, w);
    mark();
    k2_stab_ss<NC, KIJ0><<<g2N, threads, 0, st>>>(s, o, io, w);
    mark();
#if PTF_NEWTON_V3
    k3_stab_newton<NC, KIJ0><<<(unsigned)(sms * stab_cta), threads, stab_bytes, st>>>(s, o, io, w);
#else
    k2_stab_newton<NC, KIJ0><<<gP, threads, tri_bytes, st>>>(s, o, io, w);
#endif
    mark();
    k_stab_decide<NC><<<gN, threads, 0, st>>>(s, o, io, w);
    mark();
    k2_split_ss<NC, KIJ0><<<gN, threads, 0, st>>>(s, o, io, w);
    mark();
#if PTF_NEWTON_V3
    k3_split_newton<NC, KIJ0><<<(unsigned)(sms * split_cta), threads, split_bytes, st>>>(s, o, io, w);
#else
    k2_split_newton<NC, KIJ0><<<gP, threads, tri_bytes, st>>>(s, o, io, w);
#endif
    k_finalize_counters<<<1, 32, 0, st>>>(w);
    mark();
    launches += 7;
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
