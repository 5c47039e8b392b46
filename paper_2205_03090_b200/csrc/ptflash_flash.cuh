// ptflash_flash.cuh -- per-mixture algorithms built from ptflash_device.cuh:
//   stab_trial   two-sided tangent-plane stability, one start (eq. 3-5; Newton B.1-B.3 PAPER.md:458-492)
//   phase_split  SS of Fig. 1 + trust-region Newton on G (eq. 8, B.4-B.5 PAPER.md:92-97, 494-512)
//   flash_one    the strategy of section 2.2.3 / Fig. 2: Wilson -> 3 probes -> stability -> split
// and the run-to-completion kernel (engine 0): one thread = one mixture from load to store.
#pragma once
#include "ptflash_device.cuh"
#include "ptflash_math.cuh"

namespace ptf {

template <int NC>
struct MixCtx {
  double sa[NC], bi[NC];  // sqrt(A_i), B_i of this (P, T)
  double z[NC], lnz[NC], d[NC];  // normalised feed, ln z, d_i = ln z_i + lnphi_i(z)
};

struct StabRes {
  double tm, tpd;
  int iters;
  bool trivial, capped;
};

// State of one stability trial between its stages (SS -> Newton -> finish).
template <int NC>
struct StabState {
  double lnW[NC];
  double tm, sumW;
  int iters;
  bool converged, stationary_exact, capped;
};

template <int NC>
struct StabEval {
  double W[NC], lp[NC], Sv[NC], r[NC];
  Eos e;
  double sumW, rmax;
};

template <int NC>
__device__ __forceinline__ void stab_eval(const Sys<NC>& S, const MixCtx<NC>& m, const double (&lnW)[NC], StabEval<NC>& v) {
  double w[NC];
  double sumW = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) { v.W[i] = (m.z[i] > 0.0) ? exp(lnW[i]) : 0.0; sumW += v.W[i]; }
  const double inv = 1.0 / sumW;
#pragma unroll
  for (int i = 0; i < NC; ++i) w[i] = v.W[i] * inv;
  lnphi_eval<NC>(S, m.sa, m.bi, w, v.lp, v.Sv, v.e);
  double rmax = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    v.r[i] = (m.z[i] > 0.0) ? lnW[i] + v.lp[i] - m.d[i] : 0.0;
    rmax = fmax(rmax, fabs(v.r[i]));
  }
  v.sumW = sumW;
  v.rmax = rmax;
}

template <int NC>
__device__ __forceinline__ double stab_tm(const StabEval<NC>& v) {
  double t = 1.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) t = fma(v.W[i], v.r[i] - 1.0, t);
  return t;
}

// start: side = +1 vapour-like lnW0 = lnz + lnK, side = -1 liquid-like lnW0 = lnz - lnK
template <int NC>
__device__ __forceinline__ void stab_init(const MixCtx<NC>& m, const double (&lnK)[NC], double side, StabState<NC>& st) {
#pragma unroll
  for (int i = 0; i < NC; ++i) st.lnW[i] = (m.z[i] > 0.0) ? fma(side, lnK[i], m.lnz[i]) : 0.0;
  st.tm = 0.0; st.sumW = 1.0; st.iters = 0;
  st.converged = false; st.stationary_exact = false; st.capped = false;
}

// successive substitution, eq. 5: lnW <- d - lnphi(W / sum W)
template <int NC>
__device__ __noinline__ void stab_ss(const Sys<NC>& S, const Opt& o, const MixCtx<NC>& m, StabState<NC>& st) {
  StabEval<NC> v;
  const int ss_max = o.use_newton ? o.stab_ss_iters : o.ss_cap;
#pragma unroll 1
  for (int k = 0; k < ss_max; ++k) {
    stab_eval<NC>(S, m, st.lnW, v);
    if (v.rmax < o.tol_ss) { st.converged = true; st.tm = stab_tm<NC>(v); st.sumW = v.sumW; return; }
#pragma unroll
    for (int i = 0; i < NC; ++i)
      if (m.z[i] > 0.0) st.lnW[i] = m.d[i] - v.lp[i];
    st.iters++;
  }
  if (!o.use_newton) {
    stab_eval<NC>(S, m, st.lnW, v);
    st.tm = stab_tm<NC>(v);
    st.sumW = v.sumW;
    st.capped = true;
  }
}

// trust-region Newton in beta = 2 sqrt(W) (B.1-B.3 PAPER.md:458-492)
template <int NC>
__device__ __noinline__ void stab_newton(const Sys<NC>& S, const Opt& o, const MixCtx<NC>& m, StabState<NC>& st) {
  StabEval<NC> v;
  double M[NC * NC], H[NC * NC], Lc[NC * NC];
  double g[NC], beta[NC], ones[NC], hi[NC], sstep[NC];
  bool act[NC];
  stab_eval<NC>(S, m, st.lnW, v);
  dlnphi<NC>(S, m.sa, m.bi, v.Sv, v.e, M);
  double tm = stab_tm<NC>(v);
  double bn = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    act[i] = m.z[i] > 0.0;
    beta[i] = 2.0 * sqrt(v.W[i]);
    bn = fma(beta[i], beta[i], bn);
    ones[i] = 1.0;
    hi[i] = 1.0e300;
  }
  double Delta = fmax(1.0, 0.5 * sqrt(bn));
  const double Delta_cap = 8.0 * Delta;
  bool converged = false;
#pragma unroll 1
  for (int it = 0; it < o.stab_tr_iters; ++it) {
    if (v.rmax < o.tol_newton_g) { converged = true; break; }
    st.iters++;
    const double isw = 1.0 / v.sumW;
#pragma unroll 1
    for (int i = 0; i < NC; ++i) {
      const double sq_i = 0.5 * beta[i];  // sqrt(W_i)
      g[i] = act[i] ? sq_i * v.r[i] : 0.0;  // B.2a
#pragma unroll 1
      for (int j = 0; j < NC; ++j) {
        double hij;
        if (act[i] && act[j]) hij = sq_i * (0.5 * beta[j]) * M[i * NC + j] * isw + ((i == j) ? (1.0 + 0.5 * v.r[i]) : 0.0);  // B.2b
        else hij = (i == j) ? 1.0 : 0.0;
        H[i * NC + j] = hij;
      }
    }
    double eta = 0.0, snorm = 0.0;
    if (!tr_subproblem<NC>(H, g, ones, Delta, 1.0e-3, beta, hi, act, sstep, eta, snorm, Lc)) { st.capped = true; break; }
    double smax = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i) smax = fmax(smax, fabs(sstep[i]));
    if (eta == 0.0 && smax < o.tol_newton_step_stab) {
      // quadratic-convergence finish: apply the full Newton step and stop
      double sumW = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i)
        if (act[i]) { beta[i] += sstep[i]; const double h = 0.5 * beta[i]; const double Wi = h * h; st.lnW[i] = log(Wi); sumW += Wi; }
      v.sumW = sumW;
      st.stationary_exact = true;
      converged = true;
      break;
    }
    double pred = 0.0;
#pragma unroll 1
    for (int i = 0; i < NC; ++i) {
      double hs = 0.0;
#pragma unroll 1
      for (int j = 0; j < NC; ++j) hs = fma(H[i * NC + j], sstep[j], hs);
      pred = fma(sstep[i], g[i] + 0.5 * hs, pred);
    }
    double lnW_old[NC];
    const double rmax_old = v.rmax, tm_old = tm;
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      lnW_old[i] = st.lnW[i];
      if (act[i]) { const double h = 0.5 * (beta[i] + sstep[i]); st.lnW[i] = log(h * h); }
    }
    stab_eval<NC>(S, m, st.lnW, v);
    const double tm_new = stab_tm<NC>(v);
    const double act_red = tm_new - tm_old;
    const bool accept = (act_red < 0.0) || (v.rmax < rmax_old);
    if (accept) {
#pragma unroll
      for (int i = 0; i < NC; ++i) beta[i] += sstep[i];
      tm = tm_new;
      if (fabs(pred) > 1.0e-13) {  // B.3
        const double ratio = fabs(act_red / pred);
        if (ratio <= 0.25) Delta *= 0.5;
        else if (ratio >= 0.75) Delta = fmin(2.0 * Delta, Delta_cap);
      }
    } else {
#pragma unroll
      for (int i = 0; i < NC; ++i) st.lnW[i] = lnW_old[i];
      stab_eval<NC>(S, m, st.lnW, v);
      Delta = 0.5 * fmin(Delta, snorm);
    }
    dlnphi<NC>(S, m.sa, m.bi, v.Sv, v.e, M);
  }
  if (!converged) { if (v.rmax < o.tol_newton_g) converged = true; else st.capped = true; }
  st.converged = converged;
  st.tm = tm;
  st.sumW = v.sumW;
}

// trivial test (C7), tm and tpd of the finished trial
template <int NC>
__device__ __forceinline__ void stab_finish(const Opt& o, const MixCtx<NC>& m, const StabState<NC>& st, StabRes& res) {
  double triv = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i)
    if (m.z[i] > 0.0) triv = fmax(triv, fabs(st.lnW[i] - m.lnz[i]));
  res.trivial = triv < o.trivial_tol;
  res.iters = st.iters;
  res.capped = st.capped;
  if (res.trivial) { res.tm = 0.0; res.tpd = 0.0; }
  else {
    res.tm = st.stationary_exact ? (1.0 - st.sumW) : st.tm;
    res.tpd = -log(1.0 - res.tm);  // tm is second-order accurate; tpd = -ln sum W = -ln(1 - tm) at a stationary point
  }
}

// one start, all stages (engine 0)
template <int NC>
__device__ __forceinline__ void stab_trial(const Sys<NC>& S, const Opt& o, const MixCtx<NC>& m, const double (&lnK)[NC],
                                           double side, double (&lnW)[NC], StabRes& res) {
  StabState<NC> st;
  stab_init<NC>(m, lnK, side, st);
  stab_ss<NC>(S, o, m, st);
  if (!st.converged && o.use_newton) stab_newton<NC>(S, o, m, st);
  stab_finish<NC>(o, m, st, res);
#pragma unroll
  for (int i = 0; i < NC; ++i) lnW[i] = st.lnW[i];
}

struct SplitRes {
  double theta;
  int iters, status;
  bool two_phase;
};

// State of one phase split between its stages (SS -> Newton -> finish).
template <int NC>
struct SplitState {
  double lnK[NC];
  double theta;
  int iters, status;
  bool converged, failed, go_newton;
};

// Successive substitution of Fig. 1: theta <- RR(K, z); x, y; lnK <- lnphi(x) - lnphi(y).
// Leaves x, y, theta consistent with st.lnK when it returns with converged or go_newton set.
template <int NC>
__device__ __noinline__ void split_ss(const Sys<NC>& S, const Opt& o, const MixCtx<NC>& m, SplitState<NC>& st,
                                      double (&x)[NC], double (&y)[NC], bool hinted) {
  double K[NC], lpx[NC], lpy[NC], Sv[NC];
  Eos e;
  st.iters = 0; st.status = 0; st.theta = 0.0;
  st.converged = false; st.failed = false; st.go_newton = false;
  double theta = 0.0, r_prev = -1.0;
  int k = 0;
#pragma unroll 1
  while (true) {
    double mk = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i)
      if (m.z[i] > 0.0) mk = fmax(mk, fabs(st.lnK[i]));
    if (mk < o.split_trivial_tol) { st.failed = true; break; }  // trivial collapse (C22)
#pragma unroll
    for (int i = 0; i < NC; ++i) K[i] = exp(st.lnK[i]);
    if (!rr_solve<NC>(K, m.z, theta, x, y)) { st.failed = true; break; }
    if (o.use_newton && k >= o.split_ss_iters && theta > 0.0 && theta < 1.0) { st.go_newton = true; break; }
    if (k >= o.ss_cap) { st.status |= ST_SPLIT_CAP; break; }
    if (hinted && k >= o.hint_ss_cap && !(theta > 0.0 && theta < 1.0)) { st.failed = true; break; }   // reading C21
    lnphi_eval<NC>(S, m.sa, m.bi, x, lpx, Sv, e);
    lnphi_eval<NC>(S, m.sa, m.bi, y, lpy, Sv, e);
    double rk = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i)
      if (m.z[i] > 0.0) { const double nk = lpx[i] - lpy[i]; rk = fmax(rk, fabs(nk - st.lnK[i])); st.lnK[i] = nk; }
    ++k;
    st.iters = k;
    bool conv = false;
    if (rk < 1.0e-14) conv = true;
    else if (r_prev > 0.0 && rk < o.tol_ss) {
      const double rho = rk / r_prev;  // linear-convergence error estimate eps = r rho/(1-rho)
      if (rho < 1.0 && rk * rho / (1.0 - rho) < o.tol_ss) conv = true;
    }
    r_prev = rk;
    if (conv) {
#pragma unroll
      for (int i = 0; i < NC; ++i) K[i] = exp(st.lnK[i]);
      if (!rr_solve<NC>(K, m.z, theta, x, y)) st.failed = true;
      else st.converged = true;
      break;
    }
  }
  st.theta = theta;
}

// Trust-region Newton on the reduced Gibbs energy G (eq. 8) in n^V (B.4-B.5 PAPER.md:494-512).
// Needs x, y, theta = RR(exp(st.lnK), z) on entry with 0 < theta < 1.
template <int NC>
__device__ __noinline__ void split_newton(const Sys<NC>& S, const Opt& o, const MixCtx<NC>& m, SplitState<NC>& st,
                                          double (&x)[NC], double (&y)[NC], bool hinted = false) {
  double Mx[NC * NC], My[NC * NC], H[NC * NC], Lc[NC * NC];
  double nV[NC], gt[NC], D[NC], sstep[NC], lpx[NC], lpy[NC], Sx[NC], Sy[NC];
  Eos ex, ey;
  bool act[NC];
  double theta = st.theta;
#pragma unroll
  for (int i = 0; i < NC; ++i) { act[i] = m.z[i] > 0.0; nV[i] = fmin(theta * y[i], m.z[i]); }
  double G = 0.0, gmax = 0.0;
  auto eval = [&]() {
    theta = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i) theta += nV[i];
    const double it = 1.0 / theta, il = 1.0 / (1.0 - theta);
#pragma unroll
    for (int i = 0; i < NC; ++i) { y[i] = nV[i] * it; x[i] = (m.z[i] - nV[i]) * il; }
    lnphi_eval<NC>(S, m.sa, m.bi, x, lpx, Sx, ex);
    lnphi_eval<NC>(S, m.sa, m.bi, y, lpy, Sy, ey);
    gmax = 0.0;
    G = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      if (act[i]) {
        const double fx = log(x[i]) + lpx[i], fy = log(y[i]) + lpy[i];
        gt[i] = fy - fx;  // B.5a
        G = fma(m.z[i] - nV[i], fx, G);
        G = fma(nV[i], fy, G);  // eq. 8
      } else gt[i] = 0.0;
      gmax = fmax(gmax, fabs(gt[i]));
    }
  };
  eval();
  double Delta = 0.25;
  bool converged = false;
  const int tr_cap = hinted ? min(o.split_tr_iters, o.hint_tr_cap) : o.split_tr_iters;   // reading C21
#pragma unroll 1
  for (int itn = 0; itn < tr_cap; ++itn) {
    // reading C8: a gradient below the target triggers one last full Newton step (applied if admissible), see DESIGN.md
    const bool last = gmax < o.tol_newton_g;
    if (!last) st.iters++;
    dlnphi<NC>(S, m.sa, m.bi, Sx, ex, Mx);
    dlnphi<NC>(S, m.sa, m.bi, Sy, ey, My);
    const double tt = theta * (1.0 - theta), itt = 1.0 / tt;
#pragma unroll 1
    for (int i = 0; i < NC; ++i) {
      D[i] = act[i] ? m.z[i] / (x[i] * y[i]) : 1.0;
#pragma unroll 1
      for (int j = 0; j < NC; ++j) {
        double hij;
        if (act[i] && act[j]) hij = (((i == j) ? D[i] : 0.0) - 1.0 + theta * Mx[i * NC + j] + (1.0 - theta) * My[i * NC + j]) * itt;  // B.5b
        else hij = (i == j) ? 1.0 : 0.0;
        H[i * NC + j] = hij;
      }
    }
    double eta = 0.0, snorm = 0.0;
    if (!tr_subproblem<NC>(H, gt, D, Delta, 1.0e-3 * itt, nV, m.z, act, sstep, eta, snorm, Lc)) {
      if (last) converged = true; else st.status |= ST_SPLIT_CAP;
      break;
    }
    double smax = 0.0;   // largest step relative to the smaller of the two mole numbers n^V_i, n^L_i = z_i - n^V_i
#pragma unroll
    for (int i = 0; i < NC; ++i)
      if (act[i]) smax = fmax(smax, fabs(sstep[i]) / fmin(nV[i], m.z[i] - nV[i]));
    if (last && eta != 0.0) { converged = true; break; }
    if (eta == 0.0 && (last || smax < o.tol_newton_step)) {
      theta = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i) { if (act[i]) nV[i] += sstep[i]; theta += nV[i]; }
      const double it = 1.0 / theta, il = 1.0 / (1.0 - theta);
#pragma unroll
      for (int i = 0; i < NC; ++i) { y[i] = nV[i] * it; x[i] = (m.z[i] - nV[i]) * il; }
      converged = true;
      break;
    }
    double pred = 0.0;
#pragma unroll 1
    for (int i = 0; i < NC; ++i) {
      double hs = 0.0;
#pragma unroll 1
      for (int j = 0; j < NC; ++j) hs = fma(H[i * NC + j], sstep[j], hs);
      pred = fma(sstep[i], gt[i] + 0.5 * hs, pred);
    }
    double nV_old[NC];
    const double G_old = G, gmax_old = gmax;
#pragma unroll
    for (int i = 0; i < NC; ++i) { nV_old[i] = nV[i]; if (act[i]) nV[i] += sstep[i]; }
    eval();
    const double act_red = G - G_old;
    const bool accept = (act_red < 0.0) || (gmax < gmax_old && act_red <= 1.0e-12 * fabs(G_old));
    if (accept) {
      if (fabs(pred) > 1.0e-13) {
        const double ratio = fabs(act_red / pred);
        if (ratio <= 0.25) Delta *= 0.5;
        else if (ratio >= 0.75) Delta = fmin(2.0 * Delta, 1.0);
      }
    } else {
#pragma unroll
      for (int i = 0; i < NC; ++i) nV[i] = nV_old[i];
      eval();
      Delta = 0.5 * fmin(Delta, snorm);
    }
  }
  if (!converged) { if (gmax < o.tol_newton_g) converged = true; else st.status |= ST_SPLIT_CAP; }
  double mkn = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i)
    if (act[i]) { st.lnK[i] = log(y[i]) - log(x[i]); mkn = fmax(mkn, fabs(st.lnK[i])); }
  if (mkn < o.split_trivial_tol) st.failed = true;   // Newton slid into the trivial solution x = y
  st.converged = converged;
  st.theta = theta;
}

template <int NC>
__device__ __forceinline__ void split_finish(const SplitState<NC>& st, SplitRes& res) {
  res.theta = st.theta;
  res.iters = st.iters;
  res.status = st.status;
  res.two_phase = false;
  if (st.failed) { res.status |= ST_SPLIT_FAILED; return; }
  if (st.converged && st.theta > 0.0 && st.theta < 1.0) res.two_phase = true;
  else if (st.converged) res.status |= ST_SPLIT_FAILED;  // converged outside (0,1): reported, not relabelled silently
}

// all stages (engine 0)
template <int NC>
__device__ __forceinline__ void phase_split(const Sys<NC>& S, const Opt& o, const MixCtx<NC>& m, double (&lnK)[NC],
                                            double (&x)[NC], double (&y)[NC], SplitRes& res, bool hinted) {
  SplitState<NC> st;
#pragma unroll
  for (int i = 0; i < NC; ++i) st.lnK[i] = lnK[i];
  split_ss<NC>(S, o, m, st, x, y, hinted);
  if (st.go_newton) split_newton<NC>(S, o, m, st, x, y, hinted);
  split_finish<NC>(st, res);
#pragma unroll
  for (int i = 0; i < NC; ++i) lnK[i] = st.lnK[i];
}

// ------------------------------------------------------------------------------------------------
// Load + validate + normalise the feed.  Returns false for invalid input (O0).
// ------------------------------------------------------------------------------------------------
template <int NC>
__device__ __forceinline__ bool load_feed(const Io& io, int64_t n, double (&z)[NC], double& P, double& T) {
  P = io.P[n];
  T = io.T[n];
  double sz = 0.0;
  bool ok = isfinite(P) && isfinite(T) && P > 0.0 && T > 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    z[i] = io.z[(int64_t)i * io.N + n];
    if (!isfinite(z[i]) || z[i] < 0.0) ok = false;
    sz += z[i];
  }
  if (!ok || !(fabs(sz - 1.0) <= 1.0e-9)) return false;
#pragma unroll
  for (int i = 0; i < NC; ++i) z[i] = z[i] / sz;  // the feed is normalised once (C20)
  return true;
}

// lnz, per-(P,T) setup and d = ln z + lnphi(z)
template <int NC>
__device__ __forceinline__ void feed_reference(const Sys<NC>& S, double P, double T, MixCtx<NC>& m, double& Zfeed) {
#pragma unroll
  for (int i = 0; i < NC; ++i) m.lnz[i] = (m.z[i] > 0.0) ? log(m.z[i]) : 0.0;
  eos_setup<NC>(S, P, T, m.sa, m.bi);
  double lp[NC], Sv[NC];
  Eos e;
  lnphi_eval<NC>(S, m.sa, m.bi, m.z, lp, Sv, e);
  Zfeed = e.Z;
#pragma unroll
  for (int i = 0; i < NC; ++i) m.d[i] = m.lnz[i] + lp[i];
}

// Wilson K (eq. 6) or the caller's lnK0 (flags bit0/bit1); returns true if lnK0 was used
template <int NC>
__device__ __forceinline__ bool start_lnK(const Sys<NC>& S, const Io& io, int64_t n, double P, double T, double (&lnKs)[NC],
                                          int& fl, int& status) {
  wilson_lnK<NC>(S, P, T, lnKs);
  fl = (io.flags && io.lnK0) ? io.flags[n] : 0;
  if (status & ST_WARM_RESTART) fl = 0;   // the caller's hint was dropped for this mixture
  if (!(fl & 3)) return false;
  double l0[NC];
  bool have0 = true;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    l0[i] = io.lnK0[(int64_t)i * io.N + n];
    if (!isfinite(l0[i]) || fabs(l0[i]) > 700.0) have0 = false;
  }
  if (have0) {
#pragma unroll
    for (int i = 0; i < NC; ++i) lnKs[i] = l0[i];
  } else status |= ST_LNK0_REJECTED;
  return have0;
}

// Does the Rachford-Rice equation (eq. 7) for K = exp(lnK) have its root inside 0 < theta < 1?  f_RR is strictly decreasing
// on its window, so this is f_RR(0) > 0 and f_RR(1) < 0 (which also implies that the window exists: some K_i > 1, some < 1).
// Used for the first Rachford-Rice of the probe.
template <int NC>
__device__ __forceinline__ bool rr_root_inside01(const double (&z)[NC], const double (&lnK)[NC]) {
  double f0 = 0.0, f1 = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    const bool a = z[i] > 0.0;
    const double K = exp_fast(a ? lnK[i] : 0.0);   // z_i = 0: K = 1 drops out of both sums
    f0 = fma(z[i], K - 1.0, f0);
    f1 = fma(z[i] * (K - 1.0), rcp_fast(K), f1);
  }
  return f0 > 0.0 && f1 < 0.0;
}

// Probe of section 2.2.3: probe_iters phase-split SS iterations from lnK, then the
// Delta G / tpd(x) / tpd(y) test.  Returns the case (1, 2 or 3); lnK is the probe's iterate.
template <int NC>
__device__ __noinline__ int probe(const Sys<NC>& S, const Opt& o, const MixCtx<NC>& m, double (&lnK)[NC], double& tpd_min,
                                  int& iters) {
  double K[NC], x[NC], y[NC], lpx[NC], lpy[NC], Sv[NC];
  Eos e;
  double theta = 0.0;
  iters = 0;
  if (o.probe_iters == 0) return 2;
#pragma unroll 1
  for (int it = 0; it < o.probe_iters; ++it) {
#pragma unroll
    for (int i = 0; i < NC; ++i) K[i] = exp(lnK[i]);
    if (!rr_solve<NC>(K, m.z, theta, x, y) || !(theta > 0.0) || !(theta < 1.0)) return 1;
    lnphi_eval<NC>(S, m.sa, m.bi, x, lpx, Sv, e);
    lnphi_eval<NC>(S, m.sa, m.bi, y, lpy, Sv, e);
#pragma unroll
    for (int i = 0; i < NC; ++i)
      if (m.z[i] > 0.0) lnK[i] = lpx[i] - lpy[i];
    iters++;
  }
  double tx = 0.0, ty = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    if (x[i] > 0.0) tx = fma(x[i], log(x[i]) + lpx[i] - m.d[i], tx);
    if (y[i] > 0.0) ty = fma(y[i], log(y[i]) + lpy[i] - m.d[i], ty);
  }
  const double dG = (1.0 - theta) * tx + theta * ty;  // reading C5
  const double mn = fmin(dG, fmin(tx, ty));
  if (mn < -o.probe_margin) { tpd_min = mn; return 3; }
  return 2;
}

// Label and K seed from the two finished trials (readings C9, C10).  Returns true if unstable.
template <int NC>
__device__ __forceinline__ bool stab_decide(const Opt& o, const MixCtx<NC>& m, const StabRes& sv, const StabRes& sl,
                                            const double (&lnWv)[NC], const double (&lnWl)[NC], double (&lnK)[NC],
                                            double& tpd_min, int& status) {
  if (sv.capped || sl.capped) status |= ST_STAB_CAP;
  tpd_min = 0.0;
  bool any = false;
  if (!sv.trivial) { tpd_min = sv.tpd; any = true; }
  if (!sl.trivial) { tpd_min = any ? fmin(tpd_min, sl.tpd) : sl.tpd; any = true; }
  const bool unstable = tpd_min < 0.0;
  if (tpd_min != 0.0 && fabs(tpd_min) < o.band) status |= ST_BAND;
  if (unstable) {
    if (sl.tm < sv.tm) {
#pragma unroll
      for (int i = 0; i < NC; ++i) lnK[i] = m.lnz[i] - lnWl[i];
    } else {
#pragma unroll
      for (int i = 0; i < NC; ++i) lnK[i] = lnWv[i] - m.lnz[i];
    }
  }
  return unstable;
}

template <int NC>
__device__ __forceinline__ void store_invalid(const Io& io, int64_t n) {
  const double nan = __longlong_as_double(0x7ff8000000000000LL);
  io.beta[n] = nan;
  io.phase[n] = -1;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    io.x[(int64_t)i * io.N + n] = nan;
    io.y[(int64_t)i * io.N + n] = nan;
    if (io.lnK) io.lnK[(int64_t)i * io.N + n] = nan;
    if (io.dbeta_dK) io.dbeta_dK[(int64_t)i * io.N + n] = nan;
  }
  if (io.iters) io.iters[n] = 0;
  if (io.tpd_min) io.tpd_min[n] = nan;
  if (io.status) io.status[n] = 0;
  if (io.stab_iters) io.stab_iters[n] = 0;
}

// Phase identity of a converged split (reading C23): true if the "y" phase has the smaller Z and must be reported as x.
template <int NC>
__device__ __noinline__ bool phase_swap_by_Z(const Sys<NC>& S, const MixCtx<NC>& m, const double (&x)[NC], const double (&y)[NC]) {
  double lp[NC], Sv[NC];
  Eos ex, ey;
  lnphi_eval<NC>(S, m.sa, m.bi, x, lp, Sv, ex);
  lnphi_eval<NC>(S, m.sa, m.bi, y, lp, Sv, ey);
  return ey.Z < ex.Z;
}

// Final store.  two == false: single phase, x = y = z, beta = 1 iff Z_feed > 1/3 (convention).
template <int NC>
__device__ __forceinline__ void store_result(const Io& io, int64_t n, bool two, double theta, const double (&z)[NC],
                                             const double (&x)[NC], const double (&y)[NC], const double (&lnK)[NC],
                                             double Zfeed, int iters, int status, double tpd_min, int stab_iters,
                                             bool swap) {
  // swap: the split's "y" phase has the smaller compressibility factor, so it is reported as the liquid x
  // (phase identity by Z, reading C23: PAPER.md:445 assigns the smallest root to the liquid, the largest to the vapour)
  io.beta[n] = two ? (swap ? 1.0 - theta : theta) : ((Zfeed > 1.0 / 3.0) ? 1.0 : 0.0);
  io.phase[n] = two ? 2 : 1;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    io.x[(int64_t)i * io.N + n] = two ? (swap ? y[i] : x[i]) : z[i];
    io.y[(int64_t)i * io.N + n] = two ? (swap ? x[i] : y[i]) : z[i];
    if (io.lnK) io.lnK[(int64_t)i * io.N + n] = two ? (swap ? -lnK[i] : lnK[i]) : 0.0;
  }
  if (io.iters) io.iters[n] = iters;
  if (io.tpd_min) io.tpd_min[n] = tpd_min;
  if (io.status) io.status[n] = status;
  if (io.stab_iters) io.stab_iters[n] = stab_iters;
  if (io.dbeta_dK) {
    // eq. 13 PAPER.md:281-286 at the reported solution: with 1 + (K_i - 1) beta = z_i / x_i the two partial derivatives of
    // f_RR (eq. 7) become  d f / d K_i = x_i^2 / z_i  and  d f / d beta = - sum_j (y_j - x_j)^2 / z_j,  so
    // d beta / d K_i = (x_i^2 / z_i) / sum_j (y_j - x_j)^2 / z_j   (unchanged by the x <-> y exchange of C23 up to K -> 1/K,
    // which is why it is formed from the compositions as reported).  Single phase: NaN.
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
    if (two) {
      double den = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i) {
        const double dxy = y[i] - x[i];
        if (z[i] > 0.0) den = fma(dxy * dxy, 1.0 / z[i], den);
      }
      const double iden = 1.0 / den;
#pragma unroll
      for (int i = 0; i < NC; ++i) {
        const double xr = swap ? y[i] : x[i];
        io.dbeta_dK[(int64_t)i * io.N + n] = (z[i] > 0.0) ? xr * xr / z[i] * iden : 0.0;
      }
    } else {
#pragma unroll
      for (int i = 0; i < NC; ++i) io.dbeta_dK[(int64_t)i * io.N + n] = nan;
    }
  }
}

// Stability-only mode (PTFLASH_OPT_STABILITY_ONLY; "determine stability (no need for phase split
// calculations)"): the store of a mixture labelled UNSTABLE -- phase = 2, x = y = z, beta = NaN (not computed), lnK = the K
// that would seed the phase split (probe iterate, caller's estimate, or the stability trial's).
template <int NC>
__device__ __forceinline__ void store_unstable_label(const Io& io, int64_t n, const double (&z)[NC], const double (&lnK)[NC],
                                                     int iters, int status, double tpd_min, int stab_iters) {
  const double nan = __longlong_as_double(0x7ff8000000000000LL);
  io.beta[n] = nan;
  io.phase[n] = 2;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    io.x[(int64_t)i * io.N + n] = z[i];
    io.y[(int64_t)i * io.N + n] = z[i];
    if (io.lnK) io.lnK[(int64_t)i * io.N + n] = (z[i] > 0.0) ? lnK[i] : 0.0;
    if (io.dbeta_dK) io.dbeta_dK[(int64_t)i * io.N + n] = nan;
  }
  if (io.iters) io.iters[n] = iters;
  if (io.tpd_min) io.tpd_min[n] = tpd_min;
  if (io.status) io.status[n] = status;
  if (io.stab_iters) io.stab_iters[n] = stab_iters;
}

// ------------------------------------------------------------------------------------------------
// Whole flash of mixture n, run to completion by one thread (engine 0).
// ------------------------------------------------------------------------------------------------
template <int NC>
__device__ void flash_one(const Sys<NC>& S, const Opt& o, const Io& io, int64_t n) {
  MixCtx<NC> m;
  double P, T, Zf;
  if (!load_feed<NC>(io, n, m.z, P, T)) { store_invalid<NC>(io, n); return; }
  feed_reference<NC>(S, P, T, m, Zf);
  const double nan = __longlong_as_double(0x7ff8000000000000LL);
  int status = 0, iters = 0, stab_iters = 0;
  bool two = false;
  double theta = 0.0, tpd_min = 0.0;
  double x[NC], y[NC], lnK[NC];
  // attempt 0 honours the caller's lnK0 / skip-stability hint; attempt 1 (only after a failed skip-stability split)
  // is the plain cold flash (status ST_WARM_RESTART makes start_lnK ignore the hint)
#pragma unroll 1
  for (int attempt = 0; attempt < 2; ++attempt) {
    int fl = 0, it_probe = 0;
    double lnKs[NC];
    const bool have0 = start_lnK<NC>(S, io, n, P, T, lnKs, fl, status);
    const bool skip_stab = have0 && (fl & 1);
#pragma unroll
    for (int i = 0; i < NC; ++i) lnK[i] = lnKs[i];
    bool unstable = false;
    tpd_min = 0.0;
    if (!skip_stab) {
      const int pcase = probe<NC>(S, o, m, lnK, tpd_min, it_probe);
      iters += it_probe;
      if (pcase == 3) unstable = true;
      else {
        // stability with the Wilson / caller K (reading C19), both starts
        double lnWv[NC], lnWl[NC];
        StabRes sv, sl;
        stab_trial<NC>(S, o, m, lnKs, +1.0, lnWv, sv);
        stab_trial<NC>(S, o, m, lnKs, -1.0, lnWl, sl);
        stab_iters = sv.iters + sl.iters;
        unstable = stab_decide<NC>(o, m, sv, sl, lnWv, lnWl, lnK, tpd_min, status);
      }
    } else {
      unstable = true;
      tpd_min = nan;
    }
    if (o.stability_only) {
      if (unstable) { store_unstable_label<NC>(io, n, m.z, lnK, iters, status, tpd_min, stab_iters); return; }
      break;
    }
    int split_status = 0;
    if (unstable) {
      SplitRes sp;
      phase_split<NC>(S, o, m, lnK, x, y, sp, skip_stab);
      iters += sp.iters;
      split_status = sp.status;
      two = sp.two_phase;
      theta = sp.theta;
      if (!two) split_status |= ST_SPLIT_FAILED;
    }
    if (!two && skip_stab) { status |= ST_WARM_RESTART; continue; }   // drop the hint, flash again from Wilson
    status |= split_status;
    break;
  }
  const bool swap = two && phase_swap_by_Z<NC>(S, m, x, y);
  store_result<NC>(io, n, two, theta, m.z, x, y, lnK, Zf, iters, status, tpd_min, stab_iters, swap);
}

template <int NC>
__global__ void __launch_bounds__(128) flash_mono_kernel(const __grid_constant__ Sys<NC> S, const __grid_constant__ Opt o,
                                                         const __grid_constant__ Io io) {
  const int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (n < io.N) flash_one<NC>(S, o, io, n);
}

}  // namespace ptf
