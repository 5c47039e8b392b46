// ptflash_flash.cuh -- per-mixture algorithms built from ptflash_device.cuh:
//   stab_trial   two-sided tangent-plane stability, one start (eq. 3-5; Newton B.1-B.3 PAPER.md:458-492)
//   phase_split  SS of Fig. 1 + trust-region Newton on G (eq. 8, B.4-B.5 PAPER.md:92-97, 494-512)
//   flash_one    the strategy of section 2.2.3 / Fig. 2: Wilson -> 3 probes -> stability -> split
// and the run-to-completion kernel (engine 0): one thread = one mixture from load to store.
#pragma once
#include "ptflash_device.cuh"

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

// ------------------------------------------------------------------------------------------------
// Stability, one start: side = +1 vapour-like lnW0 = lnz + lnK, side = -1 liquid-like lnW0 = lnz - lnK.
// ------------------------------------------------------------------------------------------------
template <int NC>
__device__ __noinline__ void stab_trial(const Sys<NC>& S, const Opt& o, const MixCtx<NC>& m, const double (&lnK)[NC],
                                        double side, double (&lnW)[NC], StabRes& res) {
  double W[NC], w[NC], lp[NC], Sv[NC], r[NC];
  Eos e;
  double sumW = 0.0, rmax = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) lnW[i] = (m.z[i] > 0.0) ? fma(side, lnK[i], m.lnz[i]) : 0.0;
  res.iters = 0;
  res.capped = false;
  bool converged = false, stationary_exact = false;

  auto eval = [&]() {
    sumW = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i) { W[i] = (m.z[i] > 0.0) ? exp(lnW[i]) : 0.0; sumW += W[i]; }
    const double inv = 1.0 / sumW;
#pragma unroll
    for (int i = 0; i < NC; ++i) w[i] = W[i] * inv;
    lnphi_eval<NC>(S, m.sa, m.bi, w, lp, Sv, e);
    rmax = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      r[i] = (m.z[i] > 0.0) ? lnW[i] + lp[i] - m.d[i] : 0.0;
      rmax = fmax(rmax, fabs(r[i]));
    }
  };
  auto tm_full = [&]() {
    double t = 1.0;
#pragma unroll
    for (int i = 0; i < NC; ++i) t = fma(W[i], r[i] - 1.0, t);
    return t;
  };

  const int ss_max = o.use_newton ? o.stab_ss_iters : o.ss_cap;
#pragma unroll 1
  for (int k = 0; k < ss_max; ++k) {
    eval();
    if (rmax < o.tol_ss) { converged = true; break; }
#pragma unroll
    for (int i = 0; i < NC; ++i)
      if (m.z[i] > 0.0) lnW[i] = m.d[i] - lp[i];  // eq. 5
    res.iters++;
  }
  double tm = 0.0;
  if (converged) {
    tm = tm_full();
  } else if (!o.use_newton) {
    eval();
    tm = tm_full();
    res.capped = true;
  } else {
    // ---- trust-region Newton in beta = 2 sqrt(W) (B.1-B.3) ----
    double M[NC * NC], H[NC * NC], Lc[NC * NC];
    double g[NC], beta[NC], ones[NC], hi[NC], sstep[NC];
    bool act[NC];
    eval();
    dlnphi<NC>(S, m.sa, m.bi, Sv, e, M);
    tm = tm_full();
    double bn = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      act[i] = m.z[i] > 0.0;
      beta[i] = 2.0 * sqrt(W[i]);
      bn = fma(beta[i], beta[i], bn);
      ones[i] = 1.0;
      hi[i] = 1.0e300;
    }
    double Delta = fmax(1.0, 0.5 * sqrt(bn));
    const double Delta_cap = 8.0 * Delta;
#pragma unroll 1
    for (int it = 0; it < o.stab_tr_iters; ++it) {
      if (rmax < o.tol_newton_g) { converged = true; break; }
      res.iters++;
      const double isw = 1.0 / sumW;
#pragma unroll 1
      for (int i = 0; i < NC; ++i) {
        const double sq_i = 0.5 * beta[i];  // sqrt(W_i)
        g[i] = act[i] ? sq_i * r[i] : 0.0;  // B.2a
#pragma unroll 1
        for (int j = 0; j < NC; ++j) {
          double hij;
          if (act[i] && act[j]) hij = sq_i * (0.5 * beta[j]) * M[i * NC + j] * isw + ((i == j) ? (1.0 + 0.5 * r[i]) : 0.0);  // B.2b
          else hij = (i == j) ? 1.0 : 0.0;
          H[i * NC + j] = hij;
        }
      }
      double eta = 0.0, snorm = 0.0;
      if (!tr_subproblem<NC>(H, g, ones, Delta, 1.0e-3, beta, hi, act, sstep, eta, snorm, Lc)) { res.capped = true; break; }
      double smax = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i) smax = fmax(smax, fabs(sstep[i]));
      if (eta == 0.0 && smax < o.tol_newton_step) {
        // quadratic-convergence finish: apply the full Newton step and stop
        sumW = 0.0;
#pragma unroll
        for (int i = 0; i < NC; ++i)
          if (act[i]) { beta[i] += sstep[i]; const double h = 0.5 * beta[i]; W[i] = h * h; lnW[i] = log(W[i]); sumW += W[i]; }
        stationary_exact = true;
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
      const double rmax_old = rmax, tm_old = tm;
#pragma unroll
      for (int i = 0; i < NC; ++i) {
        lnW_old[i] = lnW[i];
        if (act[i]) { const double h = 0.5 * (beta[i] + sstep[i]); lnW[i] = log(h * h); }
      }
      eval();
      const double tm_new = tm_full();
      const double act_red = tm_new - tm_old;
      const bool accept = (act_red < 0.0) || (rmax < rmax_old);
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
        for (int i = 0; i < NC; ++i) lnW[i] = lnW_old[i];
        eval();
        Delta = 0.5 * fmin(Delta, snorm);
      }
      dlnphi<NC>(S, m.sa, m.bi, Sv, e, M);
    }
    if (!converged) { if (rmax < o.tol_newton_g) converged = true; else res.capped = true; }
  }
  double triv = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i)
    if (m.z[i] > 0.0) triv = fmax(triv, fabs(lnW[i] - m.lnz[i]));
  res.trivial = triv < o.trivial_tol;
  if (res.trivial) { res.tm = 0.0; res.tpd = 0.0; }
  else {
    res.tm = stationary_exact ? (1.0 - sumW) : tm;
    res.tpd = -log(1.0 - res.tm);  // tm is second-order accurate; tpd = -ln sumW = -ln(1 - tm) at a stationary point
  }
}

struct SplitRes {
  double theta;
  int iters, status;
  bool two_phase;
};

// ------------------------------------------------------------------------------------------------
// Phase split from lnK.
// ------------------------------------------------------------------------------------------------
template <int NC>
__device__ __noinline__ void phase_split(const Sys<NC>& S, const Opt& o, const MixCtx<NC>& m, double (&lnK)[NC],
                                         double (&x)[NC], double (&y)[NC], SplitRes& res) {
  double K[NC], lpx[NC], lpy[NC], Sx[NC], Sy[NC];
  Eos ex, ey;
  res.iters = 0;
  res.status = 0;
  res.two_phase = false;
  double theta = 0.0, r_prev = -1.0;
  bool converged = false, failed = false, go_newton = false;
  int k = 0;
#pragma unroll 1
  while (true) {
    double mk = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i)
      if (m.z[i] > 0.0) mk = fmax(mk, fabs(lnK[i]));
    if (mk < 1.0e-9) { failed = true; break; }
#pragma unroll
    for (int i = 0; i < NC; ++i) K[i] = exp(lnK[i]);
    if (!rr_solve<NC>(K, m.z, theta, x, y)) { failed = true; break; }
    if (o.use_newton && k >= o.split_ss_iters && theta > 0.0 && theta < 1.0) { go_newton = true; break; }
    if (k >= o.ss_cap) { res.status |= ST_SPLIT_CAP; break; }
    lnphi_eval<NC>(S, m.sa, m.bi, x, lpx, Sx, ex);
    lnphi_eval<NC>(S, m.sa, m.bi, y, lpy, Sy, ey);
    double rk = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i)
      if (m.z[i] > 0.0) { const double nk = lpx[i] - lpy[i]; rk = fmax(rk, fabs(nk - lnK[i])); lnK[i] = nk; }
    ++k;
    res.iters = k;
    if (rk < 1.0e-14) converged = true;
    else if (r_prev > 0.0 && rk < o.tol_ss) {
      const double rho = rk / r_prev;
      if (rho < 1.0 && rk * rho / (1.0 - rho) < o.tol_ss) converged = true;
    }
    r_prev = rk;
    if (converged) {
#pragma unroll
      for (int i = 0; i < NC; ++i) K[i] = exp(lnK[i]);
      if (!rr_solve<NC>(K, m.z, theta, x, y)) { failed = true; converged = false; }
      break;
    }
  }

  if (go_newton) {
    // ---- trust-region Newton on G in n^V (B.4-B.5) ----
    double Mx[NC * NC], My[NC * NC], H[NC * NC], Lc[NC * NC];
    double nV[NC], gt[NC], D[NC], sstep[NC];
    bool act[NC];
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
#pragma unroll 1
    for (int itn = 0; itn < o.split_tr_iters; ++itn) {
      if (gmax < o.tol_newton_g) { converged = true; break; }
      res.iters++;
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
      if (!tr_subproblem<NC>(H, gt, D, Delta, 1.0e-3 * itt, nV, m.z, act, sstep, eta, snorm, Lc)) { res.status |= ST_SPLIT_CAP; break; }
      double smax = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i) smax = fmax(smax, fabs(sstep[i]));
      if (eta == 0.0 && smax < o.tol_newton_step) {
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
      const bool accept = (act_red < 0.0) || (gmax < gmax_old);
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
    if (!converged) { if (gmax < o.tol_newton_g) converged = true; else res.status |= ST_SPLIT_CAP; }
#pragma unroll
    for (int i = 0; i < NC; ++i)
      if (act[i]) lnK[i] = log(y[i]) - log(x[i]);
  }
  res.theta = theta;
  if (failed) { res.status |= ST_SPLIT_FAILED; return; }
  if (converged && theta > 0.0 && theta < 1.0) res.two_phase = true;
  else if (converged) res.status |= ST_SPLIT_FAILED;
}

// ------------------------------------------------------------------------------------------------
// Load + validate + per-(P,T) setup + d = ln z + lnphi(z).  Returns false for invalid input.
// ------------------------------------------------------------------------------------------------
template <int NC>
__device__ __forceinline__ bool load_mixture(const Sys<NC>& S, const Io& io, int64_t n, MixCtx<NC>& m, double& P, double& T,
                                             double& Zfeed) {
  P = io.P[n];
  T = io.T[n];
  double zin[NC], sz = 0.0;
  bool ok = isfinite(P) && isfinite(T) && P > 0.0 && T > 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    zin[i] = io.z[(int64_t)i * io.N + n];
    if (!isfinite(zin[i]) || zin[i] < 0.0) ok = false;
    sz += zin[i];
  }
  if (!ok || !(fabs(sz - 1.0) <= 1.0e-9)) return false;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    m.z[i] = zin[i] / sz;
    m.lnz[i] = (m.z[i] > 0.0) ? log(m.z[i]) : 0.0;
  }
  eos_setup<NC>(S, P, T, m.sa, m.bi);
  double lp[NC], Sv[NC];
  Eos e;
  lnphi_eval<NC>(S, m.sa, m.bi, m.z, lp, Sv, e);
  Zfeed = e.Z;
#pragma unroll
  for (int i = 0; i < NC; ++i) m.d[i] = m.lnz[i] + lp[i];
  return true;
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
  }
  if (io.iters) io.iters[n] = 0;
  if (io.tpd_min) io.tpd_min[n] = nan;
  if (io.status) io.status[n] = 0;
  if (io.stab_iters) io.stab_iters[n] = 0;
}

// ------------------------------------------------------------------------------------------------
// Whole flash of mixture n, run to completion by one thread (engine 0).
// ------------------------------------------------------------------------------------------------
template <int NC>
__device__ void flash_one(const Sys<NC>& S, const Opt& o, const Io& io, int64_t n) {
  MixCtx<NC> m;
  double P, T, Zf;
  if (!load_mixture<NC>(S, io, n, m, P, T, Zf)) { store_invalid<NC>(io, n); return; }
  const double nan = __longlong_as_double(0x7ff8000000000000LL);
  int status = 0, iters = 0, stab_iters = 0;

  double lnKs[NC], lnK[NC];
  wilson_lnK<NC>(S, P, T, lnKs);
  const int fl = (io.flags && io.lnK0) ? io.flags[n] : 0;
  bool have0 = false;
  if (fl & 3) {
    double l0[NC];
    have0 = true;
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      l0[i] = io.lnK0[(int64_t)i * io.N + n];
      if (!isfinite(l0[i]) || fabs(l0[i]) > 700.0) have0 = false;
    }
    if (have0) {
#pragma unroll
      for (int i = 0; i < NC; ++i) lnKs[i] = l0[i];
    } else status |= ST_LNK0_REJECTED;
  }
  const bool skip_stab = have0 && (fl & 1);
#pragma unroll
  for (int i = 0; i < NC; ++i) lnK[i] = lnKs[i];

  bool unstable = false;
  double tpd_min = 0.0;
  double x[NC], y[NC];
  if (!skip_stab) {
    // ---- probe: 3 phase-split SS iterations ----
    double K[NC], lpx[NC], lpy[NC], Sv[NC];
    Eos e;
    double theta = 0.0;
    int pcase = 0;
#pragma unroll 1
    for (int it = 0; it < o.probe_iters; ++it) {
#pragma unroll
      for (int i = 0; i < NC; ++i) K[i] = exp(lnK[i]);
      if (!rr_solve<NC>(K, m.z, theta, x, y) || !(theta > 0.0) || !(theta < 1.0)) { pcase = 1; break; }
      lnphi_eval<NC>(S, m.sa, m.bi, x, lpx, Sv, e);
      lnphi_eval<NC>(S, m.sa, m.bi, y, lpy, Sv, e);
#pragma unroll
      for (int i = 0; i < NC; ++i)
        if (m.z[i] > 0.0) lnK[i] = lpx[i] - lpy[i];
      iters++;
    }
    if (o.probe_iters == 0) pcase = 2;
    if (pcase == 0) {
      double tx = 0.0, ty = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i) {
        if (x[i] > 0.0) tx = fma(x[i], log(x[i]) + lpx[i] - m.d[i], tx);
        if (y[i] > 0.0) ty = fma(y[i], log(y[i]) + lpy[i] - m.d[i], ty);
      }
      const double dG = (1.0 - theta) * tx + theta * ty;
      const double mn = fmin(dG, fmin(tx, ty));
      if (mn < -o.probe_margin) { pcase = 3; unstable = true; tpd_min = mn; }
      else pcase = 2;
    }
    if (pcase != 3) {
      // ---- stability with the Wilson / caller K ----
      double lnWv[NC], lnWl[NC];
      StabRes sv, sl;
      stab_trial<NC>(S, o, m, lnKs, +1.0, lnWv, sv);
      stab_trial<NC>(S, o, m, lnKs, -1.0, lnWl, sl);
      stab_iters = sv.iters + sl.iters;
      if (sv.capped || sl.capped) status |= ST_STAB_CAP;
      tpd_min = 0.0;
      bool any = false;
      if (!sv.trivial) { tpd_min = sv.tpd; any = true; }
      if (!sl.trivial) { tpd_min = any ? fmin(tpd_min, sl.tpd) : sl.tpd; any = true; }
      unstable = tpd_min < 0.0;
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
    }
  } else {
    unstable = true;
    tpd_min = nan;
  }

  bool two = false;
  double beta = 0.0;
  if (unstable) {
    SplitRes sp;
    phase_split<NC>(S, o, m, lnK, x, y, sp);
    iters += sp.iters;
    status |= sp.status;
    if (sp.two_phase) { two = true; beta = sp.theta; }
    else status |= ST_SPLIT_FAILED;
  }
  if (!two) {
    beta = (Zf > 1.0 / 3.0) ? 1.0 : 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i) { x[i] = m.z[i]; y[i] = m.z[i]; lnK[i] = 0.0; }
  }
  io.beta[n] = beta;
  io.phase[n] = two ? 2 : 1;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    io.x[(int64_t)i * io.N + n] = x[i];
    io.y[(int64_t)i * io.N + n] = y[i];
    if (io.lnK) io.lnK[(int64_t)i * io.N + n] = lnK[i];
  }
  if (io.iters) io.iters[n] = iters;
  if (io.tpd_min) io.tpd_min[n] = tpd_min;
  if (io.status) io.status[n] = status;
  if (io.stab_iters) io.stab_iters[n] = stab_iters;
}

template <int NC>
__global__ void __launch_bounds__(128) flash_mono_kernel(const __grid_constant__ Sys<NC> S, const __grid_constant__ Opt o,
                                                         const __grid_constant__ Io io) {
  const int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (n < io.N) flash_one<NC>(S, o, io, n);
}

}  // namespace ptf
