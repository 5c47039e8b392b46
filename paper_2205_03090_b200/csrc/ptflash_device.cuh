// ptflash_device.cuh -- fp64 device functions of the batched SRK two-phase flash for sm_100a.
//
// One thread owns one mixture (or one stability trial); the component count NC is a template parameter
// (2..16) so that every per-component loop is fully unrolled and the per-component state lives in
// registers.  Component constants arrive as a __grid_constant__ kernel parameter (constant bank), so with
// unrolled loops they are immediate constant-bank operands of the DFMA instructions.
//
// The operations are the paper's (PAPER.md = /root/reference/PAPER.md):
//   eos_setup      A.2d-g  PAPER.md:420-427   (dimensionless A_i, B_i; R cancels)
//   pick_root      A.3-A.5 PAPER.md:431-445   (cubic in Z, admissible roots Z > B, minimum Gibbs energy)
//   lnphi_eval     A.2a-c, A.6 PAPER.md:412-418, 447-450
//   dlnphi         PAPER.md:452 (explicit composition derivative; formula derived in DESIGN.md section 3)
//   wilson_lnK     eq. 6
//   rr_solve       eq. 7, App. C
//   tr_subproblem  B.1b / B.4a PAPER.md:468, 502 (restricted step)
// This file shares nothing with oracle/ (the CPU oracle is test infrastructure).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace ptf {

// ------------------------------------------------------------------------------------------------
// parameter blocks
// ------------------------------------------------------------------------------------------------
struct Opt {
  double tol_ss, tol_newton_g, tol_newton_step, tol_newton_step_stab, probe_margin, trivial_tol, band, split_trivial_tol;
  double triv_lo, triv_hi;   // exp(-trivial_tol), exp(+trivial_tol): |ln W_i - ln z_i| < trivial_tol  <=>  triv_lo < W_i / z_i < triv_hi
  int probe_iters, stab_ss_iters, stab_tr_iters, split_ss_iters, split_tr_iters, use_newton, ss_cap, hint_ss_cap, hint_tr_cap;
  int stability_only;   // 1: stop after the label; no phase split
  int early_split_ss;   // 1: the SS stage of the probe-found splits starts right after the probe (PTFLASH_OPT_EARLY_SPLIT_SS)
  int hint_eta_search;  // 1: splits entered through a skip-stability hint run the eta search of B.4a (the oracle's path)
  // host only: cudaEvent_t[PTF_MAX_STAGE_EVENTS] recorded between the stage kernels when stage profiling is on (else null)
  void* prof_events;
  int* prof_count;   // host only: number of events recorded by the last launch
  // host only: second stream of the handle and two events (fork / join) so that the phase split of the mixtures the probe
  // already found unstable runs concurrently with the stability analysis of the others (null: everything on one stream)
  void *aux_stream, *ev_fork, *ev_join;
  // host only: third stream for the crawlers of the phase split (stage2: split part 2) with its three events
  void *aux2_stream, *ev_c0, *ev_c1, *ev_cjoin, *ev_probe;
  // host only: per-handle cache of the resident-CTA counts of the persistent kernels (0 = not yet queried); a handle is
  // bound to one device and one component system, so the occupancy query runs once per handle
  int* cta_cache;
};
#define PTF_MAX_STAGE_EVENTS 24

// Per-system constants, precomputed on the host in ptflash_create:
//   sqrt(A_i) = sqrt(P)/T * |u_i - v_i sqrt(T)|,  u_i = sqrt(0.42748/Pc_i) Tc_i (1+m_i),  v_i = sqrt(0.42748/Pc_i) sqrt(Tc_i) m_i
//   B_i       = (P/T) * wb_i,                     wb_i = 0.08664 Tc_i / Pc_i
//   ln K_i    = lnpc_i - ln P + wil_i (1 - tc_i/T), wil_i = 5.373 (1 + omega_i)
//   omk[i][j] = 1 - k_ij
template <int NC>
struct Sys {
  double u[NC], v[NC], wb[NC], lnpc[NC], wil[NC], tc[NC];
  double omk[NC * NC];
  int kij_zero;
};

struct Io {
  int64_t N;
  const double *z, *P, *T, *lnK0;
  const uint8_t* flags;
  double *beta, *x, *y;
  int32_t *phase, *iters;
  double *tpd_min, *lnK;
  int32_t *status, *stab_iters;
  double* dbeta_dK;   // optional [nc][N]: d beta / d K_i at the solution (eq. 13)
};

enum : int { ST_STAB_CAP = 1, ST_SPLIT_CAP = 2, ST_BAND = 4, ST_SPLIT_FAILED = 8, ST_LNK0_REJECTED = 32, ST_WARM_RESTART = 64,
              ST_INTERNAL_SKIPPED = 128 /* workspace only: mixture entered the split through PTFLASH_FLAG_SKIP_STABILITY */ };

struct Eos {
  double A, B, Z, L, q, lnZmB;
};

// ------------------------------------------------------------------------------------------------
// A.2d-g: per-mixture sqrt(A_i) and B_i from (P, T)
// ------------------------------------------------------------------------------------------------
template <int NC>
__device__ __forceinline__ void eos_setup(const Sys<NC>& S, double P, double T, double (&sa)[NC], double (&bi)[NC]) {
  const double sT = sqrt(T);
  const double invT = 1.0 / T;
  const double spt = sqrt(P) * invT;
  const double pt = P * invT;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    sa[i] = spt * fabs(fma(-S.v[i], sT, S.u[i]));
    bi[i] = pt * S.wb[i];
  }
}

// ------------------------------------------------------------------------------------------------
// Cubic A.3: f(Z) = Z^3 - Z^2 + rho1 Z - rho0.  Monotone Newton from the side with the right curvature
// (inflection at Z = 1/3; f(B) = -2B^2 < 0; f(1+B) = A > 0), deflation A.5, polish, admissible roots
// Z > B, minimum-Gibbs choice between the smallest and the largest admissible root (tie -> smaller Z).
// Returns Z and the two logarithms of the chosen root that A.6 needs.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double cub_f(double Z, double r1, double r0) { return fma(fma(Z - 1.0, Z, r1), Z, -r0); }
__device__ __forceinline__ double cub_df(double Z, double r1) { return fma(fma(3.0, Z, -2.0), Z, r1); }

__device__ __forceinline__ double cub_polish(double Z, double r1, double r0) {
#pragma unroll 1
  for (int k = 0; k < 3; ++k) {
    const double f = cub_f(Z, r1, r0), df = cub_df(Z, r1);
    if (df == 0.0) break;
    const double Zn = Z - f / df;
    if (!(fabs(cub_f(Zn, r1, r0)) < fabs(f))) break;
    Z = Zn;
  }
  return Z;
}

static __device__ __noinline__ double pick_root(double A, double B, double& lnZmB, double& L) {
  const double r0 = A * B, r1 = A - B * (1.0 + B);
  const double third = 1.0 / 3.0;
  const bool up = (B < third) && (cub_f(third, r1, r0) > 0.0);
  double Z = up ? B : 1.0 + B;
#pragma unroll 1
  for (int k = 0; k < 100; ++k) {
    const double df = cub_df(Z, r1);
    if (!(df > 0.0)) break;
    const double Zn = Z - cub_f(Z, r1, r0) / df;
    if (up ? !(Zn > Z) : !(Zn < Z)) break;
    Z = Zn;
  }
  double zmin = Z, zmax = Z;
  const double p = Z - 1.0, q = fma(p, Z, r1);
  const double disc = fma(p, p, -4.0 * q);
  if (disc >= 0.0) {
    const double sq = sqrt(disc);
    const double t = (p >= 0.0) ? -0.5 * (p + sq) : 0.5 * (sq - p);
    double ra = t, rb = (t != 0.0) ? q / t : -p - t;
    ra = cub_polish(ra, r1, r0);
    rb = cub_polish(rb, r1, r0);
    if (ra > B) { zmin = fmin(zmin, ra); zmax = fmax(zmax, ra); }
    if (rb > B) { zmin = fmin(zmin, rb); zmax = fmax(zmax, rb); }
  }
  const double AoB = A / B;
  double lz = log(zmin - B), ll = log1p(B / zmin);
  if (zmax != zmin) {
    const double lz2 = log(zmax - B), ll2 = log1p(B / zmax);
    const double gl = zmin - 1.0 - lz - AoB * ll;
    const double gv = zmax - 1.0 - lz2 - AoB * ll2;
    if (gv < gl) { zmin = zmax; lz = lz2; ll = ll2; }
  }
  lnZmB = lz;
  L = ll;
  return zmin;
}

// ------------------------------------------------------------------------------------------------
// A.2a-c + A.6: S_i = sum_j A_ij c_j, A = sum c_i S_i, B = sum c_i B_i,
//   lnphi_i = (B_i/B)(Z-1) - ln(Z-B) - (1/B) ln(1+B/Z) (2 S_i - A B_i/B).   c must sum to 1.
// ------------------------------------------------------------------------------------------------
template <int NC>
__device__ __forceinline__ void lnphi_eval(const Sys<NC>& S, const double (&sa)[NC], const double (&bi)[NC],
                                           const double (&c)[NC], double (&lp)[NC], double (&Sv)[NC], Eos& e) {
  double t[NC];
#pragma unroll
  for (int j = 0; j < NC; ++j) t[j] = sa[j] * c[j];
  if (S.kij_zero) {
    double sum = 0.0;
#pragma unroll
    for (int j = 0; j < NC; ++j) sum += t[j];
#pragma unroll
    for (int i = 0; i < NC; ++i) Sv[i] = sa[i] * sum;
  } else {
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      double acc = 0.0;
#pragma unroll
      for (int j = 0; j < NC; ++j) acc = fma(S.omk[i * NC + j], t[j], acc);
      Sv[i] = sa[i] * acc;
    }
  }
  double A = 0.0, B = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    A = fma(c[i], Sv[i], A);
    B = fma(c[i], bi[i], B);
  }
  e.A = A;
  e.B = B;
  e.Z = pick_root(A, B, e.lnZmB, e.L);
  const double invB = 1.0 / B;
  e.q = e.L * invB;
  const double zm1 = e.Z - 1.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    const double b = bi[i] * invB;
    lp[i] = fma(b, zm1, -e.lnZmB) - e.q * fma(2.0, Sv[i], -A * b);
  }
}

// M_ij = n dlnphi_i/dn_j at unit total moles (row-major NC x NC), from the quantities lnphi_eval left behind.
template <int NC>
__device__ __noinline__ void dlnphi(const Sys<NC>& S, const double (&sa)[NC], const double (&bi)[NC],
                                    const double (&Sv)[NC], const Eos& e, double* __restrict__ M) {
  const double A = e.A, B = e.B, Z = e.Z, L = e.L, q = e.q;
  const double invB = 1.0 / B;
  const double FZ = fma(fma(3.0, Z, -2.0), Z, A - B - B * B);
  const double ZA = -(Z - B) / FZ;
  const double ZB = fma(1.0 + 2.0 * B, Z, A) / FZ;
  const double invZmB = 1.0 / (Z - B);
  const double invZZB = 1.0 / (Z * (Z + B));
#pragma unroll 1
  for (int j = 0; j < NC; ++j) {
    const double bj = bi[j] * invB;
    const double DB = bi[j] - B;
    const double DA = 2.0 * (Sv[j] - A);
    const double DZ = ZA * DA + ZB * DB;
    const double DL = (Z * DB - B * DZ) * invZZB;
    const double Dq = (DL - L * DB * invB) * invB;
    const double c0 = (DZ - DB) * invZmB;
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      const double b = bi[i] * invB;
      const double Dbi = -b * (bj - 1.0);
      const double Aij = S.omk[i * NC + j] * sa[i] * sa[j];
      const double DSi = Aij - Sv[i];
      M[i * NC + j] = Dbi * (Z - 1.0) + b * DZ - c0 - Dq * (2.0 * Sv[i] - A * b) - q * (2.0 * DSi - DA * b - A * Dbi);
    }
  }
}

// eq. 6
template <int NC>
__device__ __forceinline__ void wilson_lnK(const Sys<NC>& S, double P, double T, double (&lnK)[NC]) {
  const double lnP = log(P);
  const double invT = 1.0 / T;
#pragma unroll
  for (int i = 0; i < NC; ++i) lnK[i] = (S.lnpc[i] - lnP) + S.wil[i] * (1.0 - S.tc[i] * invT);
}

// ------------------------------------------------------------------------------------------------
// Rachford-Rice (eq. 7; App. C): root of f(theta) = sum z_i (K_i-1)/(1+(K_i-1) theta) on the window
// (1/(1-Kmax), 1/(1-Kmin)).  Newton on the Leibovici-Neoschil helper h = (theta-al)(ar-theta) f, kept inside a
// shrinking sign bracket with bisection as the fallback; runs until the step is below rounding or f == 0.
// Components with z_i == 0 are skipped.  Returns false when there is no window.
// On success also returns x_i = z_i/(1+(K_i-1) theta), y_i = K_i x_i, both renormalised.
// ------------------------------------------------------------------------------------------------
template <int NC>
__device__ __forceinline__ bool rr_solve(const double (&K)[NC], const double (&z)[NC], double& theta,
                                         double (&x)[NC], double (&y)[NC]) {
  double Kmax = 0.0, Kmin = 1.0e300;
  double km1[NC];
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    km1[i] = (z[i] > 0.0) ? K[i] - 1.0 : 0.0;   // z_i == 0: the term and its pole drop out
    if (z[i] > 0.0) { Kmax = fmax(Kmax, K[i]); Kmin = fmin(Kmin, K[i]); }
  }
  if (!(Kmax > 1.0) || !(Kmin < 1.0)) return false;
  const double al = 1.0 / (1.0 - Kmax), ar = 1.0 / (1.0 - Kmin);
  double lo = al, hi = ar;
  // tighten with the two cheap evaluations f(0) = sum z K - 1, f(1) = 1 - sum z/K
  double f0 = 0.0, f1 = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    f0 = fma(z[i], km1[i], f0);
    f1 += z[i] * km1[i] / K[i];
  }
  double th;
  if (f0 > 0.0) { lo = 0.0; if (f1 < 0.0) { hi = 1.0; th = f0 / (f0 - f1); } else { lo = 1.0; th = fmin(1.0 + 0.5 * (ar - 1.0), 2.0); if (f1 == 0.0) { hi = 1.0; th = 1.0; } } }
  else if (f0 < 0.0) { hi = 0.0; th = fmax(0.5 * al, -1.0); }
  else { lo = hi = 0.0; th = 0.0; }
  if (!(th > lo && th < hi)) th = 0.5 * (lo + hi);
#pragma unroll 1
  for (int it = 0; it < 200; ++it) {
    if (!(hi > lo)) break;
    double f = 0.0, df = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      const double r = 1.0 / fma(km1[i], th, 1.0);
      const double a = z[i] * km1[i] * r;
      f += a;
      df = fma(-a, km1[i] * r, df);
    }
    if (f > 0.0) lo = th; else if (f < 0.0) hi = th; else break;
    // Newton on h = (th-al)(ar-th) f
    const double u = th - al, w = ar - th;
    const double h = u * w * f;
    const double dh = (w - u) * f + u * w * df;
    double tn = th - h / dh;
    if (!(tn > lo && tn < hi)) tn = 0.5 * (lo + hi);
    if (tn == th || fabs(tn - th) <= 2.3e-16 * fabs(th)) { th = tn; break; }
    th = tn;
  }
  theta = th;
  double sx = 0.0, sy = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    const double xi = (z[i] > 0.0) ? z[i] / fma(km1[i], th, 1.0) : 0.0;
    x[i] = xi;
    y[i] = K[i] * xi;
    sx += xi;
    sy += y[i];
  }
  const double isx = 1.0 / sx, isy = 1.0 / sy;
#pragma unroll
  for (int i = 0; i < NC; ++i) { x[i] *= isx; y[i] *= isy; }
  return true;
}

// ------------------------------------------------------------------------------------------------
// dense SPD solve (H + eta diag(D)) s = -g by Cholesky; H, Lc row-major n x n in local memory.
// ------------------------------------------------------------------------------------------------
template <int NC>
__device__ __noinline__ bool chol_solve(const double* __restrict__ H, const double* __restrict__ D, double eta,
                                        const double* __restrict__ g, double* __restrict__ s, double* __restrict__ Lc) {
#pragma unroll 1
  for (int i = 0; i < NC; ++i) {
#pragma unroll 1
    for (int j = 0; j <= i; ++j) {
      double acc = H[i * NC + j];
      if (i == j) acc = fma(eta, D[i], acc);
#pragma unroll 1
      for (int k = 0; k < j; ++k) acc = fma(-Lc[i * NC + k], Lc[j * NC + k], acc);
      if (i == j) {
        if (!(acc > 0.0)) return false;
        Lc[i * NC + i] = sqrt(acc);
      } else {
        Lc[i * NC + j] = acc / Lc[j * NC + j];
      }
    }
  }
  double yv[NC];
#pragma unroll 1
  for (int i = 0; i < NC; ++i) {
    double acc = -g[i];
#pragma unroll 1
    for (int k = 0; k < i; ++k) acc = fma(-Lc[i * NC + k], yv[k], acc);
    yv[i] = acc / Lc[i * NC + i];
  }
#pragma unroll 1
  for (int i = NC - 1; i >= 0; --i) {
    double acc = yv[i];
#pragma unroll 1
    for (int k = i + 1; k < NC; ++k) acc = fma(-Lc[k * NC + i], s[k], acc);
    s[i] = acc / Lc[i * NC + i];
  }
  return true;
}

// Restricted-step sub-problem (B.1b / B.4a): eta = 0 if admissible, else geometric growth (x8 from eta0) to the
// first admissible eta, then geometric bisection until ||s|| >= Delta/2 or the bracket ratio < 1.5.
// Admissible = positive definite, ||s|| <= Delta, lo < v + s < hi.  Inactive components (act[i] == false)
// must come in with H row/col = identity and g = 0 so that their step is zero.
template <int NC>
__device__ __noinline__ bool tr_subproblem(const double* __restrict__ H, const double* __restrict__ g,
                                           const double* __restrict__ D, double Delta, double eta0,
                                           const double* __restrict__ v, const double* __restrict__ hi,
                                           const bool* __restrict__ act, double* __restrict__ s, double& eta_out,
                                           double& snorm_out, double* __restrict__ Lc) {
  double st[NC];
  double sn = 0.0;
  auto attempt = [&](double eta) -> bool {
    if (!chol_solve<NC>(H, D, eta, g, st, Lc)) return false;
    sn = 0.0;
    bool feas = true;
#pragma unroll 1
    for (int a = 0; a < NC; ++a) {
      sn = fma(st[a], st[a], sn);
      if (act[a]) {
        const double nv = v[a] + st[a];
        if (!(nv > 0.0) || !(nv < hi[a])) feas = false;
      }
    }
    sn = sqrt(sn);
    return feas && sn <= Delta;
  };
  auto keep = [&](double eta) {
#pragma unroll 1
    for (int a = 0; a < NC; ++a) s[a] = st[a];
    eta_out = eta;
    snorm_out = sn;
  };
  if (attempt(0.0)) { keep(0.0); return true; }
  double eta_lo = 0.0, eta_hi = 0.0, eta = eta0;
  bool found = false;
#pragma unroll 1
  for (int k = 0; k < 60; ++k) {
    if (attempt(eta)) { eta_hi = eta; keep(eta); found = true; break; }
    eta_lo = eta;
    eta *= 8.0;
  }
  if (!found) return false;
#pragma unroll 1
  for (int k = 0; k < 12; ++k) {
    if (snorm_out >= 0.5 * Delta) break;
    if (eta_lo > 0.0 && eta_hi / eta_lo < 1.5) break;
    const double mid = (eta_lo > 0.0) ? sqrt(eta_lo * eta_hi) : eta_hi * 0.125;
    if (attempt(mid)) { eta_hi = mid; keep(mid); } else eta_lo = mid;
  }
  return true;
}

}  // namespace ptf
