// ptflash_fast.cuh -- register-resident, warm-started variants of the device functions in ptflash_device.cuh,
// used by the stage kernels of engine 1.  Same operations, same decisions (admissible roots Z > B, minimum
// Gibbs energy, Rachford-Rice window), different iteration paths:
//   * the cubic (A.3) is iterated from the previous root of the same phase (2-3 Newton steps) and falls back to
//     the monotone side-selected Newton; the other roots come from the deflated quadratic (A.5);
//   * Rachford-Rice (eq. 7) starts from the previous theta and stops after the first Newton step below 1e-8
//     of the window (App. C: "When the Newton step size is smaller than 1.0e-8, the iteration stops";
//     the step is applied, so the error is ~1e-16);
//   * everything is __forceinline__ so per-mixture vectors stay in registers (no struct passing through local memory).
#pragma once
#include "ptflash_device.cuh"
#include "ptflash_math.cuh"

namespace ptf {

// Newton polish of the two deflated roots (A.5), interleaved: a step is taken only if it lowers |f| (near a double root
// the deflated value is already the best available), twice.
__device__ __forceinline__ void cub_polish2(double& za, double& zb, double r1, double r0) {
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const double fa = cub_f(za, r1, r0), fb = cub_f(zb, r1, r0);
    const double na = za - fa * rcp_nr1(cub_df(za, r1)), nb = zb - fb * rcp_nr1(cub_df(zb, r1));
    za = (fabs(cub_f(na, r1, r0)) < fabs(fa)) ? na : za;   // a NaN step (df == 0) fails the test and is dropped
    zb = (fabs(cub_f(nb, r1, r0)) < fabs(fb)) ? nb : zb;
  }
}

// ------------------------------------------------------------------------------------------------
// cubic with warm start.  Zg: previous root of this phase (<= 0: none).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double pick_root_fast(double A, double B, double Zg, double& lnZmB, double& L) {
  const double r0 = A * B, r1 = A - B * (1.0 + B);
  double Z = Zg;
  bool ok = false;
  if (Zg > B) {
    // Halley's iteration (A.4, third order) from the previous root: a step below 1e-5 Z leaves an error ~ step^3, i.e.
    // rounding level, so the typical warm start costs two evaluations (Newton needed three plus a confirming one).
#pragma unroll 1
    for (int k = 0; k < 4; ++k) {
      const double f = cub_f(Z, r1, r0), df = cub_df(Z, r1);
      const double d2 = fma(3.0, Z, -1.0);                     // f'' / 2
      const double dz = f * df * rcp_nr1(fma(df, df, -f * d2));
      const double Zn = Z - dz;
      if (!(Zn > B) || !(Zn < 2.0 + B)) break;   // also catches NaN / a vanishing denominator
      Z = Zn;
      if (fabs(dz) <= 1.0e-5 * Zn) { ok = true; break; }
    }
    if (ok) {
      // one Newton step brings the root to rounding and detects a linear-rate (nearly double) root
      const double dz = cub_f(Z, r1, r0) * rcp_nr1(cub_df(Z, r1));
      if (fabs(dz) <= 1.0e-11 * Z) Z -= dz; else ok = false;
    }
  }
  if (!ok) {
    const double third = 1.0 / 3.0;
    const bool up = (B < third) && (cub_f(third, r1, r0) > 0.0);
    Z = up ? B : 1.0 + B;
#pragma unroll 1
    for (int k = 0; k < 100; ++k) {
      const double df = cub_df(Z, r1);
      if (!(df > 0.0)) break;
      const double Zn = Z - cub_f(Z, r1, r0) * rcp_nr1(df);
      if (up ? !(Zn > Z) : !(Zn < Z)) break;
      Z = Zn;
    }
  }
  double zmin = Z, zmax = Z;
  const double p = Z - 1.0, q = fma(p, Z, r1);
  const double disc = fma(p, p, -4.0 * q);
  if (disc >= 0.0) {
    const double sq = sqrt_fast(disc);
    const double t = (p >= 0.0) ? -0.5 * (p + sq) : 0.5 * (sq - p);
    double ra = t, rb = (t != 0.0) ? div_fast(q, t) : -p - t;
    cub_polish2(ra, rb, r1, r0);
    if (ra > B) { zmin = dmin(zmin, ra); zmax = dmax(zmax, ra); }
    if (rb > B) { zmin = dmin(zmin, rb); zmax = dmax(zmax, rb); }
  }
  double lz = log_fast(zmin - B), ll = log1p_fast(B * rcp_fast(zmin));
  if (zmax != zmin) {
    const double AoB = A * rcp_fast(B);
    const double lz2 = log_fast(zmax - B), ll2 = log1p_fast(B * rcp_fast(zmax));
    const double gl = zmin - 1.0 - lz - AoB * ll;
    const double gv = zmax - 1.0 - lz2 - AoB * ll2;
    if (gv < gl) { zmin = zmax; lz = lz2; ll = ll2; }
  }
  lnZmB = lz;
  L = ll;
  return zmin;
}

// ------------------------------------------------------------------------------------------------
// lnphi of composition c (sum c = 1) given sqrt(A_i), B_i.  e.Z on entry = warm start (<= 0: none).
// KIJ0: all k_ij == 0, S_i = sqrt(A_i) * sum_j sqrt(A_j) c_j.
// ------------------------------------------------------------------------------------------------
template <int NC, bool KIJ0>
__device__ __forceinline__ void lnphi_fast(const Sys<NC>& S, const double (&sa)[NC], const double (&bi)[NC],
                                           const double (&c)[NC], double (&lp)[NC], double (&Sv)[NC], Eos& e) {
  double t[NC];
#pragma unroll
  for (int j = 0; j < NC; ++j) t[j] = sa[j] * c[j];
  if (KIJ0) {
    double sum = 0.0;
#pragma unroll
    for (int j = 0; j < NC; ++j) sum += t[j];
#pragma unroll
    for (int i = 0; i < NC; ++i) Sv[i] = sa[i] * sum;
  } else {
    // symmetric k_ij with a zero diagonal: every 1 - k_ij serves two products (see lnphi_pt)
    double a[NC];
#pragma unroll
    for (int i = 0; i < NC; ++i) a[i] = t[i];
#pragma unroll
    for (int i = 0; i < NC; ++i) {
#pragma unroll
      for (int j = 0; j < NC; ++j) {
        if (j > i) {
          const double c = S.omk[i * NC + j];
          a[i] = fma(c, t[j], a[i]);
          a[j] = fma(c, t[i], a[j]);
        }
      }
    }
#pragma unroll
    for (int i = 0; i < NC; ++i) Sv[i] = sa[i] * a[i];
  }
  double A = 0.0, B = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    A = fma(c[i], Sv[i], A);
    B = fma(c[i], bi[i], B);
  }
  e.A = A;
  e.B = B;
  e.Z = pick_root_fast(A, B, e.Z, e.lnZmB, e.L);
  const double invB = rcp_fast(B);
  e.q = e.L * invB;
  const double zm1 = e.Z - 1.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    const double b = bi[i] * invB;
    lp[i] = fma(b, zm1, -e.lnZmB) - e.q * fma(2.0, Sv[i], -A * b);
  }
}

// Register-lean variant: sqrt(A_i) and B_i are rebuilt from three per-mixture scalars (sqrt(P)/T, sqrt(T), P/T)
// and the per-component constants in the constant bank instead of living in 2 nc registers.
template <int NC>
struct PT3 { double spt, sT, pt; };
template <int NC>
__device__ __forceinline__ double sa_of(const Sys<NC>& S, const PT3<NC>& q, int i) { return q.spt * fabs(fma(-S.v[i], q.sT, S.u[i])); }
template <int NC>
__device__ __forceinline__ double bi_of(const Sys<NC>& S, const PT3<NC>& q, int i) { return q.pt * S.wb[i]; }

template <int NC, bool KIJ0>
__device__ __forceinline__ void lnphi_pt(const Sys<NC>& S, const PT3<NC>& q, const double (&c)[NC], double (&lp)[NC],
                                         double (&Sv)[NC], Eos& e) {
  double t[NC], sa[NC];
  double B0 = 0.0, B1 = 0.0;   // two accumulation chains each (depth NC/2 instead of NC)
#pragma unroll
  for (int j = 0; j < NC; ++j) {
    sa[j] = sa_of<NC>(S, q, j);
    t[j] = sa[j] * c[j];
    if (j & 1) B1 = fma(c[j], S.wb[j], B1); else B0 = fma(c[j], S.wb[j], B0);
  }
  const double B = q.pt * (B0 + B1);   // B_i = (P/T) wb_i
  if (KIJ0) {
    double s0 = 0.0, s1 = 0.0;
#pragma unroll
    for (int j = 0; j < NC; ++j) { if (j & 1) s1 += t[j]; else s0 += t[j]; }
    const double sum = s0 + s1;
#pragma unroll
    for (int i = 0; i < NC; ++i) Sv[i] = sa[i] * sum;
  } else {
    // k_ij is symmetric with a zero diagonal (checked by ptflash_create), so every 1 - k_ij serves two products and the
    // diagonal needs none: 45 constant operands instead of 100 at nc = 10.  (A DFMA whose constant cannot stay in a uniform
    // register costs an LDCU, and a stream of such pairs runs at half the DFMA rate on sm_100a, measured.)
    {
      double a[NC];
#pragma unroll
      for (int i = 0; i < NC; ++i) a[i] = t[i];
#pragma unroll
      for (int i = 0; i < NC; ++i) {
#pragma unroll
        for (int j = 0; j < NC; ++j) {
          if (j > i) {
            const double c = S.omk[i * NC + j];
            a[i] = fma(c, t[j], a[i]);
            a[j] = fma(c, t[i], a[j]);
          }
        }
      }
#pragma unroll
      for (int i = 0; i < NC; ++i) Sv[i] = sa[i] * a[i];
    }
  }
  double A0 = 0.0, A1 = 0.0;
#pragma unroll
  for (int i = 0; i < NC; i += 2) {
    A0 = fma(c[i], Sv[i], A0);
    if (i + 1 < NC) A1 = fma(c[i + 1], Sv[i + 1], A1);
  }
  const double A = A0 + A1;
  e.A = A;
  e.B = B;
  e.Z = pick_root_fast(A, B, e.Z, e.lnZmB, e.L);
  const double invB = rcp_fast(B);
  e.q = e.L * invB;
  const double zm1 = e.Z - 1.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    const double b = bi_of<NC>(S, q, i) * invB;
    lp[i] = fma(b, zm1, -e.lnZmB) - e.q * fma(2.0, Sv[i], -A * b);
  }
}

// ------------------------------------------------------------------------------------------------
// Rachford-Rice with warm start (eq. 7, App. C).  theta on entry: previous solution (used if inside the sign
// bracket).  Returns false when there is no window.  Produces normalised x, y.
//
// The Leibovici-Neoschil Newton iteration on h = (theta-al)(ar-theta) f inside a shrinking sign bracket, with
// bisection as the fallback, until the applied step is below 1e-8 of the window.
// (A single-precision pre-iteration was tried and measured slower on B200: the fp32 loop diverged more than it saved.)
// ------------------------------------------------------------------------------------------------
template <int NC>
__device__ __forceinline__ bool rr_fast(const double (&K)[NC], const double (&z)[NC], double& theta, double (&x)[NC],
                                        double (&y)[NC]) {
  double Kmax = 0.0, Kmin = 1.0e300;
  double km1[NC];
  double f0 = 0.0, f1 = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    const bool a = z[i] > 0.0;
    km1[i] = a ? K[i] - 1.0 : 0.0;
    if (a) { Kmax = dmax(Kmax, K[i]); Kmin = dmin(Kmin, K[i]); }
    f0 = fma(z[i], km1[i], f0);
    f1 = fma(z[i] * km1[i], rcp_fast(K[i]), f1);
  }
  if (!(Kmax > 1.0) || !(Kmin < 1.0)) return false;
  const double al = div_fast(1.0, 1.0 - Kmax), ar = div_fast(1.0, 1.0 - Kmin);
  double lo = al, hi = ar, th;
  if (f0 > 0.0) {
    if (f1 < 0.0) { lo = 0.0; hi = 1.0; th = f0 * rcp_fast(f0 - f1); }
    else if (f1 == 0.0) { lo = hi = 1.0; th = 1.0; }
    else { lo = 1.0; th = dmin(1.0 + 0.5 * (ar - 1.0), 2.0); }
  } else if (f0 < 0.0) { hi = 0.0; th = dmax(0.5 * al, -1.0); }
  else { lo = hi = 0.0; th = 0.0; }
  const bool warm = (theta > lo && theta < hi);
  if (warm) th = theta;
  if (!(th > lo && th < hi)) th = 0.5 * (lo + hi);
  const double width = dmin(ar - al, 1.0);

  const double scale = 1.0e-8 * width;
#pragma unroll 1
  for (int it = 0; it < 100; ++it) {
    if (!(hi > lo)) break;
    double f = 0.0, df = 0.0;
#pragma unroll
    for (int i = 0; i < NC; ++i) {
      const double r = rcp_nr1(fma(km1[i], th, 1.0));   // 2^-40 is enough inside the iteration: the error of the final theta
      const double a = z[i] * km1[i] * r;                // is (relative error of the last step) x (last step <= 1e-8 window)
      f += a;
      df = fma(-a, km1[i] * r, df);
    }
    if (f > 0.0) lo = th; else if (f < 0.0) hi = th; else break;
    const double u = th - al, w = ar - th;
    const double h = u * w * f;
    const double dh = (w - u) * f + u * w * df;
    double tn = th - h * rcp_fast(dh);
    // Newton step below the tolerance: apply it and stop (quadratic convergence leaves an error ~ step^2).  th is an end
    // of the sign bracket here, so a converged tn can land ON or an ulp beyond that end; it is clamped, not bisected
    // (bisecting from a converged iterate cost ~25 extra iterations in 1 % of the calls, i.e. in every fourth warp).
    if (fabs(tn - th) <= scale) { th = dmin(dmax(tn, lo), hi); break; }
    const bool inside = (tn > lo && tn < hi);
    if (!inside) tn = 0.5 * (lo + hi);
    if (fabs(tn - th) <= 2.3e-16 * fabs(tn)) { th = tn; break; }
    th = tn;
  }
  theta = th;
  double sx = 0.0, sy = 0.0;
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    const double xi = z[i] * rcp_fast(fma(km1[i], th, 1.0));   // z_i = 0: km1_i = 0, x_i = 0
    x[i] = xi;
    y[i] = K[i] * xi;
    sx += xi;
    sy += y[i];
  }
  const double isx = rcp_fast(sx), isy = rcp_fast(sy);
#pragma unroll
  for (int i = 0; i < NC; ++i) { x[i] *= isx; y[i] *= isy; }
  return true;
}

}  // namespace ptf
