// ptflash_oracle.cpp -- CPU ORACLE for the batched isothermal two-phase SRK flash (PTFlash, arXiv 2205.03090).
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may build, load or call it.  It shares no code with the CUDA
// path under paper_2205_03090_b200/csrc (no common headers, helpers, tables or constants) and is
// deliberately plain: one mixture at a time, scalar loops, no blocking/fusion/SIMD, `real` = double
// (or long double with -DORACLE_REAL="long double" for adjudicating disagreements).
//
// Every function cites the passage of /root/reference/PAPER.md it follows (PAPER.md:<line>, section /
// equation) and, where the paper is silent or garbled, the reading C<n> listed in DESIGN.md section 3
// (taken from SURVEY.md section 8(c)).  Pins (tests/test_oracle_*.py, -m "not gpu"):
//   cubic            : Vieta, trigonometric/Cardano closed form, f(B) = -2B^2, f(1+B) = A
//   lnphi            : sum c_i lnphi_i = g(Z) closed form, ideal-gas limit, pure-component saturation
//   dlnphi           : central finite differences of lnphi, symmetry, Gibbs-Duhem
//   rachford_rice    : monotonicity, sign change across the bracket, binary closed form
//   stability        : binary brute force on a composition grid (lower convex hull), tm = 1 - sum W
//   split            : material balance, iso-fugacity, G_two-phase < G_feed, hull tangent points,
//                      Newton finish == long pure successive substitution, long double == double
// Not pinned ("parity unpinned"): nothing on the hot path; the paper prints no worked (P,T,z) example,
// so whole-flash pins are invariants + brute force, not printed values.
//
// Build: g++ -O2 -std=c++17 -fPIC -shared [-fopenmp] ptflash_oracle.cpp -o libptflash_oracle.so
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <algorithm>
#ifndef ORACLE_REAL
#define ORACLE_REAL double
#endif
typedef ORACLE_REAL real;

#define MAXC 16

static inline real r_sqrt(real x) { return std::sqrt(x); }
static inline real r_log(real x) { return std::log(x); }
static inline real r_exp(real x) { return std::exp(x); }
static inline real r_abs(real x) { return std::fabs(x); }
static inline real r_acos(real x) { return std::acos(x); }
static inline real r_cos(real x) { return std::cos(x); }
static inline real r_cbrt(real x) { return std::cbrt(x); }

// ------------------------------------------------------------------------------------------------
// Options (tolerances and caps).  Defaults = DESIGN.md section 3 (C8) / PAPER.md:79,90,97,105,558.
// ------------------------------------------------------------------------------------------------
struct Opts {
  double tol_ss;          // [0] successive-substitution residual target (stability r, split r_k, eps_k)  1e-10
  double tol_newton_g;    // [1] Newton: gradient target                                                 1e-12
  double tol_newton_step; // [2] Newton: full-step size below which the step is applied and we stop        1e-10
  double probe_margin;    // [3] "negative" in the probe test means < -margin (C6)                         1e-8
  double trivial_tol;     // [4] trivial stability solution: max|lnW - lnz| < tol (C7)                     1e-6
  double band;            // [5] near-zero TPD band (C9)                                                   1e-9
  double probe_iters;     // [6] 3
  double stab_ss_iters;   // [7] 9
  double stab_tr_iters;   // [8] 60  (paper: 20; larger here because targets are tighter)
  double split_ss_iters;  // [9] 9
  double split_tr_iters;  // [10] 60
  double use_newton;      // [11] 1; 0 = pure successive substitution everywhere (used by pins)
  double ss_cap;          // [12] cap on SS iterations when use_newton == 0                               100000
  double hint_ss_cap;     // [13] a skip-stability hint whose split SS is still outside 0 < theta < 1 after this
                          //      many iterations is dropped (reading C21)                  12
  double eta_growth;      // [14] restricted step (C11): geometric growth factor of eta                            8
  double eta_ratio;       // [15] restricted step (C11): the bisection of eta stops at this bracket ratio          1.5
                          //      ([14], [15] exist so that tests/oracle_path_sensitivity.py can perturb the schedule)
  double split_trivial_tol; // [16] the split has collapsed into the trivial solution x = y when max|ln K_i| < tol     1e-5
                          //      (reading C22: a Newton iteration sliding into x = y "converges" -- its gradient vanishes
                          //      with |ln K| -- at |ln K| ~ 1e-8, theta ~ 1e-9; genuine solutions of the workloads have
                          //      max|ln K| > 3e-2)
  double stability_only;  // [17] 1 = stop after the label (probe + stability analysis, no phase split): the mode the
                          //      paper uses to label 10^6 samples for its classifier                  0
  double hint_tr_cap;     // [18] a skip-stability hint whose split has not converged after this many trust-region iterations
                          //      is dropped (reading C21: on the warm-start workload converging hinted splits need at most
                          //      11, failing ones wander until the cap)                                                   15
};
static Opts default_opts() {
  Opts o = {1e-10, 1e-12, 1e-10, 1e-8, 1e-6, 1e-9, 3, 9, 60, 9, 60, 1, 100000, 12, 8, 1.5, 1e-5, 0, 15};
  return o;
}
#define NOPTS 19
static Opts opts_from(const double* p) {
  Opts o = default_opts();
  if (p) std::memcpy(&o, p, sizeof(double) * NOPTS);
  return o;
}

// status bits (same meaning as include/ptflash.h but defined independently)
enum { ST_STAB_CAP = 1, ST_SPLIT_CAP = 2, ST_BAND = 4, ST_SPLIT_FAILED = 8, ST_LNK0_REJECTED = 32, ST_WARM_RESTART = 64 };

// ------------------------------------------------------------------------------------------------
// O1 Setup: dimensionless SRK groups.  PAPER.md:412-434 (A.2a-g, A.3).  R never appears:
//   A_i = 0.42748 alpha_i (P/Pc_i)/(T/Tc_i)^2, B_i = 0.08664 (P/Pc_i)/(T/Tc_i), A_ij = (1-k_ij) sqrt(A_i A_j).
// ------------------------------------------------------------------------------------------------
struct Setup {
  int nc;
  real Ai[MAXC], Bi[MAXC], Aij[MAXC][MAXC];
};
static void setup(int nc, const double* Tc, const double* Pc, const double* omega, const double* kij,
                  real P, real T, Setup& s) {
  s.nc = nc;
  for (int i = 0; i < nc; ++i) {
    real Tr = T / (real)Tc[i];
    real Pr = P / (real)Pc[i];
    real om = (real)omega[i];
    real m = (real)0.480 + (real)1.574 * om - (real)0.176 * om * om;      // A.2g PAPER.md:426
    real sa = (real)1 + m * ((real)1 - r_sqrt(Tr));                       // A.2f PAPER.md:424
    real alpha = sa * sa;
    s.Ai[i] = (real)0.42748 * alpha * Pr / (Tr * Tr);                     // A.2d with A = a alpha P/(RT)^2
    s.Bi[i] = (real)0.08664 * Pr / Tr;                                    // A.2e with B = bP/(RT)
  }
  for (int i = 0; i < nc; ++i)
    for (int j = 0; j < nc; ++j) {
      real k = kij ? (real)kij[i * nc + j] : (real)0;
      s.Aij[i][j] = ((real)1 - k) * r_sqrt(s.Ai[i] * s.Ai[j]);            // A.2b PAPER.md:415
    }
}

// ------------------------------------------------------------------------------------------------
// Cubic (A.3) f(Z) = Z^3 - Z^2 + rho1 Z - rho0, rho0 = AB, rho1 = A - B(1+B).  PAPER.md:431-445.
// The paper iterates one root (A.4), deflates (A.5) and solves the quadratic.  Reading C15: the
// iteration is a monotone Newton started on the side where f has the right curvature
// (inflection at Z = 1/3 for every A, B; f(B) = -2B^2 < 0; f(1+B) = A > 0), run until the iterate stops
// moving; the other two roots come from the deflated quadratic and are polished on the full cubic.
// Returns the number of real roots (1 or 3) sorted ascending in r[].
// ------------------------------------------------------------------------------------------------
static inline real cubic_f(real Z, real rho1, real rho0) { return ((Z - (real)1) * Z + rho1) * Z - rho0; }
static inline real cubic_df(real Z, real rho1) { return ((real)3 * Z - (real)2) * Z + rho1; }

static real polish(real Z, real rho1, real rho0) {
  for (int k = 0; k < 3; ++k) {
    real f = cubic_f(Z, rho1, rho0), df = cubic_df(Z, rho1);
    if (df == (real)0) break;
    real Zn = Z - f / df;
    if (!(r_abs(cubic_f(Zn, rho1, rho0)) < r_abs(f))) break;
    Z = Zn;
  }
  return Z;
}

static int cubic_roots(real A, real B, real r[3]) {
  const real rho0 = A * B, rho1 = A - B * ((real)1 + B);
  const real third = (real)1 / (real)3;
  const real f13 = cubic_f(third, rho1, rho0);
  real Z;
  if (B < third && f13 > (real)0) {
    // root in (B, 1/3): f concave there, f(B) < 0 -> Newton from B increases monotonically
    Z = B;
    for (int k = 0; k < 500; ++k) {
      real df = cubic_df(Z, rho1);
      if (!(df > (real)0)) break;
      real Zn = Z - cubic_f(Z, rho1, rho0) / df;
      if (!(Zn > Z)) break;
      Z = Zn;
    }
  } else {
    // largest root lies in [max(B,1/3), 1+B): f convex there, f(1+B) = A > 0 -> Newton decreases monotonically
    Z = (real)1 + B;
    for (int k = 0; k < 500; ++k) {
      real df = cubic_df(Z, rho1);
      if (!(df > (real)0)) break;
      real Zn = Z - cubic_f(Z, rho1, rho0) / df;
      if (!(Zn < Z)) break;
      Z = Zn;
    }
  }
  const real Z0 = Z;
  // deflation A.5 PAPER.md:443-445: f = (Z - Z0)(Z^2 + pZ + q), p = Z0 - 1, q = p Z0 + rho1
  const real p = Z0 - (real)1, q = p * Z0 + rho1;
  const real disc = p * p - (real)4 * q;
  if (disc < (real)0) { r[0] = Z0; return 1; }
  const real sq = r_sqrt(disc);
  // cancellation-free quadratic roots
  real t = (p >= (real)0) ? -(p + sq) / (real)2 : (-p + sq) / (real)2;
  real ra = t, rb = (t != (real)0) ? q / t : -p - t;
  ra = polish(ra, rho1, rho0);
  rb = polish(rb, rho1, rho0);
  r[0] = Z0; r[1] = ra; r[2] = rb;
  std::sort(r, r + 3);
  return 3;
}

// Closed form (trigonometric / Cardano) for the same cubic -- used ONLY as a pin for cubic_roots.
static int cubic_roots_closed(real A, real B, real r[3]) {
  const real rho0 = A * B, rho1 = A - B * ((real)1 + B);
  // Z = t + 1/3 : t^3 + pp t + qq = 0
  const real pp = rho1 - (real)1 / (real)3;
  const real qq = -(real)2 / (real)27 + rho1 / (real)3 - rho0;
  const real D = qq * qq / (real)4 + pp * pp * pp / (real)27;
  if (D > (real)0) {
    const real s = r_sqrt(D);
    r[0] = r_cbrt(-qq / (real)2 + s) + r_cbrt(-qq / (real)2 - s) + (real)1 / (real)3;
    return 1;
  }
  const real m = (real)2 * r_sqrt(-pp / (real)3);
  real arg = (real)3 * qq / (pp * m);
  if (arg > (real)1) arg = (real)1;
  if (arg < (real)-1) arg = (real)-1;
  const real th = r_acos(arg) / (real)3;
  const real pi = (real)3.14159265358979323846264338327950288L;
  for (int k = 0; k < 3; ++k) r[k] = m * r_cos(th - (real)2 * pi * (real)k / (real)3) + (real)1 / (real)3;
  std::sort(r, r + 3);
  return 3;
}

// Reduced residual Gibbs energy of a phase at root Z: g = sum c_i lnphi_i = Z - 1 - ln(Z-B) - (A/B) ln(1+B/Z)  (C4)
static inline real gibbs_of_root(real Z, real A, real B) {
  return Z - (real)1 - r_log(Z - B) - (A / B) * r_log((real)1 + B / Z);
}

// Root choice (PAPER.md:445 + C3, C4): admissible roots are Z > B; candidates are the smallest and the
// largest admissible root; the one with the lower g wins; exact tie -> smaller Z.
static real choose_root(real A, real B) {
  real r[3];
  int n = cubic_roots(A, B, r);
  real zmin = (real)0, zmax = (real)0;
  bool have = false;
  for (int k = 0; k < n; ++k)
    if (r[k] > B) {
      if (!have) { zmin = zmax = r[k]; have = true; }
      else { if (r[k] < zmin) zmin = r[k]; if (r[k] > zmax) zmax = r[k]; }
    }
  if (!have) return std::numeric_limits<real>::quiet_NaN();
  if (zmin == zmax) return zmin;
  real gl = gibbs_of_root(zmin, A, B), gv = gibbs_of_root(zmax, A, B);
  return (gv < gl) ? zmax : zmin;
}

// ------------------------------------------------------------------------------------------------
// O2 lnphi(c): A.2a-c mixing rules, cubic, root choice, A.6 in A, B, S form:
//   S_i = sum_j A_ij c_j, A = sum_i c_i S_i, B = sum_i c_i B_i
//   lnphi_i = (B_i/B)(Z-1) - ln(Z-B) - (1/B) ln(1+B/Z) (2 S_i - A B_i/B)
// c must sum to 1.  Components with c_i == 0 still get a (finite) lnphi_i.
// If M != nullptr also returns M_ij = n dlnphi_i/dn_j at unit total moles (formula not printed in the
// paper; derived in DESIGN.md section 3, pinned by finite differences).
// ------------------------------------------------------------------------------------------------
static void lnphi(const Setup& s, const real* c, real* out, real* Zout, real (*M)[MAXC]) {
  const int nc = s.nc;
  real S[MAXC], A = 0, B = 0;
  for (int i = 0; i < nc; ++i) {
    real acc = 0;
    for (int j = 0; j < nc; ++j) acc += s.Aij[i][j] * c[j];
    S[i] = acc;
  }
  for (int i = 0; i < nc; ++i) { A += c[i] * S[i]; B += c[i] * s.Bi[i]; }
  const real Z = choose_root(A, B);
  const real L = r_log((real)1 + B / Z);
  const real q = L / B;
  const real lnZmB = r_log(Z - B);
  for (int i = 0; i < nc; ++i) {
    real bi = s.Bi[i] / B;
    out[i] = bi * (Z - (real)1) - lnZmB - q * ((real)2 * S[i] - A * bi);
  }
  if (Zout) *Zout = Z;
  if (M) {
    const real FZ = (real)3 * Z * Z - (real)2 * Z + A - B - B * B;
    const real ZA = -(Z - B) / FZ;
    const real ZB = (((real)1 + (real)2 * B) * Z + A) / FZ;
    for (int j = 0; j < nc; ++j) {
      real bj = s.Bi[j] / B;
      real DB = s.Bi[j] - B;
      real DA = (real)2 * (S[j] - A);
      real DZ = ZA * DA + ZB * DB;
      real DL = (Z * DB - B * DZ) / (Z * (Z + B));
      real Dq = DL / B - L * DB / (B * B);
      for (int i = 0; i < nc; ++i) {
        real bi = s.Bi[i] / B;
        real Dbi = -bi * (bj - (real)1);
        real DSi = s.Aij[i][j] - S[i];
        M[i][j] = Dbi * (Z - (real)1) + bi * DZ - (DZ - DB) / (Z - B) - Dq * ((real)2 * S[i] - A * bi)
                  - q * ((real)2 * DSi - DA * bi - A * Dbi);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// O3 Wilson K-values, eq. 6 PAPER.md:74.
// ------------------------------------------------------------------------------------------------
static void wilson_lnK(int nc, const double* Tc, const double* Pc, const double* omega, real P, real T, real* lnK) {
  for (int i = 0; i < nc; ++i)
    lnK[i] = r_log((real)Pc[i] / P) + (real)5.373 * ((real)1 + (real)omega[i]) * ((real)1 - (real)Tc[i] / T);
}

// ------------------------------------------------------------------------------------------------
// O6 Rachford-Rice, eq. 7 PAPER.md:85 and App. C PAPER.md:514-525.  f_RR is strictly decreasing on
// (alpha_l, alpha_r) = (1/(1-Kmax), 1/(1-Kmin)) with poles at both ends; the oracle finds the unique
// root by plain bisection down to an (at most) 2-ulp bracket (C14).  Components with z_i == 0 are
// skipped (C12).  Returns false when there is no window (Kmin >= 1 or Kmax <= 1, C13).
// ------------------------------------------------------------------------------------------------
static real rr_f(int nc, const real* K, const real* z, real th) {
  real f = 0;
  for (int i = 0; i < nc; ++i)
    if (z[i] > (real)0) f += (K[i] - (real)1) * z[i] / ((real)1 + (K[i] - (real)1) * th);
  return f;
}
static bool rachford_rice(int nc, const real* K, const real* z, real* theta) {
  real Kmax = -1, Kmin = -1;
  bool first = true;
  for (int i = 0; i < nc; ++i)
    if (z[i] > (real)0) {
      if (first) { Kmax = Kmin = K[i]; first = false; }
      else { if (K[i] > Kmax) Kmax = K[i]; if (K[i] < Kmin) Kmin = K[i]; }
    }
  if (first || !(Kmax > (real)1) || !(Kmin < (real)1)) return false;
  real lo = (real)1 / ((real)1 - Kmax), hi = (real)1 / ((real)1 - Kmin);
  for (int it = 0; it < 20000; ++it) {
    real mid = lo + (hi - lo) / (real)2;
    if (!(mid > lo) || !(mid < hi)) break;
    real f = rr_f(nc, K, z, mid);
    if (f > (real)0) lo = mid; else if (f < (real)0) hi = mid; else { lo = hi = mid; break; }
  }
  // of the two bracket ends return the one with the smaller residual that keeps all denominators positive
  real cand = lo + (hi - lo) / (real)2;
  *theta = cand;
  return true;
}

// x_i = z_i / (1 + (K_i-1) theta), y_i = K_i x_i, renormalised (O4/O8)
static void phases_from_theta(int nc, const real* K, const real* z, real th, real* x, real* y) {
  real sx = 0, sy = 0;
  for (int i = 0; i < nc; ++i) {
    if (z[i] > (real)0) { x[i] = z[i] / ((real)1 + (K[i] - (real)1) * th); y[i] = K[i] * x[i]; }
    else { x[i] = 0; y[i] = 0; }
    sx += x[i]; sy += y[i];
  }
  for (int i = 0; i < nc; ++i) { x[i] /= sx; y[i] /= sy; }
}

// d theta / d K_i at a root of f_RR by the implicit-function theorem, eq. 13 PAPER.md:281-286:
//   d theta / d K = -[d f_RR / d theta]^-1 d f_RR / d K,  with f_RR of eq. 7 differentiated term by term:
//   d f / d K_i = z_i / (1 + (K_i - 1) theta) - (K_i - 1) z_i theta / (1 + (K_i - 1) theta)^2,
//   d f / d theta = - sum_i (K_i - 1)^2 z_i / (1 + (K_i - 1) theta)^2.        Components with z_i = 0 get 0 (C12).
static void rr_dtheta_dK(int nc, const real* K, const real* z, real th, real* dth) {
  real dfdth = 0;
  for (int i = 0; i < nc; ++i)
    if (z[i] > (real)0) { const real den = (real)1 + (K[i] - (real)1) * th; dfdth -= (K[i] - (real)1) * (K[i] - (real)1) * z[i] / (den * den); }
  for (int i = 0; i < nc; ++i) {
    if (z[i] > (real)0) {
      const real den = (real)1 + (K[i] - (real)1) * th;
      const real dfdK = z[i] / den - (K[i] - (real)1) * z[i] * th / (den * den);
      dth[i] = -dfdK / dfdth;
    } else dth[i] = 0;
  }
}

static inline real xlnx_term(real c, real t) { return (c > (real)0) ? c * t : (real)0; }

// reduced tangent plane distance of trial composition w against the feed, eq. 3
static real tpd_of(int nc, const real* w, const real* lnphi_w, const real* d) {
  real t = 0;
  for (int i = 0; i < nc; ++i)
    if (w[i] > (real)0) t += w[i] * (r_log(w[i]) + lnphi_w[i] - d[i]);
  return t;
}

// ------------------------------------------------------------------------------------------------
// dense SPD solve by Cholesky (plain textbook LL^T); returns false if not positive definite
// ------------------------------------------------------------------------------------------------
static bool chol_solve(int n, real (*H)[MAXC], const real* rhs, real* sol) {
  real L[MAXC][MAXC];
  for (int i = 0; i < n; ++i)
    for (int j = 0; j <= i; ++j) {
      real acc = H[i][j];
      for (int k = 0; k < j; ++k) acc -= L[i][k] * L[j][k];
      if (i == j) {
        if (!(acc > (real)0)) return false;
        L[i][i] = r_sqrt(acc);
      } else L[i][j] = acc / L[j][j];
    }
  real yv[MAXC];
  for (int i = 0; i < n; ++i) {
    real acc = rhs[i];
    for (int k = 0; k < i; ++k) acc -= L[i][k] * yv[k];
    yv[i] = acc / L[i][i];
  }
  for (int i = n - 1; i >= 0; --i) {
    real acc = yv[i];
    for (int k = i + 1; k < n; ++k) acc -= L[k][i] * sol[k];
    sol[i] = acc / L[i][i];
  }
  return true;
}


// ------------------------------------------------------------------------------------------------
// Trust-region sub-problem shared by B.1b and B.4a:
//   (H + eta D) s = -g,  ||s|| <= Delta,  lo < v + s < hi,
// with D = I for the stability analysis and D = diag(z/(xy)) for the phase split.  The paper cites
// Hebden [25] and gives no details (C11).  Reading: eta = 0 if that step is admissible; otherwise
// grow eta geometrically (x8 from eta0) to the first admissible value, then refine between the last
// inadmissible and the first admissible eta by geometric bisection until ||s|| >= Delta/2 or the
// bracket ratio is below 1.5.  "Admissible" = Cholesky succeeds (positive definite), the step is
// inside the trust region and inside the box.  Returns false if no admissible eta was found.
// ------------------------------------------------------------------------------------------------
static bool tr_subproblem(int n, real (*H)[MAXC], const real* g, const real* D, real Delta, real eta0,
                          const real* v, const real* lo, const real* hi, real* s, real* eta_out, real* snorm_out,
                          real growth = (real)8, real ratio_stop = (real)1.5) {
  real Hh[MAXC][MAXC], neg[MAXC], st[MAXC];
  for (int a = 0; a < n; ++a) neg[a] = -g[a];
  real sn = 0;
  auto attempt = [&](real eta) -> bool {
    for (int a = 0; a < n; ++a) for (int b = 0; b < n; ++b) Hh[a][b] = H[a][b] + ((a == b) ? eta * D[a] : (real)0);
    if (!chol_solve(n, Hh, neg, st)) return false;
    sn = 0;
    for (int a = 0; a < n; ++a) {
      sn += st[a] * st[a];
      real nv = v[a] + st[a];
      if (!(nv > lo[a]) || !(nv < hi[a])) return false;
    }
    sn = r_sqrt(sn);
    return sn <= Delta;
  };
  auto keep = [&](real eta) { for (int a = 0; a < n; ++a) s[a] = st[a]; *eta_out = eta; *snorm_out = sn; };
  if (attempt((real)0)) { keep((real)0); return true; }
  real eta_lo = 0, eta_hi = 0, eta = eta0;
  bool found = false;
  for (int k = 0; k < 60; ++k) {
    if (attempt(eta)) { eta_hi = eta; keep(eta); found = true; break; }
    eta_lo = eta; eta = eta * growth;
  }
  if (!found) return false;
  for (int k = 0; k < 12; ++k) {
    if (*snorm_out >= Delta / (real)2) break;
    if (eta_lo > (real)0 && eta_hi / eta_lo < ratio_stop) break;
    real mid = (eta_lo > (real)0) ? r_sqrt(eta_lo * eta_hi) : eta_hi / growth;
    if (attempt(mid)) { eta_hi = mid; keep(mid); } else eta_lo = mid;
  }
  return true;
}

// ------------------------------------------------------------------------------------------------
// O5 Stability of the feed for one start (eq. 3-5; Newton: App. B.1).
//   side = +1: vapour-like lnW0 = lnz + lnK ; side = -1: liquid-like lnW0 = lnz - lnK
//   SS (eq. 5): lnW <- d - lnphi(W/sumW), d_i = ln z_i + lnphi_i(z), up to stab_ss_iters iterations,
//   then trust-region Newton in beta = 2 sqrt(W) (B.1), gradient g_i = sqrt(W_i) r_i (B.2a),
//   H_ij = sqrt(W_i W_j) M_ij(w)/sumW + delta_ij (1 + r_i/2) (B.2b as read in C11), Delta_max rule (B.3).
//   tm = 1 + sum W_i (lnW_i + lnphi_i - d_i - 1) (eq. 4 with Michelsen's leading 1, C1);
//   at a stationary point tm = 1 - sumW and tpd = -ln sumW (C2).
// Outputs: lnW, tm, tpd, trivial flag (C7), iterations (ss, tr), cap flag.
// ------------------------------------------------------------------------------------------------
struct StabOut { real lnW[MAXC]; real tm, tpd; int trivial, ss_iters, tr_iters, capped, entered_newton; };

static void stability_trial(const Setup& s, const real* z, const real* lnz, const real* d, const real* lnK, int side,
                            const Opts& o, StabOut& out) {
  const int nc = s.nc;
  real lnW[MAXC], W[MAXC], w[MAXC], lp[MAXC], r[MAXC];
  for (int i = 0; i < nc; ++i) lnW[i] = (z[i] > (real)0) ? lnz[i] + (real)side * lnK[i] : (real)0;
  out.ss_iters = out.tr_iters = 0; out.capped = 0; out.entered_newton = 0;
  bool converged = false;
  real sumW = 0, rmax = 0;
  auto eval = [&](real (*M)[MAXC]) {
    sumW = 0;
    for (int i = 0; i < nc; ++i) { W[i] = (z[i] > (real)0) ? r_exp(lnW[i]) : (real)0; sumW += W[i]; }
    for (int i = 0; i < nc; ++i) w[i] = W[i] / sumW;
    lnphi(s, w, lp, nullptr, M);
    rmax = 0;
    for (int i = 0; i < nc; ++i) {
      r[i] = (z[i] > (real)0) ? lnW[i] + lp[i] - d[i] : (real)0;
      if (r_abs(r[i]) > rmax) rmax = r_abs(r[i]);
    }
  };
  auto tm_full = [&]() { real t = 1; for (int i = 0; i < nc; ++i) t += W[i] * (r[i] - (real)1); return t; };

  const int ss_max = (o.use_newton != 0) ? (int)o.stab_ss_iters : (int)o.ss_cap;
  for (int k = 0; k < ss_max; ++k) {
    eval(nullptr);
    if (rmax < (real)o.tol_ss) { converged = true; break; }
    for (int i = 0; i < nc; ++i) if (z[i] > (real)0) lnW[i] = d[i] - lp[i];                // eq. 5
    out.ss_iters++;
  }
  real tm = 0;
  bool stationary_exact = false;  // true when the last Newton step was applied without re-evaluation
  if (converged) {
    tm = tm_full();
  } else if (o.use_newton == 0) {
    eval(nullptr); tm = tm_full(); out.capped = 1;
  } else {
    // ---- trust-region Newton, B.1-B.3 ----
    out.entered_newton = 1;
    // active components (z_i > 0)
    int idx[MAXC], na = 0;
    for (int i = 0; i < nc; ++i) if (z[i] > (real)0) idx[na++] = i;
    real M[MAXC][MAXC];
    eval(M);
    tm = tm_full();
    real beta[MAXC];
    real bn = 0;
    for (int a = 0; a < na; ++a) { beta[a] = (real)2 * r_sqrt(W[idx[a]]); bn += beta[a] * beta[a]; }
    real Delta = std::max((real)1, r_sqrt(bn) / (real)2);                                   // C11
    const real Delta_cap = (real)8 * Delta;
    const int kmax = (int)o.stab_tr_iters;
    bool done = false;
    for (int it = 0; it < kmax && !done; ++it) {
      if (rmax < (real)o.tol_newton_g) { done = true; converged = true; break; }
      out.tr_iters++;
      real g[MAXC], H[MAXC][MAXC], sstep[MAXC];
      for (int a = 0; a < na; ++a) {
        int i = idx[a];
        g[a] = r_sqrt(W[i]) * r[i];                                                          // B.2a
        for (int b = 0; b < na; ++b) {
          int j = idx[b];
          H[a][b] = r_sqrt(W[i] * W[j]) * M[i][j] / sumW + ((a == b) ? ((real)1 + r[i] / (real)2) : (real)0);  // B.2b / C11
        }
      }
      real eta = 0, snorm = 0, ones[MAXC], lo[MAXC], hi[MAXC];
      for (int a = 0; a < na; ++a) { ones[a] = 1; lo[a] = 0; hi[a] = std::numeric_limits<real>::infinity(); }
      bool ok = tr_subproblem(na, H, g, ones, Delta, (real)1e-3, beta, lo, hi, sstep, &eta, &snorm, (real)o.eta_growth, (real)o.eta_ratio);
      if (!ok) { out.capped = 1; break; }
      real smax = 0;
      for (int a = 0; a < na; ++a) smax = std::max(smax, r_abs(sstep[a]));
      if (eta == (real)0 && smax < (real)o.tol_newton_step) {
        // quadratic-convergence finish: apply the full Newton step and stop (error ~ smax^2)
        for (int a = 0; a < na; ++a) { beta[a] += sstep[a]; real h = beta[a] / (real)2; W[idx[a]] = h * h; lnW[idx[a]] = r_log(W[idx[a]]); }
        sumW = 0; for (int i = 0; i < nc; ++i) sumW += W[i];
        stationary_exact = true; converged = true; done = true; break;
      }
      // predicted reduction
      real pred = 0;
      for (int a = 0; a < na; ++a) {
        real hs = 0;
        for (int b = 0; b < na; ++b) hs += H[a][b] * sstep[b];
        pred += sstep[a] * (g[a] + hs / (real)2);
      }
      // trial point
      real lnW_old[MAXC], W_old[MAXC], r_old[MAXC], M_old[MAXC][MAXC];
      std::memcpy(lnW_old, lnW, sizeof lnW); std::memcpy(W_old, W, sizeof W); std::memcpy(r_old, r, sizeof r);
      std::memcpy(M_old, M, sizeof M);
      real sumW_old = sumW, rmax_old = rmax, tm_old = tm;
      for (int a = 0; a < na; ++a) { real h = (beta[a] + sstep[a]) / (real)2; lnW[idx[a]] = r_log(h * h); }
      eval(M);
      real tm_new = tm_full();
      real act = tm_new - tm_old;
      bool accept = (act < (real)0) || (rmax < rmax_old);
      if (accept) {
        for (int a = 0; a < na; ++a) beta[a] += sstep[a];
        tm = tm_new;
        real ratio = (pred != (real)0) ? r_abs(act / pred) : (real)1;
        if (r_abs(pred) > (real)1e-13) {                                                     // B.3 PAPER.md:485-490
          if (ratio <= (real)0.25) Delta = Delta / (real)2;
          else if (ratio >= (real)0.75) Delta = std::min(Delta * (real)2, Delta_cap);
        }
      } else {
        std::memcpy(lnW, lnW_old, sizeof lnW); std::memcpy(W, W_old, sizeof W); std::memcpy(r, r_old, sizeof r);
        std::memcpy(M, M_old, sizeof M);
        sumW = sumW_old; rmax = rmax_old; tm = tm_old;
        Delta = std::min(Delta, snorm) / (real)2;
      }
    }
    if (!converged) { if (rmax < (real)o.tol_newton_g) converged = true; else out.capped = 1; }
  }
  // results
  real triv = 0;
  for (int i = 0; i < nc; ++i) if (z[i] > (real)0) triv = std::max(triv, r_abs(lnW[i] - lnz[i]));
  out.trivial = (triv < (real)o.trivial_tol) ? 1 : 0;
  for (int i = 0; i < nc; ++i) out.lnW[i] = lnW[i];
  if (out.trivial) { out.tm = 0; out.tpd = 0; }
  else {
    // tm is second-order accurate in the residual r; at a stationary point tm = 1 - sumW and
    // tpd = -ln sumW = -ln(1 - tm) (C2)
    out.tm = stationary_exact ? ((real)1 - sumW) : tm;
    out.tpd = -r_log((real)1 - out.tm);
  }
}

// ------------------------------------------------------------------------------------------------
// O8 Phase split (Fig. 1; Newton: App. B.2).
//   SS: theta <- RR(K, z); x, y; lnK <- lnphi(x) - lnphi(y); r_k = max|dlnK|; stop when r_k < tol and the
//   linear-convergence error estimate eps_k = r_k rho/(1-rho), rho = r_k/r_{k-1}, is < tol, or r_k < 1e-14 (C8).
//   After split_ss_iters SS iterations (and only while 0 < theta < 1): trust-region Newton on the reduced
//   Gibbs energy G (eq. 8) in n^V with gradient (B.5a), Hessian (B.5b with unit-total-mole M, C18), damping
//   matrix D(z/(xy)) (B.4a) and the Delta_max rule (B.3).
// Outputs: theta, x, y, lnK, iterations, status bits.  two_phase = converged with 0 < theta < 1.
// ------------------------------------------------------------------------------------------------
struct SplitOut { real theta, x[MAXC], y[MAXC], lnK[MAXC]; int two_phase, ss_iters, tr_iters, status, entered_newton; real rate, dc; };

static real gibbs_two_phase(int nc, const real* nL, const real* nV, const real* x, const real* y, const real* lpx, const real* lpy) {
  real G = 0;                                                                                // eq. 8
  for (int i = 0; i < nc; ++i) {
    if (nL[i] > (real)0 && x[i] > (real)0) G += nL[i] * (r_log(x[i]) + lpx[i]);
    if (nV[i] > (real)0 && y[i] > (real)0) G += nV[i] * (r_log(y[i]) + lpy[i]);
  }
  return G;
}

// `hinted`: the split was entered through the caller's skip-stability hint (reading C21): a hinted split whose successive
// substitution is still outside 0 < theta < 1 after hint_ss_cap iterations is declared failed at once (the caller's
// estimate points at the wrong side of the phase boundary -- the failure mode of PAPER.md:363 -- and SS would crawl
// towards the trivial solution for up to ss_cap iterations); flash_one then drops the hint and flashes from Wilson.
static void phase_split(const Setup& s, const real* z, const real* lnK_in, const Opts& o, bool hinted, SplitOut& out) {
  const int nc = s.nc;
  real lnK[MAXC], K[MAXC], x[MAXC], y[MAXC], lpx[MAXC], lpy[MAXC];
  for (int i = 0; i < nc; ++i) lnK[i] = lnK_in[i];
  out.ss_iters = out.tr_iters = 0; out.status = 0; out.two_phase = 0; out.rate = 0; out.theta = 0; out.entered_newton = 0;
  real theta = 0, r_prev = -1;
  bool converged = false, failed = false;
  const bool newton = (o.use_newton != 0);
  const int ss_switch = (int)o.split_ss_iters;
  const int ss_cap = (int)o.ss_cap;
  int k = 0;
  bool go_newton = false;
  while (true) {
    // trivial collapse
    real mk = 0;
    for (int i = 0; i < nc; ++i) if (z[i] > (real)0) mk = std::max(mk, r_abs(lnK[i]));
    if (mk < (real)o.split_trivial_tol) { failed = true; break; }
    for (int i = 0; i < nc; ++i) K[i] = r_exp(lnK[i]);
    if (!rachford_rice(nc, K, z, &theta)) { failed = true; break; }
    phases_from_theta(nc, K, z, theta, x, y);
    if (newton && k >= ss_switch && theta > (real)0 && theta < (real)1) { go_newton = true; break; }
    if (k >= ss_cap) { out.status |= ST_SPLIT_CAP; break; }
    if (hinted && k >= (int)o.hint_ss_cap && !(theta > (real)0 && theta < (real)1)) { failed = true; break; }   // C21
    lnphi(s, x, lpx, nullptr, nullptr);
    lnphi(s, y, lpy, nullptr, nullptr);
    real rk = 0;
    for (int i = 0; i < nc; ++i)
      if (z[i] > (real)0) { real nk = lpx[i] - lpy[i]; rk = std::max(rk, r_abs(nk - lnK[i])); lnK[i] = nk; }
    ++k; out.ss_iters = k;
    if (rk < (real)1e-14) { converged = true; }
    else if (r_prev > (real)0 && rk < (real)o.tol_ss) {
      real rho = rk / r_prev;
      out.rate = rho;
      if (rho < (real)1 && rk * rho / ((real)1 - rho) < (real)o.tol_ss) converged = true;
    }
    if (r_prev > (real)0) out.rate = rk / r_prev;
    r_prev = rk;
    if (converged) {
      // x, y, theta consistent with the final lnK
      for (int i = 0; i < nc; ++i) K[i] = r_exp(lnK[i]);
      if (!rachford_rice(nc, K, z, &theta)) { failed = true; converged = false; }
      else phases_from_theta(nc, K, z, theta, x, y);
      break;
    }
  }

  if (go_newton) {
    // ---- trust-region Newton on G in n^V, B.4-B.5 ----
    out.entered_newton = 1;
    int idx[MAXC], na = 0;
    for (int i = 0; i < nc; ++i) if (z[i] > (real)0) idx[na++] = i;
    real nV[MAXC], nL[MAXC], Mx[MAXC][MAXC], My[MAXC][MAXC], gt[MAXC];
    for (int i = 0; i < nc; ++i) { nV[i] = theta * y[i]; if (nV[i] > z[i]) nV[i] = z[i]; nL[i] = z[i] - nV[i]; }
    real G = 0, gmax = 0;
    auto eval = [&]() {
      theta = 0; for (int i = 0; i < nc; ++i) theta += nV[i];
      for (int i = 0; i < nc; ++i) { nL[i] = z[i] - nV[i]; y[i] = nV[i] / theta; x[i] = nL[i] / ((real)1 - theta); }
      lnphi(s, x, lpx, nullptr, Mx);
      lnphi(s, y, lpy, nullptr, My);
      gmax = 0;
      for (int i = 0; i < nc; ++i) {
        gt[i] = (z[i] > (real)0) ? (r_log(y[i]) + lpy[i] - r_log(x[i]) - lpx[i]) : (real)0;   // B.5a
        gmax = std::max(gmax, r_abs(gt[i]));
      }
      G = gibbs_two_phase(nc, nL, nV, x, y, lpx, lpy);
    };
    eval();
    real Delta = (real)0.25;   // n^V lives in the box (0, z), |n^V| < 1; Delta is capped at 1 (C11)
    const int kmax = hinted ? std::min((int)o.split_tr_iters, (int)o.hint_tr_cap) : (int)o.split_tr_iters;   // C21
    for (int it = 0; it < kmax; ++it) {
      // Reading C8: the gradient test does not end the iteration by itself.  Near a critical point (d_c -> 0, eq. 14
      // PAPER.md:318) and next to the phase boundary the Hessian is nearly singular, so a gradient below 1e-12 does not
      // bound the error of n^V (error ~ gradient / smallest eigenvalue); the Newton step is the error estimate.  A
      // gradient below the target therefore triggers ONE last full Newton step ("polish"), applied if it is admissible.
      const bool last = gmax < (real)o.tol_newton_g;
      if (!last) out.tr_iters++;
      real g[MAXC], H[MAXC][MAXC], D[MAXC], sstep[MAXC];
      const real tt = theta * ((real)1 - theta);
      for (int a = 0; a < na; ++a) {
        int i = idx[a];
        g[a] = gt[i];
        D[a] = z[i] / (x[i] * y[i]);
        for (int b = 0; b < na; ++b) {
          int j = idx[b];
          H[a][b] = (((a == b) ? D[a] : (real)0) - (real)1 + theta * Mx[i][j] + ((real)1 - theta) * My[i][j]) / tt;  // B.5b / C18
        }
      }
      real eta = 0, snorm = 0, va[MAXC], lo[MAXC], hi[MAXC];
      for (int a = 0; a < na; ++a) { va[a] = nV[idx[a]]; lo[a] = 0; hi[a] = z[idx[a]]; }
      bool ok = tr_subproblem(na, H, g, D, Delta, (real)1e-3 / tt, va, lo, hi, sstep, &eta, &snorm, (real)o.eta_growth, (real)o.eta_ratio);   // B.4a
      if (!ok) { if (last) converged = true; else out.status |= ST_SPLIT_CAP; break; }
      real smax = 0;
      for (int a = 0; a < na; ++a) smax = std::max(smax, r_abs(sstep[a]));
      if (last && eta != (real)0) { converged = true; break; }   // no admissible full step: keep the evaluated point
      if (eta == (real)0 && (last || smax < (real)o.tol_newton_step)) {
        for (int a = 0; a < na; ++a) nV[idx[a]] += sstep[a];
        theta = 0; for (int i = 0; i < nc; ++i) theta += nV[i];
        for (int i = 0; i < nc; ++i) { nL[i] = z[i] - nV[i]; y[i] = nV[i] / theta; x[i] = nL[i] / ((real)1 - theta); }
        converged = true; break;
      }
      real pred = 0;
      for (int a = 0; a < na; ++a) {
        real hs = 0;
        for (int b = 0; b < na; ++b) hs += H[a][b] * sstep[b];
        pred += sstep[a] * (g[a] + hs / (real)2);
      }
      real nV_old[MAXC], Mx_old[MAXC][MAXC], My_old[MAXC][MAXC];
      std::memcpy(nV_old, nV, sizeof nV); std::memcpy(Mx_old, Mx, sizeof Mx); std::memcpy(My_old, My, sizeof My);
      real G_old = G, gmax_old = gmax;
      for (int a = 0; a < na; ++a) nV[idx[a]] += sstep[a];
      eval();
      real act = G - G_old;
      // accept if G fell; a smaller gradient is accepted instead only where the change of G is below its rounding
      // resolution (next to the solution), so that the iteration is a descent method on G everywhere else (reading C11)
      bool accept = (act < (real)0) || (gmax < gmax_old && act <= (real)1e-12 * r_abs(G_old));
      if (accept) {
        real ratio = (pred != (real)0) ? r_abs(act / pred) : (real)1;
        if (r_abs(pred) > (real)1e-13) {
          if (ratio <= (real)0.25) Delta = Delta / (real)2;
          else if (ratio >= (real)0.75) Delta = std::min(Delta * (real)2, (real)1);
        }
      } else {
        std::memcpy(nV, nV_old, sizeof nV);
        eval();  // restores x, y, lnphi, M, G, gmax at the old point (plain, not clever)
        (void)Mx_old; (void)My_old;
        Delta = std::min(Delta, snorm) / (real)2;
      }
    }
    if (!converged) { if (gmax < (real)o.tol_newton_g) converged = true; else out.status |= ST_SPLIT_CAP; }
    for (int i = 0; i < nc; ++i) lnK[i] = (z[i] > (real)0) ? r_log(y[i]) - r_log(x[i]) : lnK[i];
    // the Newton iteration can also slide into the trivial solution x = y (G is flat there): same test as in the SS loop
    real mkn = 0;
    for (int i = 0; i < nc; ++i) if (z[i] > (real)0) mkn = std::max(mkn, r_abs(lnK[i]));
    if (mkn < (real)o.split_trivial_tol) failed = true;
  }

  out.theta = theta;
  real dc = 0;
  for (int i = 0; i < nc; ++i) { out.x[i] = x[i]; out.y[i] = y[i]; out.lnK[i] = lnK[i]; if (z[i] > (real)0) dc += lnK[i] * lnK[i]; }
  out.dc = r_sqrt(dc);                                                                       // eq. 14
  if (failed) { out.status |= ST_SPLIT_FAILED; return; }
  if (converged && theta > (real)0 && theta < (real)1) out.two_phase = 1;
  else if (converged) out.status |= ST_SPLIT_FAILED;   // converged outside (0,1): reported, not relabelled silently
}

// ------------------------------------------------------------------------------------------------
// Whole flash, Algorithm O (section 2.2.3, Fig. 2 as described).
// ------------------------------------------------------------------------------------------------
struct FlashOut {
  int phase, iters, status, stab_iters, probe_case;
  real beta, x[MAXC], y[MAXC], lnK[MAXC], tpd_min, Zfeed, dc, rate;
  real dbeta_dK[MAXC];   // eq. 13 at the reported (beta, K = y / x); NaN unless two phases
  // per-stage counts (the columns of the paper's profiler, Table 4), summed over a warm restart
  int stab_ss[2], stab_tr[2], stab_newton_trials, split_ss, split_tr, split_entered, split_newton;
  int stab_entered_tr[2], stab_capped[2];   // per start: went on to the trust-region stage / hit an iteration cap
};

static void flash_one(int nc, const double* Tc, const double* Pc, const double* omega, const double* kij,
                      real P, real T, const real* z_in, const real* lnK0, int flags, const Opts& o, FlashOut& out) {
  const real* z = z_in;
  const real nan = std::numeric_limits<real>::quiet_NaN();
  out.phase = -1; out.iters = 0; out.status = 0; out.stab_iters = 0; out.probe_case = 0;
  out.beta = nan; out.tpd_min = nan; out.Zfeed = nan; out.dc = 0; out.rate = 0;
  out.stab_ss[0] = out.stab_ss[1] = out.stab_tr[0] = out.stab_tr[1] = 0;
  out.stab_newton_trials = out.split_ss = out.split_tr = out.split_entered = out.split_newton = 0;
  out.stab_entered_tr[0] = out.stab_entered_tr[1] = out.stab_capped[0] = out.stab_capped[1] = 0;
  for (int i = 0; i < nc; ++i) { out.x[i] = nan; out.y[i] = nan; out.lnK[i] = nan; out.dbeta_dK[i] = nan; }
  // O0 validate
  bool ok = std::isfinite((double)P) && std::isfinite((double)T) && P > (real)0 && T > (real)0;
  real sz = 0;
  for (int i = 0; i < nc; ++i) { if (!std::isfinite((double)z[i]) || z[i] < (real)0) ok = false; sz += z[i]; }
  if (!ok || !(r_abs(sz - (real)1) <= (real)1e-9)) return;
  // the feed is normalised once (z <- z / sum z) so that every identity below holds with sum z = 1
  // exactly to rounding (reading C20); single-phase outputs return this z.
  real zn[MAXC];
  for (int i = 0; i < nc; ++i) zn[i] = z_in[i] / sz;
  z = zn;

  Setup s;
  setup(nc, Tc, Pc, omega, kij, P, T, s);
  real lnz[MAXC], d[MAXC], lpz[MAXC], Zf;
  lnphi(s, z, lpz, &Zf, nullptr);
  out.Zfeed = Zf;
  for (int i = 0; i < nc; ++i) { lnz[i] = (z[i] > (real)0) ? r_log(z[i]) : (real)0; d[i] = lnz[i] + lpz[i]; }

  // O3 Wilson or caller-supplied lnK0 (bit1 / bit0 of flags; non-finite or |lnK0| > 700 -> Wilson)
  real lnKw[MAXC];
  wilson_lnK(nc, Tc, Pc, omega, P, T, lnKw);
  bool have0 = false;
  if (lnK0 && (flags & 3)) {
    have0 = true;
    for (int i = 0; i < nc; ++i) if (!std::isfinite((double)lnK0[i]) || r_abs(lnK0[i]) > (real)700) have0 = false;
    if (!have0) out.status |= ST_LNK0_REJECTED;   // overflowing / non-finite estimates are ignored and reported
  }
  real lnKs[MAXC];
  for (int i = 0; i < nc; ++i) lnKs[i] = have0 ? lnK0[i] : lnKw[i];
  const bool skip_stab = have0 && (flags & 1);

  real lnK[MAXC];
  for (int i = 0; i < nc; ++i) lnK[i] = lnKs[i];
  bool unstable = false;
  real tpd_min = 0;

  if (!skip_stab) {
    // O4 probe: 3 phase-split SS iterations
    real K[MAXC], x[MAXC], y[MAXC], lpx[MAXC], lpy[MAXC], theta = 0;
    int pcase = 0;
    const int np = (int)o.probe_iters;
    for (int it = 0; it < np; ++it) {
      for (int i = 0; i < nc; ++i) K[i] = r_exp(lnK[i]);
      if (!rachford_rice(nc, K, z, &theta) || !(theta > (real)0) || !(theta < (real)1)) { pcase = 1; break; }
      phases_from_theta(nc, K, z, theta, x, y);
      lnphi(s, x, lpx, nullptr, nullptr);
      lnphi(s, y, lpy, nullptr, nullptr);
      for (int i = 0; i < nc; ++i) if (z[i] > (real)0) lnK[i] = lpx[i] - lpy[i];
      out.iters++;
    }
    if (np == 0) pcase = 2;   // probe disabled: every mixture goes through the full stability analysis
    if (pcase == 0) {
      real tx = tpd_of(nc, x, lpx, d), ty = tpd_of(nc, y, lpy, d);
      real dG = ((real)1 - theta) * tx + theta * ty;                                         // C5
      real mn = std::min(dG, std::min(tx, ty));
      if (mn < -(real)o.probe_margin) { pcase = 3; unstable = true; tpd_min = mn; }
      else pcase = 2;
    }
    out.probe_case = pcase;
    if (pcase != 3) {
      // O5 stability with the Wilson / caller K (C19)
      StabOut sv, sl;
      stability_trial(s, z, lnz, d, lnKs, +1, o, sv);
      stability_trial(s, z, lnz, d, lnKs, -1, o, sl);
      out.stab_iters = sv.ss_iters + sv.tr_iters + sl.ss_iters + sl.tr_iters;
      out.stab_ss[0] = sv.ss_iters; out.stab_ss[1] = sl.ss_iters; out.stab_tr[0] = sv.tr_iters; out.stab_tr[1] = sl.tr_iters;
      out.stab_newton_trials = (sv.entered_newton ? 1 : 0) + (sl.entered_newton ? 1 : 0);
      out.stab_entered_tr[0] = sv.entered_newton ? 1 : 0; out.stab_entered_tr[1] = sl.entered_newton ? 1 : 0;
      out.stab_capped[0] = sv.capped ? 1 : 0; out.stab_capped[1] = sl.capped ? 1 : 0;
      if (sv.capped || sl.capped) out.status |= ST_STAB_CAP;
      // O7 label
      tpd_min = 0;
      bool any = false;
      if (!sv.trivial) { tpd_min = sv.tpd; any = true; }
      if (!sl.trivial) { tpd_min = any ? std::min(tpd_min, sl.tpd) : sl.tpd; any = true; }
      if (!any) tpd_min = 0;
      unstable = tpd_min < (real)0;
      if (tpd_min != (real)0 && r_abs(tpd_min) < (real)o.band) out.status |= ST_BAND;
      if (unstable) {
        if (sl.tm < sv.tm) for (int i = 0; i < nc; ++i) lnK[i] = lnz[i] - sl.lnW[i];         // PAPER.md:79, C10
        else for (int i = 0; i < nc; ++i) lnK[i] = sv.lnW[i] - lnz[i];
      }
    }
  } else {
    unstable = true; tpd_min = nan; out.probe_case = 4;
  }
  out.tpd_min = tpd_min;

  if (o.stability_only != 0) {
    // Stability-only mode ("determine stability (no need for phase split calculations)"): the label of
    // Fig. 2 up to the entry of the phase split.  phase = 2 means "unstable" (a split would be attempted), 1 "stable";
    // x = y = z; beta is the single-phase convention for a stable feed and NaN for an unstable one (not computed);
    // lnK is the K that would seed the split (probe iterate, or the stability trial's).
    out.phase = unstable ? 2 : 1;
    out.beta = unstable ? nan : ((Zf > (real)1 / (real)3) ? (real)1 : (real)0);
    for (int i = 0; i < nc; ++i) { out.x[i] = z[i]; out.y[i] = z[i]; out.lnK[i] = unstable ? ((z[i] > (real)0) ? lnK[i] : (real)0) : (real)0; }
    return;
  }

  bool two = false;
  if (unstable) {
    SplitOut sp;
    phase_split(s, z, lnK, o, skip_stab, sp);
    out.iters += sp.ss_iters + sp.tr_iters;
    out.split_ss = sp.ss_iters; out.split_tr = sp.tr_iters; out.split_entered = 1; out.split_newton = sp.entered_newton;
    out.status |= sp.status;
    out.dc = sp.dc; out.rate = sp.rate;
    if (sp.two_phase) {
      two = true;
      out.phase = 2; out.beta = sp.theta;
      for (int i = 0; i < nc; ++i) { out.x[i] = sp.x[i]; out.y[i] = sp.y[i]; out.lnK[i] = sp.lnK[i]; }
      // Phase identity (reading C23): the phase with the larger compressibility factor is
      // reported as the vapour y ("smallest root ... liquid phase ... largest ... vapor").  Without this
      // the identity follows the sign of the K that seeded the split, and when both stability starts reach the SAME
      // stationary point (tm^L = tm^V up to rounding) the paper's rule "tm^L < tm^V" is decided by noise.
      real lpt[MAXC], Zx, Zy;
      lnphi(s, sp.x, lpt, &Zx, nullptr);
      lnphi(s, sp.y, lpt, &Zy, nullptr);
      if (Zy < Zx) {
        out.beta = (real)1 - sp.theta;
        for (int i = 0; i < nc; ++i) { out.x[i] = sp.y[i]; out.y[i] = sp.x[i]; out.lnK[i] = -sp.lnK[i]; }
      }
      // derivative output, eq. 13, at the reported solution (K = y / x solves f_RR(beta, K) = 0)
      real Kr[MAXC];
      for (int i = 0; i < nc; ++i) Kr[i] = (z[i] > (real)0) ? out.y[i] / out.x[i] : (real)1;
      rr_dtheta_dK(nc, Kr, z, out.beta, out.dbeta_dK);
    } else if (!(sp.status & ST_SPLIT_FAILED)) out.status |= ST_SPLIT_FAILED;
  }
  if (!two && skip_stab) {
    // The caller's "known unstable + lnK0" hint did not lead to a two-phase solution (trivial collapse, theta outside
    // (0,1) or an iteration cap -- cf. the initializer-only failure reported at PAPER.md:363).  The hint is dropped and
    // the mixture is flashed again from Wilson with the full stability analysis; the restart is reported (reading C21).
    FlashOut cold;
    flash_one(nc, Tc, Pc, omega, kij, P, T, z_in, nullptr, 0, o, cold);
    cold.iters += out.iters;
    cold.status |= ST_WARM_RESTART | (out.status & ST_LNK0_REJECTED);
    cold.split_ss += out.split_ss; cold.split_tr += out.split_tr; cold.split_entered += 1; cold.split_newton += out.split_newton;
    out = cold;
    return;
  }
  if (!two) {
    // single phase: x = y = z, beta = 1 iff Z_feed > 1/3 (convention)
    out.phase = 1;
    out.beta = (Zf > (real)1 / (real)3) ? (real)1 : (real)0;
    for (int i = 0; i < nc; ++i) { out.x[i] = z[i]; out.y[i] = z[i]; out.lnK[i] = (real)0; }
  }
}

// ================================================================================================
// C entry points (ctypes).  All arrays are HOST double; z/x/y/lnK are [nc][N] component-major.
// ================================================================================================
extern "C" {

int orc_real_bytes() { return (int)sizeof(real); }
int orc_num_opts() { return NOPTS; }
void orc_default_opts(double* o) { Opts d = default_opts(); std::memcpy(o, &d, sizeof(double) * NOPTS); }

// cubic: all real roots (unfiltered, ascending); closed != 0 -> trigonometric/Cardano pin routine
int orc_cubic_roots(double A, double B, double* r, int closed) {
  real rr[3] = {0, 0, 0};
  int n = closed ? cubic_roots_closed((real)A, (real)B, rr) : cubic_roots((real)A, (real)B, rr);
  for (int k = 0; k < 3; ++k) r[k] = (double)rr[k];
  return n;
}
double orc_choose_root(double A, double B) { return (double)choose_root((real)A, (real)B); }
double orc_gibbs_of_root(double Z, double A, double B) { return (double)gibbs_of_root((real)Z, (real)A, (real)B); }

// setup: Ai[nc], Bi[nc], Aij[nc*nc]
void orc_setup(int nc, const double* Tc, const double* Pc, const double* omega, const double* kij,
               double P, double T, double* Ai, double* Bi, double* Aij) {
  Setup s; setup(nc, Tc, Pc, omega, kij, (real)P, (real)T, s);
  for (int i = 0; i < nc; ++i) { Ai[i] = (double)s.Ai[i]; Bi[i] = (double)s.Bi[i]; for (int j = 0; j < nc; ++j) Aij[i * nc + j] = (double)s.Aij[i][j]; }
}

// lnphi (and optionally M[nc*nc]) of one composition c[nc]
void orc_lnphi(int nc, const double* Tc, const double* Pc, const double* omega, const double* kij,
               double P, double T, const double* c, double* out, double* Z, double* M) {
  Setup s; setup(nc, Tc, Pc, omega, kij, (real)P, (real)T, s);
  real cc[MAXC], lp[MAXC], Zr, Mm[MAXC][MAXC];
  for (int i = 0; i < nc; ++i) cc[i] = (real)c[i];
  lnphi(s, cc, lp, &Zr, M ? Mm : nullptr);
  for (int i = 0; i < nc; ++i) out[i] = (double)lp[i];
  if (Z) *Z = (double)Zr;
  if (M) for (int i = 0; i < nc; ++i) for (int j = 0; j < nc; ++j) M[i * nc + j] = (double)Mm[i][j];
}

// lnphi for n compositions c[n][nc] (row-major, one composition per row) at the same (P, T); out[n][nc], Z[n]
void orc_lnphi_many(int nc, const double* Tc, const double* Pc, const double* omega, const double* kij,
                    double P, double T, int64_t n, const double* c, double* out, double* Z) {
  Setup s; setup(nc, Tc, Pc, omega, kij, (real)P, (real)T, s);
  for (int64_t k = 0; k < n; ++k) {
    real cc[MAXC], lp[MAXC], Zr;
    for (int i = 0; i < nc; ++i) cc[i] = (real)c[k * nc + i];
    lnphi(s, cc, lp, &Zr, nullptr);
    for (int i = 0; i < nc; ++i) out[k * nc + i] = (double)lp[i];
    if (Z) Z[k] = (double)Zr;
  }
}

void orc_wilson(int nc, const double* Tc, const double* Pc, const double* omega, double P, double T, double* lnK) {
  real l[MAXC]; wilson_lnK(nc, Tc, Pc, omega, (real)P, (real)T, l);
  for (int i = 0; i < nc; ++i) lnK[i] = (double)l[i];
}

// Rachford-Rice: returns 1 and theta if a window exists, else 0; also f_RR at a given theta
int orc_rachford_rice(int nc, const double* K, const double* z, double* theta) {
  real k[MAXC], zz[MAXC], th = 0;
  for (int i = 0; i < nc; ++i) { k[i] = (real)K[i]; zz[i] = (real)z[i]; }
  bool ok = rachford_rice(nc, k, zz, &th);
  *theta = (double)th;
  return ok ? 1 : 0;
}
// eq. 13: d theta / d K at (theta, K)
void orc_rr_dtheta_dK(int nc, const double* K, const double* z, double theta, double* dth) {
  real k[MAXC], zz[MAXC], d[MAXC];
  for (int i = 0; i < nc; ++i) { k[i] = (real)K[i]; zz[i] = (real)z[i]; }
  rr_dtheta_dK(nc, k, zz, (real)theta, d);
  for (int i = 0; i < nc; ++i) dth[i] = (double)d[i];
}
// Batched Rachford-Rice (what the paper's initializer training calls): per mixture theta from (lnK, z),
// x, y (eq. 7 / PAPER.md:83) and d theta / d K (eq. 13).  lnK, z, x, y, dth are [nc][N]; no window -> theta = NaN, ok = 0.
void orc_rr_batch(int nc, int64_t N, const double* lnK, const double* z, double* theta, double* x, double* y, double* dth, int32_t* ok) {
  const real nan = std::numeric_limits<real>::quiet_NaN();
  for (int64_t n = 0; n < N; ++n) {
    real k[MAXC], zz[MAXC], xx[MAXC], yy[MAXC], d[MAXC], th = nan, sz = 0;
    for (int i = 0; i < nc; ++i) { k[i] = r_exp((real)lnK[(int64_t)i * N + n]); zz[i] = (real)z[(int64_t)i * N + n]; sz += zz[i]; }
    for (int i = 0; i < nc; ++i) zz[i] /= sz;
    const bool good = rachford_rice(nc, k, zz, &th);
    if (good) { phases_from_theta(nc, k, zz, th, xx, yy); rr_dtheta_dK(nc, k, zz, th, d); }
    theta[n] = good ? (double)th : (double)nan;
    if (ok) ok[n] = good ? 1 : 0;
    for (int i = 0; i < nc; ++i) {
      if (x) x[(int64_t)i * N + n] = good ? (double)xx[i] : (double)nan;
      if (y) y[(int64_t)i * N + n] = good ? (double)yy[i] : (double)nan;
      if (dth) dth[(int64_t)i * N + n] = good ? (double)d[i] : (double)nan;
    }
  }
}
double orc_rr_f(int nc, const double* K, const double* z, double theta) {
  real k[MAXC], zz[MAXC];
  for (int i = 0; i < nc; ++i) { k[i] = (real)K[i]; zz[i] = (real)z[i]; }
  return (double)rr_f(nc, k, zz, (real)theta);
}

// one stability trial of feed z with seed lnK and side (+1 vapour-like, -1 liquid-like)
// res = {tm, tpd, trivial, ss_iters, tr_iters, capped}
void orc_stability_trial(int nc, const double* Tc, const double* Pc, const double* omega, const double* kij,
                         double P, double T, const double* z, const double* lnK, int side, const double* opts,
                         double* lnW, double* res) {
  Opts o = opts_from(opts);
  Setup s; setup(nc, Tc, Pc, omega, kij, (real)P, (real)T, s);
  real zz[MAXC], lnz[MAXC], d[MAXC], lp[MAXC], lk[MAXC];
  for (int i = 0; i < nc; ++i) { zz[i] = (real)z[i]; lk[i] = (real)lnK[i]; }
  lnphi(s, zz, lp, nullptr, nullptr);
  for (int i = 0; i < nc; ++i) { lnz[i] = (zz[i] > 0) ? r_log(zz[i]) : (real)0; d[i] = lnz[i] + lp[i]; }
  StabOut so; stability_trial(s, zz, lnz, d, lk, side, o, so);
  for (int i = 0; i < nc; ++i) lnW[i] = (double)so.lnW[i];
  res[0] = (double)so.tm; res[1] = (double)so.tpd; res[2] = so.trivial; res[3] = so.ss_iters; res[4] = so.tr_iters; res[5] = so.capped;
}

// phase split from a given lnK.  res = {theta, two_phase, ss_iters, tr_iters, status, rate, dc}
void orc_phase_split(int nc, const double* Tc, const double* Pc, const double* omega, const double* kij,
                     double P, double T, const double* z, const double* lnK, const double* opts,
                     double* x, double* y, double* lnK_out, double* res) {
  Opts o = opts_from(opts);
  Setup s; setup(nc, Tc, Pc, omega, kij, (real)P, (real)T, s);
  real zz[MAXC], lk[MAXC];
  for (int i = 0; i < nc; ++i) { zz[i] = (real)z[i]; lk[i] = (real)lnK[i]; }
  SplitOut sp; phase_split(s, zz, lk, o, false, sp);
  for (int i = 0; i < nc; ++i) { x[i] = (double)sp.x[i]; y[i] = (double)sp.y[i]; lnK_out[i] = (double)sp.lnK[i]; }
  res[0] = (double)sp.theta; res[1] = sp.two_phase; res[2] = sp.ss_iters; res[3] = sp.tr_iters; res[4] = sp.status;
  res[5] = (double)sp.rate; res[6] = (double)sp.dc;
}

// Batched flash (the oracle of ptflash_flash / ptflash_flash_ex).  lnK0 [nc][N] and flags [N] may be NULL.
// Optional outputs (may be NULL): tpd_min [N], lnK [nc][N], status [N], stab_iters [N], probe_case [N],
// diag [3][N] = {Z_feed, d_c, last SS rate}; stage [9][N] int32 = {stability SS iterations vapour-like, liquid-like,
// trust-region iterations vapour-like, liquid-like, trials that entered the Newton stage, split SS iterations, split
// trust-region iterations, splits entered, splits that entered the Newton stage}.
// nthreads <= 1 -> serial; otherwise OpenMP over mixtures.
// Returns the number of threads actually used.
int orc_flash_batch(int nc, const double* Tc, const double* Pc, const double* omega, const double* kij,
                    int64_t N, const double* z, const double* P, const double* T,
                    const double* lnK0, const uint8_t* flags, const double* opts,
                    double* out_beta, double* out_x, double* out_y, int32_t* out_phase, int32_t* out_iters,
                    double* out_tpd_min, double* out_lnK, int32_t* out_status, int32_t* out_stab_iters,
                    int32_t* out_probe_case, double* out_diag, int32_t* out_stage, double* out_dbeta_dK, int nthreads) {
  Opts o = opts_from(opts);
  int used = 1;
#ifdef _OPENMP
  if (nthreads > 1) used = nthreads;
#pragma omp parallel for schedule(dynamic, 256) num_threads(used)
#endif
  for (int64_t n = 0; n < N; ++n) {
    real zz[MAXC], l0[MAXC];
    for (int i = 0; i < nc; ++i) { zz[i] = (real)z[(int64_t)i * N + n]; if (lnK0) l0[i] = (real)lnK0[(int64_t)i * N + n]; }
    FlashOut fo;
    flash_one(nc, Tc, Pc, omega, kij, (real)P[n], (real)T[n], zz, lnK0 ? l0 : nullptr, flags ? flags[n] : 0, o, fo);
    out_beta[n] = (double)fo.beta; out_phase[n] = fo.phase;
    if (out_iters) out_iters[n] = fo.iters;
    for (int i = 0; i < nc; ++i) {
      out_x[(int64_t)i * N + n] = (double)fo.x[i]; out_y[(int64_t)i * N + n] = (double)fo.y[i];
      if (out_lnK) out_lnK[(int64_t)i * N + n] = (double)fo.lnK[i];
    }
    if (out_tpd_min) out_tpd_min[n] = (double)fo.tpd_min;
    if (out_status) out_status[n] = fo.status;
    if (out_stab_iters) out_stab_iters[n] = fo.stab_iters;
    if (out_probe_case) out_probe_case[n] = fo.probe_case;
    if (out_diag) { out_diag[n] = (double)fo.Zfeed; out_diag[N + n] = (double)fo.dc; out_diag[2 * N + n] = (double)fo.rate; }
    if (out_stage) {
      const int v[13] = {fo.stab_ss[0], fo.stab_ss[1], fo.stab_tr[0], fo.stab_tr[1], fo.stab_newton_trials, fo.split_ss, fo.split_tr,
                         fo.split_entered, fo.split_newton, fo.stab_entered_tr[0], fo.stab_entered_tr[1], fo.stab_capped[0], fo.stab_capped[1]};
      for (int k = 0; k < 13; ++k) out_stage[(int64_t)k * N + n] = v[k];
    }
    if (out_dbeta_dK) for (int i = 0; i < nc; ++i) out_dbeta_dK[(int64_t)i * N + n] = (double)fo.dbeta_dK[i];
  }
  return used;
}

}  // extern "C"
