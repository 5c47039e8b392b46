// ptflash_newton.cuh -- trust-region Newton stages of engine 1 (B.1-B.3 stability, B.4-B.5 phase split),
// third generation: matrix-free Hessian rows + row-wise Cholesky with the factor in shared memory.
//
// Why: the second-generation kernels (k2_*_newton) kept the packed nc x nc Hessian in registers (110 registers at
// nc = 10) next to the lane state of the refill loop; at 255 registers they spilled to local memory (the split kernel
// moved 3.7 GB through DRAM for 2.3 GFLOP of work) and ran two warps per scheduler.  Here
//   * the Hessian is never stored: M = n dlnphi/dn is a bilinear form in the basis F_i = (1, B_i, S_i),
//         M_ij = sum_ab F_ia C_ab F_jb - 2 q A_ij          (C: 3 x 3 from the scalars of the cubic, mc3() below),
//     so row i of H is generated in registers from C F_i (9 FMAs) and four per-component vectors, 5-6 FMAs per entry;
//   * the Cholesky is row-wise (Banachiewicz): the current row lives in registers, finished rows L[j][.] are read from
//     shared memory (one LDS per FMA, conflict-free: element k of thread t at [k * 128 + t]), the forward substitution
//     is fused into the row loop, the inverse diagonal stays in registers;
//   * the lane state that must survive a trip (accepted point, pending step) is parked in shared memory, so the
//     register file only holds what the current phase of the trip needs.
// The trust-region logic (EtaSearch, acceptance rule, B.3 radius update, lane refill from a ticket) is unchanged.
#pragma once
#include "ptflash_fast.cuh"
#include "ptflash_staged.cuh"

namespace ptf {

#ifndef PTF_NEWTON_THREADS
#define PTF_NEWTON_THREADS 128
#endif
constexpr int NEWTON_THREADS = PTF_NEWTON_THREADS;

#ifndef PTF_CHOL_R
#define PTF_CHOL_R 2   // rows eliminated together by the row-wise Cholesky of the Newton kernels
#endif
#ifndef PTF_NEWTON_CTA_SYNC
#define PTF_NEWTON_CTA_SYNC 1
#endif

// Coefficients of M_ij = sum_ab F_ia C[a][b] F_jb - q2 A_ij with F_i = (1, B_i, S_i) (B_i, not B_i/B).
// Derivation: DESIGN.md section 2 (M_ij = e_i p_j + c_j - Dq_j u_i + 2q(S_i - A_ij) with p, c, Dq affine in
// e_j - 1 and S_j - A, u_i = 2 S_i - A e_i, e_i = B_i/B).
struct MC3 {
  double c00, c01, c02, c10, c11, c12, c20, c21, c22, q2;
};
__device__ __forceinline__ MC3 mc3(const Eos& e) {
  const double A = e.A, B = e.B, Z = e.Z, q = e.q;
  const double FZ = fma(fma(3.0, Z, -2.0), Z, A - B - B * B);
  const double iFZ = rcp_fast(FZ);
  const double ZA = -(Z - B) * iFZ;
  const double ZB = fma(1.0 + 2.0 * B, Z, A) * iFZ;
  const double iZZB = rcp_fast(Z * (Z + B));
  const double invB = rcp_fast(B);
  const double invZmB = rcp_fast(Z - B);
  const double q2 = 2.0 * q;
  const double zA2 = 2.0 * ZA, zBB = ZB * B;
  const double p1 = zBB - (Z - 1.0) - q * A, p2 = zA2 + q2, p0 = -p1 - p2 * A;
  const double c1 = -(zBB - B) * invZmB, c2 = -zA2 * invZmB, c0 = -c1 - c2 * A;
  const double d1 = (Z - zBB) * iZZB - q, d2 = -zA2 * iZZB, d0 = -d1 - d2 * A;
  MC3 m;
  m.q2 = q2;
  m.c00 = c0;
  m.c01 = c1 * invB;
  m.c02 = c2;
  m.c10 = fma(A, d0, p0) * invB;
  m.c11 = fma(A, d1, p1) * invB * invB;
  m.c12 = fma(A, d2, p2) * invB;
  m.c20 = q2 - 2.0 * d0;
  m.c21 = -2.0 * d1 * invB;
  m.c22 = -2.0 * d2;
  return m;
}

// strict lower triangle of the Cholesky factor, one column of shared memory per thread
// (volatile: without it the compiler forwards every stored L[i][j] to its later loads -- all indices are compile-time --
// and the factor is back in registers, 255 of them plus spills)
template <int NC>
struct LRows {
  volatile double* p;
  __device__ __forceinline__ volatile double& at(int i, int j) const { return p[(i * (i - 1) / 2 + j) * NEWTON_THREADS]; }
};

// Eliminate row i of a row-wise Cholesky.  On entry row[0..i] = H[i][0..i]; on exit row[j < i] = L[i][j], invd[i] = 1 / L[i][i],
// yv[i] = forward substitution of rhs.  Rows 1 .. NC-2 are stored to shared memory; the LAST row is never read by a later
// row, so it stays in registers and the first step of the back substitution is taken right here (s[NC-1], yv updated).
// `i` is a compile-time constant after unrolling, so every j < i / k < j test disappears.
// MOD (modified Cholesky): a pivot that is not safely positive is replaced by max(-pivot, 1e-10 |H_ii|) and pd is cleared --
// the factor then belongs to H + E with a diagonal E >= 0, so the solve still gives a descent direction (a negative
// curvature direction is followed with its Newton length, sign flipped).
template <int NC>
__device__ __forceinline__ void chol_row(const int i, double (&row)[NC], const LRows<NC>& L, double (&invd)[NC],
                                         double (&yv)[NC], double (&s)[NC], const double rhs, bool& pd, const bool MOD = false) {
  const double hii = row[i];
#pragma unroll
  for (int j = 0; j < NC; ++j) {
    if (j < i) {
      double acc = row[j];
#pragma unroll
      for (int k = 0; k < NC; ++k)
        if (k < j) acc = fma(-row[k], L.at(j, k), acc);
      row[j] = acc * invd[j];
    }
  }
  double acc = row[i], a = rhs;
#pragma unroll
  for (int k = 0; k < NC; ++k)
    if (k < i) { acc = fma(-row[k], row[k], acc); a = fma(-row[k], yv[k], a); }
  if (MOD) {
    const double fl = 1.0e-10 * fabs(hii);
    if (!(acc > fl)) { acc = dmax(-acc, fl); pd = false; }
  } else {
    pd = pd && (acc > 0.0);
  }
  const double inv = rsqrt_fast(acc);
  invd[i] = inv;
  yv[i] = a * inv;
  if (i < NC - 1) {
#pragma unroll
    for (int j = 0; j < NC; ++j)
      if (j < i) L.at(i, j) = row[j];
  } else {
    const double sl = yv[i] * inv;
    s[i] = sl;
#pragma unroll
    for (int k = 0; k < NC; ++k)
      if (k < i) yv[k] = fma(-row[k], sl, yv[k]);
  }
}

// The same for rows i and i + 1 TOGETHER (i + 1 < NC).  Within a row every element depends on the previous one, so one row
// at a time is a single dependent chain (critical path 16 i cycles against 2 (i^2 / 2) cycles of work on sm_100a: latency
// bound at two warps per scheduler).  Two rows give the in-order warp two independent chains, every finished L[j][k] read
// from shared memory serves two products, and L[i+1][i] is formed from row i while it is still in registers.
template <int NC>
__device__ __forceinline__ void chol_pivot(double& acc, const double hii, bool& pd, const bool MOD) {
  if (MOD) {
    const double fl = 1.0e-10 * fabs(hii);
    if (!(acc > fl)) { acc = dmax(-acc, fl); pd = false; }
  } else {
    pd = pd && (acc > 0.0);
  }
}
// Rows i .. i + R - 1 together (all < NC); rw[r] is row i + r.  R = 2 is what pays (3, 4, 5, 10 measured: no further gain).
template <int NC, int R>
__device__ __forceinline__ void chol_rowsR(const int i, double (&rw)[R][NC], const LRows<NC>& L, double (&invd)[NC],
                                           double (&yv)[NC], double (&s)[NC], const double (&rhs)[R], bool& pd, const bool MOD = false) {
  double hd[R];
#pragma unroll
  for (int r = 0; r < R; ++r) hd[r] = rw[r][i + r];
  // columns j < i: every finished L[j][k] serves R products
#pragma unroll
  for (int j = 0; j < NC; ++j) {
    if (j < i) {
      double acc[R];
#pragma unroll
      for (int r = 0; r < R; ++r) acc[r] = rw[r][j];
#pragma unroll
      for (int k = 0; k < NC; ++k) {
        if (k < j) {
          const double l = L.at(j, k);
#pragma unroll
          for (int r = 0; r < R; ++r) acc[r] = fma(-rw[r][k], l, acc[r]);
        }
      }
#pragma unroll
      for (int r = 0; r < R; ++r) rw[r][j] = acc[r] * invd[j];
    }
  }
  // the R x R block on the diagonal, row by row, from the registers of the rows above
#pragma unroll
  for (int r = 0; r < R; ++r) {
    const int ir = i + r;
#pragma unroll
    for (int c = 0; c < R; ++c) {
      if (c < r) {          // element (i + r, i + c)
        const int jc = i + c;
        double acc = rw[r][jc];
#pragma unroll
        for (int k = 0; k < NC; ++k)
          if (k < jc) acc = fma(-rw[r][k], rw[c][k], acc);
        rw[r][jc] = acc * invd[jc];
      }
    }
    double d = rw[r][ir], a = rhs[r];
#pragma unroll
    for (int k = 0; k < NC; ++k)
      if (k < ir) { d = fma(-rw[r][k], rw[r][k], d); a = fma(-rw[r][k], yv[k], a); }
    chol_pivot<NC>(d, hd[r], pd, MOD);
    const double inv = rsqrt_fast(d);
    invd[ir] = inv;
    yv[ir] = a * inv;
    if (ir < NC - 1) {
      if (ir > 0) {
#pragma unroll
        for (int j = 0; j < NC; ++j)
          if (j < ir) L.at(ir, j) = rw[r][j];
      }
    } else {
      // the last row stays in registers: first step of the back substitution (see chol_row)
      const double sl = yv[ir] * inv;
      s[ir] = sl;
#pragma unroll
      for (int k = 0; k < NC; ++k)
        if (k < ir) yv[k] = fma(-rw[r][k], sl, yv[k]);
    }
  }
}

// back substitution L^T s = yv for rows NC-2 .. 0 (row NC-1 was done by chol_row)
template <int NC>
__device__ __forceinline__ void chol_back(const LRows<NC>& L, const double (&invd)[NC], const double (&yv)[NC], double (&s)[NC]) {
#pragma unroll
  for (int i = NC - 2; i >= 0; --i) {
    double acc = yv[i];
#pragma unroll
    for (int k = 0; k < NC - 1; ++k)
      if (k > i) acc = fma(-L.at(k, i), s[k], acc);
    s[i] = acc * invd[i];
  }
}

#ifndef PTF_STABN_MINB
#define PTF_STABN_MINB 2
#endif
#ifndef PTF_SPLITN_MINB
#define PTF_SPLITN_MINB 2
#endif

template <int NC>
constexpr int newton_lrows() { return (NC - 1) * (NC - 2) / 2; }            // rows 1 .. NC-2 of the strict lower triangle
template <int NC>
constexpr int stabn_smem_doubles() { return newton_lrows<NC>() + 4 * NC; }   // per thread: L, beta, pending step, residual r, d
// B200: 228 KB of shared memory per SM, 1 KB reserved per CTA, at most 227 KB per CTA; the 255-register kernels fit 2 CTAs
constexpr int newton_ctas_by_smem(int doubles_per_thread) {
  const int bytes = doubles_per_thread * NEWTON_THREADS * 8;
  const int n = bytes > 232448 ? 0 : 233472 / (bytes + 1024);
  return n > 2 ? 2 : n;
}
// the split kernel keeps the feed z in shared memory where that does not cost a resident CTA (else it is re-read through L1)
template <int NC>
constexpr bool split_z_in_smem() { return newton_ctas_by_smem(newton_lrows<NC>() + 7 * NC) == newton_ctas_by_smem(newton_lrows<NC>() + 6 * NC); }
template <int NC>                                                              // per thread: L, n^V, pending step, g, D, S(x), S(y) [, z]
constexpr int splitn_smem_doubles() { return newton_lrows<NC>() + (split_z_in_smem<NC>() ? 7 : 6) * NC; }

// ---- K3: stability trust-region Newton (B.1-B.3), persistent warps with lane refill --------------
template <int NC, bool KIJ0>
__global__ void __launch_bounds__(NEWTON_THREADS, PTF_STABN_MINB)
k3_stab_newton(const __grid_constant__ Sys<NC> S, const __grid_constant__ Opt o, const __grid_constant__ Io io,
               const __grid_constant__ Work w) {
  constexpr int NL = newton_lrows<NC>();
  constexpr unsigned FULL = 0xffffffffu;
  extern __shared__ double ptf_smem[];
  double* const sm = ptf_smem + threadIdx.x;
  const LRows<NC> L{sm};
  double* const sb = sm + NL * NEWTON_THREADS;   // accepted point beta = 2 sqrt(W) (B.1a)
  double* const sp = sb + NC * NEWTON_THREADS;   // pending / best-so-far step
  double* const sr = sp + NC * NEWTON_THREADS;   // residual r_i = ln W_i + lnphi_i(w) - d_i at the evaluated point
  double* const sdd = sr + NC * NEWTON_THREADS;  // d_i = ln z_i + lnphi_i(z) of the lane's mixture
  const int64_t N = io.N;
  const int n_front = w.qcount[Q_STAB_NEWTON];           // trials expected to be long (k2_stab_ss): taken first
  const int total = n_front + w.qcount[Q_STAB_NEWTON_E];  // the others sit at the end of the same array
  int* ticket = &w.qcount[Q_TICKET_STAB];
  // ---- lane state (scalars only) ----
  bool busy = false, exhausted = false, first = true, reeval = false, searching = false, exact = false;
  int n = 0, sidx = 0, iters = 0, tr_it = 0;
  unsigned act = 0u;
  PT3<NC> q;
  q.spt = 0.0; q.sT = 0.0; q.pt = 0.0;
  double tm = 0.0, rmax_acc = 0.0, pred = 0.0, Delta = 1.0, Delta_cap = 8.0, snorm = 0.0, Zw = 0.0, kept_sn = 0.0;
  EtaSearch es;
  es.start(1.0e-3);
  int my_max = 0;   // Table-4 counter, published after the loop

#pragma unroll 1
  while (true) {
    // ---- refill idle lanes from the ticket ----
    if (__any_sync(FULL, !busy && !exhausted)) {
      const int64_t tk = take_ticket(!busy && !exhausted, ticket);
      if (tk >= 0) {
        if (tk < total) {
          const int item = w.q_stab_newton[tk < n_front ? tk : 2 * N - 1 - (tk - n_front)];
          n = item >> 1;
          sidx = item & 1;
          const double P = io.P[n], T = io.T[n];
          { const double iT = rcp_fast(T); q.sT = sqrt_fast(T); q.spt = sqrt_fast(P) * iT; q.pt = P * iT; }
          act = (unsigned)w.actmask[n];
#pragma unroll
          for (int i = 0; i < NC; ++i) {
            sb[i * NEWTON_THREADS] = w.lnW[((int64_t)sidx * NC + i) * N + n];   // k2_stab_ss left beta = 2 sqrt(W) here
            sp[i * NEWTON_THREADS] = 0.0;
            sdd[i * NEWTON_THREADS] = __ldg(&w.d[(int64_t)i * N + n]);
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
#if PTF_NEWTON_CTA_SYNC
    // CTA-wide trip alignment: the four warps of a CTA walk the (larger than the instruction cache) trip body together,
    // so one instruction fetch serves all of them
    if (!__syncthreads_or(busy)) break;
#else
    if (!__any_sync(FULL, busy)) break;
#endif

    double Sv[NC];
    double sumW = 0.0;
    Eos e;
    e.Z = Zw;
    bool finish = false, fin_conv = false, fin_exact = false, fin_cap = false;
    if (busy) {
      // ---- evaluate tm and its gradient: at the trial point beta + s, or at beta while an eta search is pending ----
      double W[NC], lp[NC], r[NC];
      double sumW1 = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i) {
        const double b = sb[i * NEWTON_THREADS], s = sp[i * NEWTON_THREADS];
        const double h = 0.5 * (searching ? b : b + s);
        W[i] = h * h;                                              // B.1d
        r[i] = 2.0 * log_fast_m(h, (act >> i) & 1u);                // ln W_i (0 for a z_i = 0 component), branch-free
        if (i & 1) sumW1 += W[i]; else sumW += W[i];                // two accumulation chains
      }
      sumW += sumW1;
      {
        const double inv = rcp_fast(sumW);
        double wn[NC];
#pragma unroll
        for (int i = 0; i < NC; ++i) wn[i] = W[i] * inv;
        lnphi_pt<NC, KIJ0>(S, q, wn, lp, Sv, e);
      }
      Zw = e.Z;
      double rmax = 0.0, rmax1 = 0.0, tm_new = 1.0, tm_new1 = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i) {
        r[i] = ((act >> i) & 1u) ? r[i] + lp[i] - sdd[i * NEWTON_THREADS] : 0.0;
        if (i & 1) { rmax1 = dmax(rmax1, fabs(r[i])); tm_new1 = fma(W[i], r[i] - 1.0, tm_new1); }
        else { rmax = dmax(rmax, fabs(r[i])); tm_new = fma(W[i], r[i] - 1.0, tm_new); }
        sr[i * NEWTON_THREADS] = r[i];
      }
      rmax = dmax(rmax, rmax1);
      tm_new += tm_new1;
      if (!searching) {
        // ---- accept / reject the pending step (B.3) ----
        bool accepted = true;
        if (first) {
          double bn = 0.0;
#pragma unroll
          for (int i = 0; i < NC; ++i) bn = fma(W[i], 4.0, bn);   // |beta|^2 = 4 sum W
          Delta = dmax(1.0, 0.5 * sqrt_fast(bn));
          Delta_cap = 8.0 * Delta;
        } else if (!reeval) {
          const double act_red = tm_new - tm;
          accepted = (act_red < 0.0) || (rmax < rmax_acc);
          if (accepted) {
            if (fabs(pred) > 1.0e-13) {
              const double ratio = fabs(act_red * rcp_fast(pred));
              if (ratio <= 0.25) Delta *= 0.5;
              else if (ratio >= 0.75) Delta = dmin(2.0 * Delta, Delta_cap);
            }
          } else {
            Delta = 0.5 * dmin(Delta, snorm);
            reeval = true;   // next trip re-evaluates at the accepted point (s = 0) and continues from there
          }
        }
        if (!accepted) {
#pragma unroll
          for (int i = 0; i < NC; ++i) sp[i * NEWTON_THREADS] = 0.0;
        } else {
#pragma unroll
          for (int i = 0; i < NC; ++i) { sb[i * NEWTON_THREADS] += sp[i * NEWTON_THREADS]; sp[i * NEWTON_THREADS] = 0.0; }
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
      // ---- ONE attempt of the restricted-step sub-problem at es.eta (B.1b) ----
      // B.2b: H_ij = sqrt(w_i w_j) M_ij + delta_ij (1 + r_i / 2) = h_i h_j Mt_ij with h_i = sqrt(w_i) and
      // Mt = M + diag((1 + r_i / 2 + eta) / w_i): the congruent matrix Mt is factored instead (same inertia), so the rows
      // need only S_j, sqrt(A_j) and constants; H s = -g becomes Mt u = -g / h = -r sqrt(sum W), s_i = u_i / h_i.
      // A component with z_i = 0 gets the diagonal 1e300, which decouples it (its step is masked to zero).
      const MC3 mc = mc3(e);
      const double isq = rsqrt_fast(sumW);
      const double sqW = sumW * isq;
      const double c01p = mc.c01 * q.pt, c10p = mc.c10 * q.pt, c11p = mc.c11 * q.pt * q.pt, c12p = mc.c12 * q.pt, c21p = mc.c21 * q.pt;
      double sa[NC];
#pragma unroll
      for (int i = 0; i < NC; ++i) sa[i] = sa_of<NC>(S, q, i);
      double invd[NC], yv[NC], st[NC];
      bool good = true;
      // row i of M: M_ij = G0 + G1 wb_j + G2 S_j - q2 sa_i omk_ij sa_j with G = C F_i, F_i = (1, wb_i, S_i)
      auto gen_row = [&](const int i, double (&row)[NC], double& rhs) {
        const double G0 = fma(Sv[i], mc.c20, fma(S.wb[i], c10p, mc.c00));
        const double G1 = fma(Sv[i], c21p, fma(S.wb[i], c11p, c01p));
        const double G2 = fma(Sv[i], mc.c22, fma(S.wb[i], c12p, mc.c02));
        const double qs = mc.q2 * sa[i];
#pragma unroll
        for (int j = 0; j < NC; ++j) {
          if (j <= i) row[j] = fma(-(KIJ0 ? qs : qs * S.omk[i * NC + j]), sa[j], fma(G2, Sv[j], fma(G1, S.wb[j], G0)));
        }
        const double ri = sr[i * NEWTON_THREADS];
        const double ih = 2.0 * sqW * rcp_fast(sb[i * NEWTON_THREADS]);          // 1 / h_i (beta_i = 2 h_i sqrt(sum W))
        const double iw = ((act >> i) & 1u) ? ih * ih : 1.0e300;
        row[i] = fma(1.0 + 0.5 * ri + es.eta, iw, row[i]);
        rhs = -ri * sqW;
      };
      {
        constexpr int R = PTF_CHOL_R;
        constexpr int NB = NC / R * R;   // rows handled in blocks of R, the remainder one by one
#pragma unroll
        for (int i = 0; i < NB; i += R) {
          double rw[R][NC], rh[R];
#pragma unroll
          for (int r = 0; r < R; ++r) gen_row(i + r, rw[r], rh[r]);
          chol_rowsR<NC, R>(i, rw, L, invd, yv, st, rh, good);
        }
#pragma unroll
        for (int i = NB; i < NC; ++i) {
          double row[NC], qa_;
          gen_row(i, row, qa_);
          chol_row<NC>(i, row, L, invd, yv, st, qa_, good);
        }
      }
      chol_back<NC>(L, invd, yv, st);
      double sn = 0.0, sg = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i) {
        const double b = sb[i * NEWTON_THREADS];
        sg = fma(st[i], sr[i * NEWTON_THREADS], sg);                             // s.g = sqrt(sum W) u.r
        st[i] = ((act >> i) & 1u) ? st[i] * (2.0 * sqW * rcp_fast(b)) : 0.0;     // s_i = u_i / h_i
        sn = fma(st[i], st[i], sn);
        if (((act >> i) & 1u) && !(b + st[i] > 0.0)) good = false;
      }
      sn = sqrt_fast(sn);
      good = good && (sn <= Delta);
      const double eta_used = es.eta;
      if (es.feed(good, sn, Delta, kept_sn)) {
#pragma unroll
        for (int i = 0; i < NC; ++i) sp[i * NEWTON_THREADS] = st[i];
        snorm = sn;
        pred = 0.5 * sg * sqW - 0.5 * eta_used * sn * sn;   // predicted reduction s.g + s.H.s/2 with H s = -g - eta s
        exact = (eta_used == 0.0);
      }
      if (es.phase == 4) { finish = true; fin_cap = true; searching = false; }
      else if (es.phase == 3) {
        searching = false;
        double smax = 0.0;
#pragma unroll
        for (int i = 0; i < NC; ++i) smax = dmax(smax, fabs(sp[i * NEWTON_THREADS]));
        if (exact && smax < o.tol_newton_step_stab) {
          // quadratic-convergence finish: apply the full Newton step and stop
          finish = true;
          fin_conv = true;
          fin_exact = true;
          sumW = 0.0;
#pragma unroll
          for (int i = 0; i < NC; ++i) {
            const double b = sb[i * NEWTON_THREADS] + sp[i * NEWTON_THREADS];
            sb[i * NEWTON_THREADS] = b;
            sumW = fma(0.5 * b, 0.5 * b, sumW);
          }
        }
      }
    }
    __syncwarp();
    if (finish) {
      // beta is stored; k_stab_decide turns it into ln W = 2 ln(beta/2) with all lanes active (TF_BETA)
#pragma unroll
      for (int i = 0; i < NC; ++i) w.lnW[((int64_t)sidx * NC + i) * N + n] = sb[i * NEWTON_THREADS];
      w.tm[(int64_t)sidx * N + n] = tm;
      w.sumW[(int64_t)sidx * N + n] = sumW;
      w.tflags[(int64_t)sidx * N + n] = (fin_conv ? TF_CONVERGED : 0) | (fin_exact ? TF_EXACT : 0) |
                                        (fin_cap ? TF_CAPPED : 0) | TF_BETA | (iters << TF_ITER_SHIFT);
      if (fin_cap) atomicAdd((unsigned long long*)&w.ctr->n_stab_capped[sidx], 1ull);   // rare
      {
        // running maxima of the trust-region iteration count per start, two 16-bit fields of one register
        const int sh = sidx << 4, it = min(tr_it, 65535);
        if (it > ((my_max >> sh) & 0xffff)) my_max = (my_max & ~(0xffff << sh)) | (it << sh);
      }
      busy = false;
    }
  }
  flush_max(my_max & 0xffff, &w.ctr->max_stab_tr[0]);
  flush_max((my_max >> 16) & 0xffff, &w.ctr->max_stab_tr[1]);
}

// ---- K6: phase-split trust-region Newton on G (B.4-B.5), persistent warps with lane refill --------
// Variables n^V (B.4).  In the code's normalisation H_ij = wx Mx_ij + wy My_ij - 1/tt + delta_ij D_i (1/tt + eta),
// tt = theta (1 - theta), wx = 1/(1 - theta), wy = 1/theta, D_i = z_i / (x_i y_i) (B.5b with the unit-total-mole M,
// reading C18).  Basis F_i = (1, B_i, Sx_i, Sy_i); the 4 x 4 coefficient matrix is wx Cx (+) wy Cy - E_00 / tt.
//
// The evaluation of a trip (two lnphi, one code copy looped over the phases) leaves S(x), S(y), the gradient and D in
// shared memory, so a lane that has to retry with a larger eta does not evaluate again.
template <int NC, bool KIJ0>
__global__ void __launch_bounds__(NEWTON_THREADS, PTF_SPLITN_MINB)
k3_split_newton(const __grid_constant__ Sys<NC> S, const __grid_constant__ Opt o, const __grid_constant__ Io io,
                const __grid_constant__ Work w, const int part) {
  constexpr int NL = newton_lrows<NC>();
  constexpr int T = NEWTON_THREADS;
  constexpr unsigned FULL = 0xffffffffu;
  extern __shared__ double ptf_smem[];
  double* const sm = ptf_smem + threadIdx.x;
  const LRows<NC> L{sm};
  double* const sn = sm + NL * T;    // accepted n^V (of the minority phase, see k2_split_ss)
  double* const sp = sn + NC * T;    // pending step
  double* const sg = sp + NC * T;    // gradient (B.5a) at the evaluated point
  double* const sD = sg + NC * T;    // D_i = z_i / (x_i y_i)
  double* const sS = sD + NC * T;    // S(x) [NC], S(y) [NC]
  constexpr bool ZS = split_z_in_smem<NC>();
  double* const sz = sS + 2 * NC * T;   // normalised feed z of the lane's mixture (read many times per trip), if it fits (ZS)
  const int64_t N = io.N;
  const int n_front = w.qcount[qid_split_newton(part)];            // slow-SS splits (k2_split_ss): taken first
  const int total = n_front + w.qcount[qid_split_newton_e(part)];   // the others sit at the end of the array
  const int* const q_in = q_split_newton_of(w, part);
  int* ticket = &w.qcount[qid_ticket_split(part)];
  bool busy = false, exhausted = false, first = true, reeval = false, searching = false, exact = false, polish = false;
  bool eta_mode = false;   // this lane's item runs the eta search of B.4a instead of the truncated modified-Cholesky step
  int tr_cap = 0;          // trust-region iteration cap of the lane's item (smaller for a skip-stability hint, reading C21)
  int n = 0, tr_it = 0, status = 0;
  unsigned act = 0u;
  PT3<NC> q;
  q.spt = 0.0; q.sT = 0.0; q.pt = 0.0;
  double G = 0.0, gmax_acc = 0.0, pred = 0.0, Delta = 0.25, snorm = 0.0, kept_sn = 0.0, theta = 0.5;
  EtaSearch es;
  es.start(1.0);
  Eos ex, ey;   // cubic scalars of the two phases at the evaluated point (Z doubles as the warm start)
  ex.A = ex.B = ex.Z = ex.q = ex.L = ex.lnZmB = 0.0;
  ey = ex;
  int my_max = 0;   // Table-4 counter, published after the loop

#pragma unroll 1
  while (true) {
    if (__any_sync(FULL, !busy && !exhausted)) {
      const int64_t tk = take_ticket(!busy && !exhausted, ticket);
      if (tk >= 0) {
        if (tk < total) {
          n = q_in[tk < n_front ? tk : N - 1 - (tk - n_front)];
          const double P = io.P[n], Tk = io.T[n];
          { const double iT = rcp_fast(Tk); q.sT = sqrt_fast(Tk); q.spt = sqrt_fast(P) * iT; q.pt = P * iT; }
          act = (unsigned)w.actmask[n];
          {
            const bool hinted = (w.pass == 0) && (w.status[n] & ST_INTERNAL_SKIPPED);
            eta_mode = o.hint_eta_search && hinted;
            tr_cap = hinted ? min(o.split_tr_iters, o.hint_tr_cap) : o.split_tr_iters;
          }
#pragma unroll
          for (int i = 0; i < NC; ++i) {
            sn[i * T] = w.lnK[(int64_t)i * N + n];   // k2_split_ss left n^V here
            sp[i * T] = 0.0;
            if (ZS) sz[i * T] = __ldg(&w.zn[(int64_t)i * N + n]);
          }
          tr_it = 0;
          status = 0;
          first = true;
          reeval = false;
          searching = false;
          polish = false;
          Delta = 0.25;
          ex.Z = w.Zxy[n];
          ey.Z = w.Zxy[N + n];
          busy = true;
        } else {
          exhausted = true;
        }
      }
    }
#if PTF_NEWTON_CTA_SYNC
    // CTA-wide trip alignment: the four warps of a CTA walk the (larger than the instruction cache) trip body together,
    // so one instruction fetch serves all of them
    if (!__syncthreads_or(busy)) break;
#else
    if (!__any_sync(FULL, busy)) break;
#endif

    bool finish = false, fin_conv = false;
    if (busy && !searching) {
      // ---- evaluate G (eq. 8) and its gradient (B.5a) at n^V + s ----
      theta = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i) theta += sn[i * T] + sp[i * T];
      const double it = rcp_fast(theta), il = rcp_fast(1.0 - theta);
      double G_new = 0.0, gmax = 0.0;
#pragma unroll
      for (int ph = 0; ph < 2; ++ph) {
        double c[NC], lp[NC], Sv[NC];
#pragma unroll
        for (int i = 0; i < NC; ++i) {
          const double v = sn[i * T] + sp[i * T];
          c[i] = ph ? v * it : ((ZS ? sz[i * T] : __ldg(&w.zn[(int64_t)i * N + n])) - v) * il;
        }
        Eos e;
        e.Z = ph ? ey.Z : ex.Z;
        lnphi_pt<NC, KIJ0>(S, q, c, lp, Sv, e);
        if (ph) ey = e; else ex = e;
        const double wph = ph ? theta : 1.0 - theta;
#pragma unroll
        for (int i = 0; i < NC; ++i) {
          const bool a = (act >> i) & 1u;
          const double f = a ? log_fast_m(c[i], a) + lp[i] : 0.0;
          G_new = fma(c[i] * wph, f, G_new);
          sS[(ph * NC + i) * T] = a ? Sv[i] : 0.0;
          if (ph == 0) {
            sg[i * T] = -f;
            sD[i * T] = c[i];
          } else {
            const double g = sg[i * T] + f;
            sg[i * T] = g;
            gmax = dmax(gmax, fabs(g));
            sD[i * T] = a ? (ZS ? sz[i * T] : __ldg(&w.zn[(int64_t)i * N + n])) * rcp_fast(sD[i * T] * c[i]) : 1.0;
          }
        }
      }
      // ---- accept / reject ----
      bool accepted = true;
      if (!first && !reeval) {
        const double act_red = G_new - G;
        // accept if G fell; a smaller gradient is accepted instead only where the change of G is below its rounding
        // resolution (next to the solution).  With the plain "G fell or the gradient fell" a modified-Cholesky step (C25)
        // that raises G is accepted whenever it happens to lower the gradient norm, and single mixtures next to the phase
        // boundary wander across the whole box 0 < n < z until the iteration cap (config 5: 1.5 per 1000).
        accepted = (act_red < 0.0) || (gmax < gmax_acc && act_red <= 1.0e-12 * fabs(G));
        if (accepted) {
          if (fabs(pred) > 1.0e-13) {
            const double ratio = fabs(act_red * rcp_fast(pred));
            if (ratio <= 0.25) Delta *= 0.5;
            else if (ratio >= 0.75) Delta = dmin(2.0 * Delta, 1.0);
          }
        } else {
          Delta = 0.5 * dmin(Delta, snorm);
          reeval = true;
        }
      }
      if (!accepted) {
#pragma unroll
        for (int i = 0; i < NC; ++i) sp[i * T] = 0.0;
      } else {
#pragma unroll
        for (int i = 0; i < NC; ++i) { sn[i * T] += sp[i * T]; sp[i * T] = 0.0; }
        G = G_new;
        gmax_acc = gmax;
        first = false;
        reeval = false;
        // Reading C8: a gradient below the target does not end the iteration by itself -- near a critical point and next
        // to the phase boundary the Hessian is nearly singular and the gradient does not bound the error of n^V -- it
        // triggers one last full Newton step (polish), applied without another evaluation if it is admissible.
        polish = gmax < o.tol_newton_g;
        if (!polish && tr_it >= tr_cap) { finish = true; status |= ST_SPLIT_CAP; }
        else {
          if (!polish) tr_it++;
          es.start(1.0e-3 * rcp_fast(theta * (1.0 - theta)));
          kept_sn = 0.0;
          searching = true;
        }
      }
    }
    __syncwarp();
    if (busy && searching) {
      // ---- ONE attempt of the restricted-step sub-problem at eta (B.4a) ----
      const MC3 mx = mc3(ex), my = mc3(ey);
      const double tt = theta * (1.0 - theta), itt = rcp_fast(tt);
      const double wx = theta * itt, wy = (1.0 - theta) * itt;   // weights of M(x), M(y) in B.5b
      const double pt = q.pt;
      // 4 x 4 coefficients in the basis (1, wb_i, Sx_i, Sy_i) (pt folded into the wb rows / columns)
      const double c00 = fma(wx, mx.c00, wy * my.c00) - itt;
      const double c01 = fma(wx, mx.c01, wy * my.c01) * pt, c10 = fma(wx, mx.c10, wy * my.c10) * pt;
      const double c11 = fma(wx, mx.c11, wy * my.c11) * pt * pt;
      const double c02 = wx * mx.c02, c20 = wx * mx.c20, c12 = wx * mx.c12 * pt, c21 = wx * mx.c21 * pt, c22 = wx * mx.c22;
      const double c03 = wy * my.c02, c30 = wy * my.c20, c13 = wy * my.c12 * pt, c31 = wy * my.c21 * pt, c33 = wy * my.c22;
      const double qa = fma(wx, mx.q2, wy * my.q2);
      const double deta = itt + es.eta;
      double one[NC], sa[NC], Sx[NC], Sy[NC];
#pragma unroll
      for (int i = 0; i < NC; ++i) {
        const bool a = (act >> i) & 1u;
        one[i] = a ? 1.0 : 0.0;
        sa[i] = a ? sa_of<NC>(S, q, i) : 0.0;
        Sx[i] = sS[i * T];
        Sy[i] = sS[(NC + i) * T];
      }
      double invd[NC], yv[NC], st[NC];
      bool pd = true;
      auto gen_row = [&](const int i, double (&row)[NC]) {
        const double ob = one[i] * S.wb[i];
        const double G0 = fma(Sy[i], c30, fma(Sx[i], c20, fma(ob, c10, one[i] * c00)));
        const double G1 = fma(Sy[i], c31, fma(Sx[i], c21, fma(ob, c11, one[i] * c01)));
        const double G2 = fma(Sx[i], c22, fma(ob, c12, one[i] * c02));
        const double G3 = fma(Sy[i], c33, fma(ob, c13, one[i] * c03));
        const double qs = qa * sa[i];
#pragma unroll
        for (int j = 0; j < NC; ++j) {
          if (j <= i) {
            double a = fma(G3, Sy[j], fma(G2, Sx[j], fma(G1, one[j] * S.wb[j], G0 * one[j])));
            a = fma(-(KIJ0 ? qs : qs * S.omk[i * NC + j]), sa[j], a);
            row[j] = a;
          }
        }
        row[i] = fma(sD[i * T], deta, row[i]);                 // + D_i / tt + eta D_i (B.4a)
      };
      {
        constexpr int R = PTF_CHOL_R;
        constexpr int NB = NC / R * R;   // rows handled in blocks of R, the remainder one by one
#pragma unroll
        for (int i = 0; i < NB; i += R) {
          double rw[R][NC], rh[R];
#pragma unroll
          for (int r = 0; r < R; ++r) { gen_row(i + r, rw[r]); rh[r] = -sg[(i + r) * T]; }
          chol_rowsR<NC, R>(i, rw, L, invd, yv, st, rh, pd, !eta_mode);
        }
#pragma unroll
        for (int i = NB; i < NC; ++i) {
          double row[NC];
          gen_row(i, row);
          chol_row<NC>(i, row, L, invd, yv, st, -sg[i * T], pd, !eta_mode);
        }
      }
      chol_back<NC>(L, invd, yv, st);
      // Restricted step without a search (C25): the direction of the (modified) factorisation is cut back to the trust region
      // and to 90 % of the way to the nearest face of the box 0 < n_i < z_i.  One factorisation, i.e. one trip, per
      // iteration; the eta search of the paper's B.4a (grow x8, then bisect: up to ten factorisations) is kept for the
      // stability kernel, whose path decides labels, and for splits entered through a skip-stability hint (eta_mode):
      // from a caller's K next to the phase boundary the truncated step slides into a face of the box and fails where the
      // search converges, and whether a hint fails is reported (C21).  Acceptance and the radius update (B.3) are shared.
      if (!eta_mode) {
        double s2 = 0.0, sgd = 0.0, over = 0.0;
#pragma unroll
        for (int i = 0; i < NC; ++i) {
          const bool a = (act >> i) & 1u;
          st[i] = a ? st[i] : 0.0;
          s2 = fma(st[i], st[i], s2);
          sgd = fma(st[i], sg[i * T], sgd);
          const double ni = sn[i * T];
          const double room = a ? dmax(st[i] < 0.0 ? ni : (ZS ? sz[i * T] : __ldg(&w.zn[(int64_t)i * N + n])) - ni, 1.0e-300) : 1.0;
          over = dmax(over, fabs(st[i]) * rcp_fast(room));
        }
        const double sl = sqrt_fast(s2);
        double t = 1.0;
        if (over > 0.9) t = 0.9 * rcp_fast(over);
        if (sl * t > Delta) t = Delta * rcp_fast(sl);
        const bool ok = (t == t) && (sl == sl) && sgd < 0.0;   // NaN-free descent direction
#pragma unroll
        for (int i = 0; i < NC; ++i) sp[i * T] = ok ? t * st[i] : 0.0;
        snorm = sl * t;
        pred = (t - 0.5 * t * t) * sgd;
        exact = pd && t == 1.0;
        es.phase = ok ? 3 : 4;
      } else {
      bool good = pd;
      double s2 = 0.0, sds = 0.0, sgd = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i) {
        s2 = fma(st[i], st[i], s2);
        sds = fma(st[i] * st[i], sD[i * T], sds);
        sgd = fma(st[i], sg[i * T], sgd);
        if ((act >> i) & 1u) {
          const double nv = sn[i * T] + st[i];
          if (!(nv > 0.0) || !(nv < (ZS ? sz[i * T] : __ldg(&w.zn[(int64_t)i * N + n])))) good = false;
        }
      }
      const double sl = sqrt_fast(s2);
      good = good && (sl <= Delta);
      const double eta_used = es.eta;
      if (es.feed(good, sl, Delta, kept_sn)) {
#pragma unroll
        for (int i = 0; i < NC; ++i) sp[i * T] = st[i];
        snorm = sl;
        pred = 0.5 * sgd - 0.5 * eta_used * sds;
        exact = (eta_used == 0.0);
      }
      }
      if (polish) {
        // last step: applied if it is the full Newton step of a positive definite Hessian inside the box and the trust
        // region; otherwise the evaluated point stands
        finish = true;
        fin_conv = true;
        searching = false;
        if (es.phase == 3 && exact) {
#pragma unroll
          for (int i = 0; i < NC; ++i) sn[i * T] += sp[i * T];
        }
      } else if (es.phase == 4) { finish = true; status |= ST_SPLIT_CAP; searching = false; }
      else if (es.phase == 3) {
        searching = false;
        double smax = 0.0;   // largest step relative to the smaller of the two mole numbers n_i, z_i - n_i
#pragma unroll
        for (int i = 0; i < NC; ++i) {
          if ((act >> i) & 1u) {
            const double ni = sn[i * T];
            smax = dmax(smax, fabs(sp[i * T]) * rcp_fast(dmin(ni, (ZS ? sz[i * T] : __ldg(&w.zn[(int64_t)i * N + n])) - ni)));
          }
        }
        if (exact && smax < o.tol_newton_step) {
          finish = true;
          fin_conv = true;
#pragma unroll
          for (int i = 0; i < NC; ++i) sn[i * T] += sp[i * T];
        }
      }
    }
    __syncwarp();
    if (finish) {
      // compositions of the accepted point
      double z[NC], x[NC], y[NC], lnK[NC];
      theta = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i) { z[i] = (ZS ? sz[i * T] : __ldg(&w.zn[(int64_t)i * N + n])); y[i] = sn[i * T]; theta += y[i]; }
      {
        const double it = rcp_fast(theta), il = rcp_fast(1.0 - theta);
#pragma unroll
        for (int i = 0; i < NC; ++i) { const double v = y[i]; y[i] = v * it; x[i] = (z[i] - v) * il; }
      }
      // trivial collapse x = y (max |ln K| < 1e-9): |y/x - 1| is the same test to first order and needs no logarithm
      double mkn = 0.0;
#pragma unroll
      for (int i = 0; i < NC; ++i)
        if ((act >> i) & 1u) mkn = dmax(mkn, fabs(y[i] - x[i]) * rcp_fast(x[i]));
      const bool trivial = mkn < o.split_trivial_tol;
      if (io.lnK) {
#pragma unroll
        for (int i = 0; i < NC; ++i) lnK[i] = ((act >> i) & 1u) ? log_fast(y[i]) - log_fast(x[i]) : 0.0;
      } else {
#pragma unroll
        for (int i = 0; i < NC; ++i) lnK[i] = 0.0;
      }
      store_split<NC>(io, w, n, z, fin_conv, trivial, theta, tr_it, status, x, y, lnK, ex.Z, ey.Z);
      if (status & ST_SPLIT_CAP) atomicAdd((unsigned long long*)&w.ctr->n_split_capped, 1ull);   // rare
      my_max = max(my_max, tr_it);
      busy = false;
    }
  }
  flush_max(my_max, &w.ctr->max_split_tr);
}

}  // namespace ptf
