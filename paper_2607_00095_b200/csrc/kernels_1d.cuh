// 1D kinds (Burgers-LF, Burgers-LF + mass rows, Fisher-KPP implicit): one persistent warp per sample
// runs the whole Gauss-Newton loop with no host round trip.
//
// Per Gauss-Newton iteration the Schur system (J J^T) lam+ = r = h - J (u - u_hat) (Eq. 24,
// W = I) is solved in product form: for these row sets J_loc is square and block lower-bidiagonal in time
// (diagonal blocks I or the SPD tridiagonal T_k, sub-diagonal blocks -A_{k-1} or -I), so J J^T = L L^T with
// L = J_loc and zero fill (oracle pin P6).  "Factor + solve" is therefore
//     forward sweep   L y = r        (k = 0 .. nt-1; fused with the residual/Jacobian evaluation a1-a3)
//     backward sweep  L^T lam = y    (k = nt-1 .. 0; fused with the step u+ = u_hat - J^T lam, J^T lam == y)
// Rows stream HBM -> shared memory through a per-warp ring of 1-D bulk (TMA) copies completing on
// mbarriers; results leave through shared memory with bulk stores.  Stencil neighbours (i +- 1) are read
// from the shared-memory rows (halo staging), reductions are fixed-order warp shuffles.
#pragma once
#include "device_utils.cuh"
#include "launch.h"
#include "snap_internal.h"
#include "tridiag.cuh"

namespace snap {

constexpr int KB = 1;  // Burgers family: lane owns cells lane + 32 j   (conflict-free shared-memory access)
constexpr int KF = 2;  // Fisher family:  lane owns cells lane*Q + j    (contiguous, for the warp tridiagonal solve)


// ------------------------------------------------------------------------------------------------
// per-warp row pipeline.  A row buffer is [pad, halo_left, data[0..nx), halo_right, pad] with the data
// start 16-byte aligned (bulk-copy destination); the halo cells hold the periodic (Burgers) or mirrored
// (Fisher, Neumann) neighbours so that every stencil access is base[i +- 1] with no index arithmetic.
// ------------------------------------------------------------------------------------------------
constexpr int kHalo = 2;  // doubles in front of the data start

template <bool TMA>
struct Pipe {
  double* stage;   // [nst][3][rp]
  double* srow;    // [5][rp]
  uint32_t bar0;   // shared address of mbarrier 0
  uint32_t phase;  // parity to wait for, one bit per stage
  int nst, rp, nx, lane;

  __device__ __forceinline__ double* row(int s, int r) const { return stage + (size_t)(s * 3 + r) * rp + kHalo; }
  __device__ __forceinline__ double* out(int r) const { return srow + (size_t)r * rp + kHalo; }

  // Load up to three global rows of nx doubles into stage s.  Called by the whole (converged) warp after
  // every lane has finished reading the previous contents of the stage.
  __device__ __forceinline__ void issue(int s, const double* g0, const double* g1, const double* g2) {
    __syncwarp();
    const uint32_t bar = bar0 + 8u * s;
    if (TMA) {
      if (lane == 0) {
        const uint32_t rb = (uint32_t)nx * 8u;
        mbar_expect_tx(bar, rb * (g2 ? 3u : 2u));
        bulk_g2s(smem_u32(row(s, 0)), g0, rb, bar);
        bulk_g2s(smem_u32(row(s, 1)), g1, rb, bar);
        if (g2) bulk_g2s(smem_u32(row(s, 2)), g2, rb, bar);
      }
    } else {
      double* d0 = row(s, 0);
      double* d1 = row(s, 1);
      double* d2 = row(s, 2);
      for (int i = lane; i < nx; i += 32) {
        d0[i] = g0[i];
        d1[i] = g1[i];
        if (g2) d2[i] = g2[i];
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar);
    }
  }
  __device__ __forceinline__ void wait(int s) {
    mbar_wait(bar0 + 8u * s, (phase >> s) & 1u);
    phase ^= (1u << s);
  }
  // After wait(): fill the halo of a freshly landed row (periodic or mirror) and make the shared-memory
  // output rows written >= 2 steps ago reusable; ends with a warp barrier.
  template <bool PERIODIC>
  __device__ __forceinline__ void ready(double* halo_row) {
    if (lane == 0) {
      if (halo_row) {
        halo_row[-1] = PERIODIC ? halo_row[nx - 1] : halo_row[0];
        halo_row[nx] = PERIODIC ? halo_row[0] : halo_row[nx - 1];
      }
      if (TMA) bulk_wait_read<1>();
    }
    __syncwarp();
  }
  // lanes have written an output row with generic stores; hand it to the bulk-store engine
  __device__ __forceinline__ void store_row(double* g, const double* s_row) {
    if (TMA && lane == 0) bulk_s2g(g, smem_u32(s_row), (uint32_t)nx * 8u);
  }
  __device__ __forceinline__ void commit() {
    if (TMA && lane == 0) bulk_commit();
  }
  // all outstanding bulk stores of this warp are complete and visible to later loads
  __device__ __forceinline__ void drain() {
    if (TMA) {
      if (lane == 0) {
        bulk_wait_all<0>();
        fence_proxy_async_all();
      }
    } else {
      __threadfence_block();
    }
    __syncwarp();
  }
};

struct SweepNorms {
  double hinf, h1, f;  // ||h||_inf, ||h||_1, 1/2 ||u - u_hat||^2
  int bad;             // non-finite residual seen
};

// ------------------------------------------------------------------------------------------------
// forward sweep: residual h (a1), Jacobian coefficients (a2), rhs (a3) and L y = r (a5), level by level.
// Reads u (point of linearisation) and u_hat rows, writes y into the multiplier buffer.
//
// Burgers family (lane owns cells lane + 32 j).  With q = y + (u - u_hat) the recurrence L y = r reads
//     q_0 = h_0 ,   q_k = h_k + A_{k-1} q_{k-1} ,   h_k = u[k] - Phi(u[k-1]) ,   y_k = q_k - (u[k] - u_hat[k])
// Phi(u[k-1])_i and the two off-diagonal coefficients of A_{k-1} are computed while level k-1 is in shared
// memory and carried in registers, so a stage is free for refill as soon as its level has been processed.
// ------------------------------------------------------------------------------------------------
template <int Q, bool FULL, bool TMA>
__device__ void fwd_sweep_b(const DevParams& P, Pipe<TMA>& pp, const double* __restrict__ u,
                            const double* __restrict__ uh, const double* __restrict__ u0, double* __restrict__ y,
                            double M0, SweepNorms& out) {
  const int nx = P.nx, nt = P.nt, lane = pp.lane, nst = pp.nst;
  const double a0 = P.bs_a0, e = P.bs_e, qs = P.bs_qs, hs = P.bs_hs;
  double hinf = 0.0, h1 = 0.0, f2 = 0.0, minf = 0.0, m1 = 0.0;
  double qo[Q], phi[Q], cpj[Q], cmj[Q];
#pragma unroll
  for (int j = 0; j < Q; ++j) {
    const int i = lane + 32 * j;
    phi[j] = (FULL || i < nx) ? u0[i] : 0.0;  // level 0: h_0 = u[0] - u0
    qo[j] = 0.0; cpj[j] = 0.0; cmj[j] = 0.0;
  }
  const int npro = nst < nt ? nst : nt;
  for (int k = 0; k < npro; ++k) pp.issue(k, u + (size_t)k * nx, uh + (size_t)k * nx, nullptr);
  // q_{-1} = 0: level 0 runs the general recurrence with zero coefficients, so the slot it reads must be finite
  {
    double* z = pp.out(3) - 1;
    for (int i = lane; i < nx + 2; i += 32) z[i] = 0.0;
  }
  int s = 0;
  for (int k = 0; k < nt; ++k) {
    pp.wait(s);
    double* su0 = pp.row(s, 0);
    pp.template ready<true>(su0);
    const double* su = su0 + lane;
    const double* sh = pp.row(s, 1) + lane;
    double* yo0 = pp.out(k & 1);
    double* qc0 = pp.out(2 + (k & 1));
    double* yo = yo0 + lane;
    double* qc = qc0 + lane;
    const double* qp = pp.out(2 + ((k + 1) & 1)) + lane;   // q_{k-1} (zero coefficients at k = 0)
    double* yg = y + (size_t)k * nx;
    double msum = 0.0;
#pragma unroll
    for (int j = 0; j < Q; ++j) {
      const int o = 32 * j;
      if (FULL || lane + o < nx) {
        const double uk = su[o], uhk = sh[o], up = su[o + 1], um = su[o - 1];
        const double h = uk - phi[j];
        const double q = fma(cpj[j], qp[o + 1], fma(cmj[j], qp[o - 1], fma(a0, qo[j], h)));
        const double w = uk - uhk;
        const double yv = q - w;
        qc[o] = q;
        if (FULL) {
          if (j == 0 && lane == 0) qc0[nx] = q;
          if (j == Q - 1 && lane == 31) qc0[-1] = q;
        } else {
          if (lane + o == 0) qc0[nx] = q;
          if (lane + o == nx - 1) qc0[-1] = q;
        }
        if (TMA) yo[o] = yv; else yg[lane + o] = yv;
        const double ah = fabs(h);
        hinf = fmax(hinf, ah);
        h1 += ah;
        f2 = fma(w, w, f2);
        msum += uk;
        phi[j] = fma(a0, uk, (up + um) * fma(-qs, up - um, e));
        cpj[j] = fma(-hs, up, e);
        cmj[j] = fma(hs, um, e);
        qo[j] = q;
      }
    }
    if (P.has_mass) {
      const double hm = fabs(P.dx * warp_sum(msum) - M0);
      minf = fmax(minf, hm);
      m1 += hm;
    }
    if (TMA) fence_proxy_async_smem();
    __syncwarp();
    pp.store_row(yg, yo0);
    pp.commit();
    if (k + nst < nt) pp.issue(s, u + (size_t)(k + nst) * nx, uh + (size_t)(k + nst) * nx, nullptr);
    if (++s == nst) s = 0;
  }
  pp.drain();
  hinf = warp_max(hinf);
  h1 = warp_sum(h1);
  f2 = warp_sum(f2);
  if (P.has_mass) {
    hinf = fmax(hinf, minf);
    h1 += m1;
  }
  out.hinf = hinf;
  out.h1 = h1;
  out.f = 0.5 * f2;
  // fmax drops NaN; the sums do not: a non-finite residual or iterate shows up in h1 / f2
  out.bad = !finite_d(hinf) | !finite_d(h1) | !finite_d(f2);
}

// Fisher family (lane owns cells lane*Q + j):  q_0 = h_0 ,  T_k q_k = h_k + q_{k-1} ,  y_k = q_k - (u[k]-u_hat[k]).
template <int Q, bool TMA>
__device__ void fwd_sweep_f(const DevParams& P, Pipe<TMA>& pp, const double* __restrict__ u,
                            const double* __restrict__ uh, const double* __restrict__ u0, double* __restrict__ y,
                            SweepNorms& out) {
  const int nx = P.nx, nt = P.nt, lane = pp.lane, nst = pp.nst;
  double hinf = 0.0, h1 = 0.0, f2 = 0.0;
  double u0r[Q], qo[Q], upr[Q];
#pragma unroll
  for (int j = 0; j < Q; ++j) {
    const int i = lane * Q + j;
    u0r[j] = (i < nx) ? u0[i] : 0.0;
    qo[j] = 0.0; upr[j] = 0.0;
  }
  const int npro = nst < nt ? nst : nt;
  for (int k = 0; k < npro; ++k) pp.issue(k, u + (size_t)k * nx, uh + (size_t)k * nx, nullptr);
  int s = 0;
  for (int k = 0; k < nt; ++k) {
    pp.wait(s);
    double* su = pp.row(s, 0);
    pp.template ready<false>(su);
    const double* sh = pp.row(s, 1);
    double* yo = pp.out(k & 1);
    double* yg = y + (size_t)k * nx;
    double uk[Q], uhk[Q], rhs[Q], a[Q], b[Q], c[Q], hv[Q];
#pragma unroll
    for (int j = 0; j < Q; ++j) {
      const int i = lane * Q + j;
      if (i < nx) {
        uk[j] = su[i];
        uhk[j] = sh[i];
        if (k == 0) {
          hv[j] = uk[j] - u0r[j];
        } else {  // h = u[k] - u[k-1] - dt (D Lap u[k] + rho u[k](1-u[k])); mirrored halo = Neumann ghost cells
          hv[j] = uk[j] - upr[j] - P.fi_a * ((su[i - 1] - uk[j]) + (su[i + 1] - uk[j])) -
                  P.fi_dtrho * uk[j] * (1.0 - uk[j]);
        }
        rhs[j] = hv[j] + qo[j];
      } else {
        uk[j] = 0.0; uhk[j] = 0.0; hv[j] = 0.0; rhs[j] = 0.0;
      }
    }
    if (k > 0) {
      fisher_matrix<Q>(P, uk, lane, a, b, c);
      warp_tridiag<Q>(a, b, c, rhs, lane);
    }
#pragma unroll
    for (int j = 0; j < Q; ++j) {
      const int i = lane * Q + j;
      if (i < nx) {
        const double q = rhs[j];
        const double w = uk[j] - uhk[j];
        const double yv = q - w;
        if (TMA) yo[i] = yv; else yg[i] = yv;
        const double ah = fabs(hv[j]);
        hinf = fmax(hinf, ah);
        h1 += ah;
        f2 = fma(w, w, f2);
        qo[j] = q;
        upr[j] = uk[j];
      }
    }
    if (TMA) fence_proxy_async_smem();
    __syncwarp();
    pp.store_row(yg, yo);
    pp.commit();
    if (k + nst < nt) pp.issue(s, u + (size_t)(k + nst) * nx, uh + (size_t)(k + nst) * nx, nullptr);
    if (++s == nst) s = 0;
  }
  pp.drain();
  hinf = warp_max(hinf);
  h1 = warp_sum(h1);
  f2 = warp_sum(f2);
  out.hinf = hinf;
  out.h1 = h1;
  out.f = 0.5 * f2;
  out.bad = !finite_d(hinf) | !finite_d(h1) | !finite_d(f2);
}

// ------------------------------------------------------------------------------------------------
// backward sweep: L^T lam = y (a5) and the step u+ = u_hat - J^T lam = u_hat - y (a8).
//   mode 0: write the trial point u+ to `unew`;  mode 1 (final solve): write the current iterate u to
//   `unew` (= u_star), lam only.  sig != nullptr: also store the level sums of lam (min-norm correction).
// Returns ||lam||_inf (NaN if anything was non-finite) and (u - u_hat)^T d, d = u+ - u.
// Burgers:  lam_{nt-1} = y_{nt-1} ,  lam_k = y_k + A_k^T lam_{k+1}   (A_k^T needs only u[k] at the own cell).
// ------------------------------------------------------------------------------------------------
template <int Q, bool FULL, bool TMA>
__device__ void bwd_sweep_b(const DevParams& P, Pipe<TMA>& pp, const double* __restrict__ u,
                            const double* __restrict__ uh, double* __restrict__ lam, double* __restrict__ unew,
                            int mode, double* __restrict__ sig, double& linf_out, double& wd_out, double& dd_out) {
  const int nx = P.nx, nt = P.nt, lane = pp.lane, nst = pp.nst;
  const double a0 = P.bs_a0, e = P.bs_e, hs = P.bs_hs;
  double linf = 0.0, wd = 0.0, dd = 0.0;
  double lo[Q];
#pragma unroll
  for (int j = 0; j < Q; ++j) lo[j] = 0.0;
  const int npro = nst < nt ? nst : nt;
  for (int t = 0; t < npro; ++t) {
    const size_t o = (size_t)(nt - 1 - t) * nx;
    pp.issue(t, lam + o, u + o, uh + o);
  }
  // lam_{nt} = 0: clear the ring slot the first step reads its neighbours from
  {
    double* z = pp.out(2) - 1;
    for (int i = lane; i < nx + 2; i += 32) z[i] = 0.0;
  }
  int s = 0, r3 = 0;
  for (int t = 0; t < nt; ++t) {
    const int k = nt - 1 - t;
    pp.wait(s);
    pp.template ready<true>(nullptr);
    const double* sy = pp.row(s, 0) + lane;
    const double* su = pp.row(s, 1) + lane;
    const double* sh = pp.row(s, 2) + lane;
    double* lc0 = pp.out(r3);
    double* lc = lc0 + lane;
    const double* lp = pp.out(r3 == 0 ? 2 : r3 - 1) + lane;
    double* uo0 = pp.out(3 + (t & 1));
    double* uo = uo0 + lane;
    double* lg = lam + (size_t)k * nx;
    double* ug = unew + (size_t)k * nx;
    double lsum = 0.0;
#pragma unroll
    for (int j = 0; j < Q; ++j) {
      const int o = 32 * j;
      if (FULL || lane + o < nx) {
        const double yv = sy[o], v = su[o], uhk = sh[o];
        const double l = fma(fma(-hs, v, e), lp[o - 1], fma(fma(hs, v, e), lp[o + 1], fma(a0, lo[j], yv)));
        lc[o] = l;
        if (FULL) {
          if (j == 0 && lane == 0) lc0[nx] = l;
          if (j == Q - 1 && lane == 31) lc0[-1] = l;
        } else {
          if (lane + o == 0) lc0[nx] = l;
          if (lane + o == nx - 1) lc0[-1] = l;
        }
        const double step = uhk - yv;
        const double un = (mode == 0) ? step : v;
        if (TMA) uo[o] = un; else { lg[lane + o] = l; ug[lane + o] = un; }
        wd = fma(v - uhk, step - v, wd);
        dd = fma(step - v, step - v, dd);
        linf = fmax(linf, fabs(l));
        lsum += l;
        lo[j] = l;
      }
    }
    if (sig) {
      const double sk = warp_sum(lsum);
      if (lane == 0) sig[k] = sk;
    }
    if (TMA) fence_proxy_async_smem();
    __syncwarp();
    pp.store_row(lg, lc0);
    pp.store_row(ug, uo0);
    pp.commit();
    if (t + nst < nt) {
      const size_t o = (size_t)(k - nst) * nx;
      pp.issue(s, lam + o, u + o, uh + o);
    }
    if (++s == nst) s = 0;
    if (++r3 == 3) r3 = 0;
  }
  pp.drain();
  linf = warp_max(linf);
  wd = warp_sum(wd);
  dd = warp_sum(dd);
  // fmax drops NaN: detect a non-finite multiplier / step through the sum as well
  linf_out = (finite_d(wd) && finite_d(dd)) ? linf : __longlong_as_double(0x7ff8000000000000LL);
  wd_out = wd;
  dd_out = dd;
}

// Fisher:  T_k lam_k = y_k + lam_{k+1}  (k >= 1, T symmetric) ,  lam_0 = y_0 + lam_1.
template <int Q, bool TMA>
__device__ void bwd_sweep_f(const DevParams& P, Pipe<TMA>& pp, const double* __restrict__ u,
                            const double* __restrict__ uh, double* __restrict__ lam, double* __restrict__ unew,
                            int mode, double& linf_out, double& wd_out, double& dd_out) {
  const int nx = P.nx, nt = P.nt, lane = pp.lane, nst = pp.nst;
  double linf = 0.0, wd = 0.0, dd = 0.0;
  double lo[Q];
#pragma unroll
  for (int j = 0; j < Q; ++j) lo[j] = 0.0;
  const int npro = nst < nt ? nst : nt;
  for (int t = 0; t < npro; ++t) {
    const size_t o = (size_t)(nt - 1 - t) * nx;
    pp.issue(t, lam + o, u + o, uh + o);
  }
  int s = 0;
  for (int t = 0; t < nt; ++t) {
    const int k = nt - 1 - t;
    pp.wait(s);
    pp.template ready<false>(nullptr);
    const double* sy = pp.row(s, 0);
    const double* su = pp.row(s, 1);
    const double* sh = pp.row(s, 2);
    double* lc = pp.out(t & 1);
    double* uo = pp.out(3 + (t & 1));
    double* lg = lam + (size_t)k * nx;
    double* ug = unew + (size_t)k * nx;
    double uk[Q], yv[Q], uhk[Q], rhs[Q], a[Q], b[Q], c[Q];
#pragma unroll
    for (int j = 0; j < Q; ++j) {
      const int i = lane * Q + j;
      if (i < nx) {
        yv[j] = sy[i]; uk[j] = su[i]; uhk[j] = sh[i];
        rhs[j] = yv[j] + lo[j];
      } else {
        yv[j] = 0.0; uk[j] = 0.0; uhk[j] = 0.0; rhs[j] = 0.0;
      }
    }
    if (k > 0) {
      fisher_matrix<Q>(P, uk, lane, a, b, c);
      warp_tridiag<Q>(a, b, c, rhs, lane);
    }
#pragma unroll
    for (int j = 0; j < Q; ++j) {
      const int i = lane * Q + j;
      if (i < nx) {
        const double l = rhs[j];
        const double step = uhk[j] - yv[j];
        const double un = (mode == 0) ? step : uk[j];
        if (TMA) { lc[i] = l; uo[i] = un; } else { lg[i] = l; ug[i] = un; }
        wd = fma(uk[j] - uhk[j], step - uk[j], wd);
        dd = fma(step - uk[j], step - uk[j], dd);
        linf = fmax(linf, fabs(l));
        lo[j] = l;
      }
    }
    if (TMA) fence_proxy_async_smem();
    __syncwarp();
    pp.store_row(lg, lc);
    pp.store_row(ug, uo);
    pp.commit();
    if (t + nst < nt) {
      const size_t o = (size_t)(k - nst) * nx;
      pp.issue(s, lam + o, u + o, uh + o);
    }
    if (++s == nst) s = 0;
  }
  pp.drain();
  linf = warp_max(linf);
  wd = warp_sum(wd);
  dd = warp_sum(dd);
  linf_out = (finite_d(wd) && finite_d(dd)) ? linf : __longlong_as_double(0x7ff8000000000000LL);
  wd_out = wd;
  dd_out = dd;
}

// Minimum-norm multiplier for the linearly dependent mass rows of kind 4 (streaming
// recipe): with level sums sigma_j of the basic solution (mass multipliers 0) and c = nx dx^2,
//   (D^T D + c I) t = -dx D^T sigma     [ <=> (I + c L1 L1^T) t = N lam_basic ; D = L1^{-1} first difference ]
//   lam_mass[k] = -t_k ;  lam_loc[j][.] += dx sum_{k>=j} t_k .
static __device__ void min_norm_burgers_mass(const DevParams& P, int lane, double* __restrict__ lam, double* __restrict__ sig,
                                      double* __restrict__ tt) {
  const int nx = P.nx, nt = P.nt;
  const double c = (double)nx * P.dx * P.dx;
  __syncwarp();
  if (lane == 0) {
    // Thomas on the SPD tridiagonal (2+c, ..., 2+c, 1+c) / off-diagonals -1; tt doubles as c' storage first
    double cp = 0.0, dp = 0.0;
    for (int k = 0; k < nt; ++k) {
      const double bk = -P.dx * (sig[k] - (k + 1 < nt ? sig[k + 1] : 0.0));
      const double diag = ((k == nt - 1) ? 1.0 : 2.0) + c;
      const double den = diag + cp;  // diag - (-1) * cp_prev, cp_prev = -1/den_prev  (stored negative)
      const double inv = 1.0 / den;
      dp = (bk + dp) * inv;          // (b_k - (-1) d_prev) / den
      cp = -inv;                     // c'_k = -1 / den
      tt[k] = dp;
      sig[k] = cp;
    }
    double x = tt[nt - 1];
    double suf = x;
    tt[nt - 1] = x;
    sig[nt - 1] = suf;  // sig now holds the suffix sums of t
    for (int k = nt - 2; k >= 0; --k) {
      x = tt[k] - sig[k] * x;
      tt[k] = x;
      suf += x;
      sig[k] = suf;
    }
  }
  __syncwarp();
  double* lmass = lam + (size_t)nt * nx;
  for (int k = lane; k < nt; k += 32) lmass[k] = -tt[k];
  for (int k = 0; k < nt; ++k) {
    const double add = P.dx * sig[k];
    double* row = lam + (size_t)k * nx;
    for (int i = lane; i < nx; i += 32) row[i] += add;
  }
}

// ------------------------------------------------------------------------------------------------
// the persistent Gauss-Newton driver (a8, a9): one warp per sample
// ------------------------------------------------------------------------------------------------
template <int KIND, int Q, bool FULL, bool TMA>
__global__ void __launch_bounds__(256) project1d_kernel(const __grid_constant__ Proj1dArgs A) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const DevParams& P = A.P;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int b = blockIdx.x * (blockDim.x >> 5) + warp;
  if (b >= A.batch) return;
  const int nx = P.nx, nt = P.nt;
  const size_t n = (size_t)P.n;

  unsigned char* base = smem_raw + (size_t)warp * A.warp_bytes;
  Pipe<TMA> pp;
  pp.stage = reinterpret_cast<double*>(base);
  pp.srow = pp.stage + (size_t)A.nst * 3 * A.rp;
  pp.bar0 = smem_u32(pp.srow + (size_t)5 * A.rp);
  pp.phase = 0;
  pp.nst = A.nst; pp.rp = A.rp; pp.nx = nx; pp.lane = lane;
  if (lane == 0) {
    for (int s = 0; s < A.nst; ++s) mbar_init(pp.bar0 + 8u * s, 1);
    mbar_fence_init();
    fence_proxy_async_smem();
  }
  // zero the output/staging rows once: halo cells and q_{-1} must read as finite zeros
  for (int i = lane; i < 5 * A.rp; i += 32) pp.srow[i] = 0.0;
  __syncwarp();

  const double* uh = A.u_hat + (size_t)b * n;
  const double* u0 = A.cdata + (size_t)b * nx;
  double* ustar = A.u_star + (size_t)b * n;
  double* lam = A.lam + (size_t)b * P.m;
  double* bufA = A.bufA + (size_t)b * n;
  double* bufB = A.bufB + (size_t)b * n;
  double* sig = A.aux + (size_t)b * 2 * nt;
  double* tt = sig + nt;

  double M0 = 0.0;
  if (P.has_mass) {
    double sm = 0.0;
    for (int i = lane; i < nx; i += 32) sm += u0[i];
    M0 = P.dx * warp_sum(sm);
  }
  double mu = 0.0;  // DESIGN.md R2/R3: the penalty parameter needs no multiplier; `warm` is ignored for 1D kinds

  const double* cur = uh;   // accepted iterate
  double* trial = bufA;     // where the next trial point goes
  bool have_trial = false, polishing = false;
  int polish_left = 0, steps = 0, solves = 0, tries = 0, status = 0, nfwd = 0, nbwd = 0, nback = 0;
  double alpha = 1.0, phi_cur = 0.0, Dphi = 0.0;
  SweepNorms nrm;
  const bool want_sig = (P.kind == SNAP_BURGERS1D_LF_MASS) && (P.lambda_mode == 0);

  while (true) {
    const double* pt = have_trial ? trial : cur;
    if constexpr (KIND == KB) fwd_sweep_b<Q, FULL, TMA>(P, pp, pt, uh, u0, lam, M0, nrm);
    else fwd_sweep_f<Q, TMA>(P, pp, pt, uh, u0, lam, nrm);
    ++nfwd;
    if (have_trial) {
      if (!polishing) {
        const double phi_t = nrm.f + mu * nrm.h1;
        const bool ok = !nrm.bad && finite_d(phi_t) && (phi_t <= phi_cur + P.ls_c1 * alpha * Dphi);
        if (!ok) {
          if (++tries > P.ls_max) { status = SNAP_ST_LINESEARCH; break; }
          for (size_t i = lane; i < n; i += 32) trial[i] = fma(P.ls_shrink, trial[i] - cur[i], cur[i]);
          __threadfence_block();
          __syncwarp();
          alpha *= P.ls_shrink;
          ++nback;
          continue;
        }
        ++steps;
      }
      cur = trial;
      trial = (trial == bufA) ? bufB : bufA;
      have_trial = false;
    } else if (nrm.bad) {
      status = SNAP_ST_NONFINITE;
      break;
    }
    ++solves;
    const bool conv = nrm.hinf < P.tol;
    bool final_solve = false;
    if (polishing) {
      final_solve = (polish_left == 0);
    } else if (conv) {
      polishing = true;
      polish_left = (nrm.hinf > kPolishSkip * P.tol) ? P.polish : 0;
      final_solve = (polish_left == 0);
    } else if (steps >= P.max_iter) {
      status = SNAP_ST_MAXITER;
      final_solve = true;
    }
    double linf, wd, dd;
    if (final_solve) {
      if constexpr (KIND == KB) bwd_sweep_b<Q, FULL, TMA>(P, pp, cur, uh, lam, ustar, 1, want_sig ? sig : nullptr, linf, wd, dd);
      else bwd_sweep_f<Q, TMA>(P, pp, cur, uh, lam, ustar, 1, linf, wd, dd);
      ++nbwd;
      if (!finite_d(linf)) status = SNAP_ST_NONFINITE;
      break;
    }
    if constexpr (KIND == KB) bwd_sweep_b<Q, FULL, TMA>(P, pp, cur, uh, lam, trial, 0, nullptr, linf, wd, dd);
    else bwd_sweep_f<Q, TMA>(P, pp, cur, uh, lam, trial, 0, linf, wd, dd);
    ++nbwd;
    if (!finite_d(linf)) { status = SNAP_ST_NONFINITE; break; }
    if (polishing) {
      --polish_left;
    } else {
      mu = merit_mu(mu, wd, dd, nrm.h1, kMuRho, kMuFloor);
      phi_cur = nrm.f + mu * nrm.h1;
      Dphi = wd - mu * nrm.h1;
      alpha = 1.0;
      tries = 0;
    }
    have_trial = true;
  }

  if (status == SNAP_ST_NONFINITE) {  // R16: u* = u_hat, lam = 0
    if (ustar != uh)
      for (size_t i = lane; i < n; i += 32) ustar[i] = uh[i];
    for (size_t i = lane; i < (size_t)P.m; i += 32) lam[i] = 0.0;
  } else if (status == SNAP_ST_LINESEARCH) {  // u* = last accepted iterate, lam = last lam+
    if (ustar != cur)
      for (size_t i = lane; i < n; i += 32) ustar[i] = cur[i];
    if (P.has_mass)
      for (int k = lane; k < nt; k += 32) lam[n + k] = 0.0;
  } else if (P.has_mass) {
    if (want_sig) {
      min_norm_burgers_mass(P, lane, lam, sig, tt);
    } else {
      for (int k = lane; k < nt; k += 32) lam[n + k] = 0.0;
    }
  }
  if (lane == 0) {
    A.iters[b] = (status == 0) ? solves : status;
    if (A.stats) {   // the traffic of this variant: forward sweep reads u, u_hat, writes y; backward reads y, u, u_hat, writes lam, u+
      long long* stat = A.stats + (size_t)b * SNAP_STAT_COUNT;
      stat[SNAP_STAT_LINEARISATIONS] = solves; stat[SNAP_STAT_PASSES] = nfwd + nbwd;
      stat[SNAP_STAT_ROWS_READ] = (long long)nt * (2 * nfwd + 3 * nbwd);
      stat[SNAP_STAT_ROWS_WRITTEN] = (long long)nt * (nfwd + 2 * nbwd);
      stat[SNAP_STAT_VARIANT] = A.variant; stat[SNAP_STAT_INNER] = 0; stat[SNAP_STAT_ROW_DOUBLES] = nx;
      stat[SNAP_STAT_BACKTRACKS] = nback;
    }
  }
}

template <int KIND, int Q, bool FULL, bool TMA>
inline int launch_1d_variant(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st) {
  auto kern = project1d_kernel<KIND, Q, FULL, TMA>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem) != cudaSuccess)
    return SNAP_ECUDA;
  kern<<<pl.grid, pl.wpc * 32, pl.smem, st>>>(a);
  return cudaGetLastError() == cudaSuccess ? SNAP_OK : SNAP_ECUDA;
}

template <int KIND, int Q>
inline int launch_1d_q(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st) {
  if (KIND == KB) {
    if (pl.tma)
      return pl.full ? launch_1d_variant<KB, Q, true, true>(a, pl, st) : launch_1d_variant<KB, Q, false, true>(a, pl, st);
    return launch_1d_variant<KB, Q, false, false>(a, pl, st);
  }
  return pl.tma ? launch_1d_variant<KF, Q, false, true>(a, pl, st) : launch_1d_variant<KF, Q, false, false>(a, pl, st);
}

template <int KIND>
inline int launch_1d_kind(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st) {
  switch (pl.q) {
    case 1: return launch_1d_q<KIND, 1>(a, pl, st);
    case 2: return launch_1d_q<KIND, 2>(a, pl, st);
    case 4: return launch_1d_q<KIND, 4>(a, pl, st);
    case 8: return launch_1d_q<KIND, 8>(a, pl, st);
    case 16: return launch_1d_q<KIND, 16>(a, pl, st);
  }
  return SNAP_EINVAL;
}

}  // namespace snap
