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
#include "snap_internal.h"

namespace snap {

constexpr int KB = 1;  // Burgers family: lane owns cells lane + 32 j   (conflict-free shared-memory access)
constexpr int KF = 2;  // Fisher family:  lane owns cells lane*Q + j    (contiguous, for the warp tridiagonal solve)

struct Proj1dArgs {
  DevParams P;
  int batch, warm;
  const double* u_hat;
  const double* cdata;
  double* u_star;
  double* lam;
  int* iters;
  double* bufA;  // [batch][n]  trial / iterate ping-pong
  double* bufB;  // [batch][n]
  double* aux;   // [batch][2*nt]  level sums and null-space coefficients (min-norm multiplier, kind 4)
  int nst;       // ring depth (levels in flight per warp)
  int nxp;       // row pitch in doubles (nx rounded up to even)
  int tma;       // 1: rows are 16-byte aligned -> bulk copies; 0: plain loads/stores
  int warp_bytes;
};

// ------------------------------------------------------------------------------------------------
// per-warp row pipeline
// ------------------------------------------------------------------------------------------------
struct Pipe {
  double* stage;   // [nst][3][nxp]
  double* srow;    // [5][nxp]
  uint32_t bar0;   // shared address of mbarrier 0
  uint32_t phase;  // parity to wait for, one bit per stage
  int nst, nxp, nx, tma, lane;

  __device__ __forceinline__ double* row(int s, int r) const { return stage + (size_t)(s * 3 + r) * nxp; }
  __device__ __forceinline__ double* out(int r) const { return srow + (size_t)r * nxp; }

  // Load up to three global rows of nx doubles into stage s.  Called by the whole (converged) warp after
  // every lane has finished reading the previous contents of the stage.
  __device__ __forceinline__ void issue(int s, const double* g0, const double* g1, const double* g2) {
    __syncwarp();
    const uint32_t bar = bar0 + 8u * s;
    if (tma) {
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
  // make the shared-memory output rows written >= 2 steps ago reusable
  __device__ __forceinline__ void out_reuse() {
    if (tma && lane == 0) bulk_wait_read<1>();
    __syncwarp();
  }
  // lanes have written an output row with generic stores; hand it to the bulk-store engine
  __device__ __forceinline__ void store_row(double* g, const double* s_row) {
    if (tma && lane == 0) bulk_s2g(g, smem_u32(s_row), (uint32_t)nx * 8u);
  }
  __device__ __forceinline__ void commit() {
    if (tma && lane == 0) bulk_commit();
  }
  // all outstanding bulk stores of this warp are complete and visible to later loads
  __device__ __forceinline__ void drain() {
    if (tma) {
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

template <int KIND, int Q>
__device__ __forceinline__ int cell(int lane, int j) {
  return KIND == KB ? lane + 32 * j : lane * Q + j;
}

// ------------------------------------------------------------------------------------------------
// warp tridiagonal solve (Fisher): rows owned contiguously, Q per lane; partition method —
// each lane eliminates its Q-1 interior unknowns against its own last unknown (the separator) and the
// previous lane's, the 32 separators are solved by parallel cyclic reduction with shuffles.
// Row j of lane p:  a[j] x_{-1} + b[j] x_j + c[j] x_{+1} = d[j].  a of the first global row and c of the
// last must be 0; padding rows are identity rows.  Solution returned in d.
// ------------------------------------------------------------------------------------------------
template <int Q>
__device__ __forceinline__ void warp_tridiag(const double (&a)[Q], const double (&b)[Q], const double (&c)[Q],
                                             double (&d)[Q], int lane) {
  double ra, rb, rc, rd;
  double v[Q], al[Q], be[Q];
  if (Q > 1) {
    double cp[Q];
    {
      const double inv = 1.0 / b[0];
      cp[0] = (Q > 2 ? c[0] : 0.0) * inv;
      v[0] = d[0] * inv;
      al[0] = a[0] * inv;
      be[0] = (Q == 2 ? c[0] : 0.0) * inv;
    }
#pragma unroll
    for (int j = 1; j < Q - 1; ++j) {
      const double inv = 1.0 / (b[j] - a[j] * cp[j - 1]);
      cp[j] = (j < Q - 2 ? c[j] : 0.0) * inv;
      v[j] = (d[j] - a[j] * v[j - 1]) * inv;
      al[j] = (-a[j] * al[j - 1]) * inv;
      be[j] = ((j == Q - 2 ? c[j] : 0.0) - a[j] * be[j - 1]) * inv;
    }
#pragma unroll
    for (int j = Q - 3; j >= 0; --j) {
      v[j] -= cp[j] * v[j + 1];
      al[j] -= cp[j] * al[j + 1];
      be[j] -= cp[j] * be[j + 1];
    }
    // separator row Q-1: a x_{Q-2} + b s_p + c x_{p+1,0} = d with x = v - s_{p-1} al - s_p be
    const double v0n = __shfl_down_sync(SNAP_FULL, v[0], 1);
    const double al0n = __shfl_down_sync(SNAP_FULL, al[0], 1);
    const double be0n = __shfl_down_sync(SNAP_FULL, be[0], 1);
    const double cl = (lane == 31) ? 0.0 : c[Q - 1];
    ra = -a[Q - 1] * al[Q - 2];
    rb = b[Q - 1] - a[Q - 1] * be[Q - 2] - cl * al0n;
    rc = -cl * be0n;
    rd = d[Q - 1] - a[Q - 1] * v[Q - 2] - cl * v0n;
  } else {
    ra = a[0];
    rb = b[0];
    rc = (lane == 31) ? 0.0 : c[0];
    rd = d[0];
  }
  if (lane == 0) ra = 0.0;
  // parallel cyclic reduction over the 32 lanes, rows kept normalised (rb == 1)
  {
    const double inv = 1.0 / rb;
    ra *= inv;
    rc *= inv;
    rd *= inv;
  }
#pragma unroll
  for (int s = 1; s < 32; s <<= 1) {
    double alo = __shfl_up_sync(SNAP_FULL, ra, s), clo = __shfl_up_sync(SNAP_FULL, rc, s),
           dlo = __shfl_up_sync(SNAP_FULL, rd, s);
    double ahi = __shfl_down_sync(SNAP_FULL, ra, s), chi = __shfl_down_sync(SNAP_FULL, rc, s),
           dhi = __shfl_down_sync(SNAP_FULL, rd, s);
    if (lane < s) { alo = 0.0; clo = 0.0; dlo = 0.0; }
    if (lane + s > 31) { ahi = 0.0; chi = 0.0; dhi = 0.0; }
    const double nb = 1.0 - clo * ra - ahi * rc;
    const double inv = 1.0 / nb;
    const double nd = (rd - dlo * ra - dhi * rc) * inv;
    const double na = (-alo * ra) * inv;
    const double nc = (-chi * rc) * inv;
    ra = na; rc = nc; rd = nd;
  }
  const double s_me = rd;
  if (Q > 1) {
    double s_prev = __shfl_up_sync(SNAP_FULL, s_me, 1);
    if (lane == 0) s_prev = 0.0;
#pragma unroll
    for (int j = 0; j < Q - 1; ++j) d[j] = v[j] - s_prev * al[j] - s_me * be[j];
  }
  d[Q - 1] = s_me;
}

// Fisher: tridiagonal T_k = I - dt D Lap_h - dt rho diag(1 - 2u) restricted to this lane's rows.
template <int Q>
__device__ __forceinline__ void fisher_matrix(const DevParams& P, const double (&uk)[Q], int lane, double (&a)[Q],
                                              double (&b)[Q], double (&c)[Q]) {
#pragma unroll
  for (int j = 0; j < Q; ++j) {
    const int i = lane * Q + j;
    if (i < P.nx) {
      const double nnb = (i == 0 || i == P.nx - 1) ? 1.0 : 2.0;
      a[j] = (i == 0) ? 0.0 : -P.fi_a;
      c[j] = (i == P.nx - 1) ? 0.0 : -P.fi_a;
      b[j] = 1.0 + P.fi_a * nnb - P.fi_dtrho * (1.0 - 2.0 * uk[j]);
    } else {
      a[j] = 0.0; b[j] = 1.0; c[j] = 0.0;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// forward sweep: residual h (a1), Jacobian coefficients (a2), rhs (a3) and L y = r (a5), level by level.
// Reads u (point of linearisation) and u_hat rows, writes y into the multiplier buffer.
// ------------------------------------------------------------------------------------------------
template <int KIND, int Q>
__device__ void fwd_sweep(const DevParams& P, Pipe& pp, const double* __restrict__ u, const double* __restrict__ uh,
                          const double* __restrict__ u0, double* __restrict__ y, double M0, SweepNorms& out) {
  const int nx = P.nx, nt = P.nt, lane = pp.lane, nst = pp.nst;
  double hinf = 0.0, h1 = 0.0, f2 = 0.0, minf = 0.0, m1 = 0.0;
  int bad = 0;
  double u0r[Q], qo[Q];
  double phi[Q], cpj[Q], cmj[Q];  // Burgers: Phi(u[k-1])_i and dPhi_i/du_{i+-1}, carried one level
  double upr[Q];                  // Fisher: u[k-1] own cells
#pragma unroll
  for (int j = 0; j < Q; ++j) {
    const int i = cell<KIND, Q>(lane, j);
    u0r[j] = (i < nx) ? u0[i] : 0.0;
    qo[j] = 0.0; phi[j] = 0.0; cpj[j] = 0.0; cmj[j] = 0.0; upr[j] = 0.0;
  }
  const int npro = nst < nt ? nst : nt;
  for (int k = 0; k < npro; ++k) pp.issue(k, u + (size_t)k * nx, uh + (size_t)k * nx, nullptr);
  int s = 0;
  for (int k = 0; k < nt; ++k) {
    pp.wait(s);
    pp.out_reuse();
    const double* su = pp.row(s, 0);
    const double* sh = pp.row(s, 1);
    double* yo = pp.out(k & 1);
    double* qc = pp.out(2 + (k & 1));
    const double* qp = pp.out(2 + ((k + 1) & 1));
    double* yg = y + (size_t)k * nx;
    double msum = 0.0;
    if (KIND == KB) {
#pragma unroll
      for (int j = 0; j < Q; ++j) {
        const int i = lane + 32 * j;
        if (i < nx) {
          const int ip = (i + 1 == nx) ? 0 : i + 1;
          const int im = (i == 0) ? nx - 1 : i - 1;
          const double uk = su[i], uhk = sh[i], up = su[ip], um = su[im];
          double h, q;
          if (k == 0) {
            h = uk - u0r[j];
            q = h;
          } else {
            h = uk - phi[j];
            q = fma(cpj[j], qp[ip], fma(cmj[j], qp[im], fma(P.bs_a0, qo[j], h)));
          }
          const double w = uk - uhk;
          const double yv = q - w;
          qc[i] = q;
          if (pp.tma) yo[i] = yv; else yg[i] = yv;
          const double ah = fabs(h);
          bad |= !finite_d(ah) | !finite_d(q);
          hinf = fmax(hinf, ah);
          h1 += ah;
          f2 = fma(w, w, f2);
          msum += uk;
          phi[j] = fma(P.bs_a0, uk, (up + um) * fma(-P.bs_qs, up - um, P.bs_e));
          cpj[j] = fma(-P.bs_hs, up, P.bs_e);
          cmj[j] = fma(P.bs_hs, um, P.bs_e);
          qo[j] = q;
        }
      }
    } else {
      double uk[Q], uhk[Q], rhs[Q], a[Q], b[Q], c[Q], hv[Q];
#pragma unroll
      for (int j = 0; j < Q; ++j) {
        const int i = lane * Q + j;
        if (i < nx) {
          uk[j] = su[i];
          uhk[j] = sh[i];
          if (k == 0) {
            hv[j] = uk[j] - u0r[j];
          } else {
            const double ul = (i > 0) ? su[i - 1] : uk[j];
            const double ur = (i < nx - 1) ? su[i + 1] : uk[j];
            // h = u[k] - u[k-1] - dt (D Lap u[k] + rho u[k](1-u[k]))
            hv[j] = uk[j] - upr[j] - P.fi_a * ((ul - uk[j]) + (ur - uk[j])) - P.fi_dtrho * uk[j] * (1.0 - uk[j]);
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
          if (pp.tma) yo[i] = yv; else yg[i] = yv;
          const double ah = fabs(hv[j]);
          bad |= !finite_d(ah) | !finite_d(q);
          hinf = fmax(hinf, ah);
          h1 += ah;
          f2 = fma(w, w, f2);
          qo[j] = q;
          upr[j] = uk[j];
        }
      }
    }
    if (P.has_mass) {
      const double hm = fabs(P.dx * warp_sum(msum) - M0);
      minf = fmax(minf, hm);
      m1 += hm;
    }
    if (pp.tma) fence_proxy_async_smem();
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
  bad = warp_or(bad);
  if (P.has_mass) {
    bad |= !finite_d(minf);
    hinf = fmax(hinf, minf);
    h1 += m1;
  }
  out.hinf = hinf;
  out.h1 = h1;
  out.f = 0.5 * f2;
  out.bad = bad | !finite_d(hinf) | !finite_d(h1) | !finite_d(f2);
}

// ------------------------------------------------------------------------------------------------
// backward sweep: L^T lam = y (a5) and the step u+ = u_hat - J^T lam = u_hat - y (a8).
//   mode 0: write the trial point u+ to `unew`;  mode 1 (final solve): write the current iterate u to
//   `unew` (= u_star), lam only.  sig != nullptr: also store the level sums of lam (min-norm correction).
// Returns ||lam||_inf and (u - u_hat)^T d, d = u+ - u.
// ------------------------------------------------------------------------------------------------
template <int KIND, int Q>
__device__ void bwd_sweep(const DevParams& P, Pipe& pp, const double* __restrict__ u, const double* __restrict__ uh,
                          double* __restrict__ lam, double* __restrict__ unew, int mode, double* __restrict__ sig,
                          double& linf_out, double& wd_out) {
  const int nx = P.nx, nt = P.nt, lane = pp.lane, nst = pp.nst;
  double linf = 0.0, wd = 0.0;
  double lo[Q];
#pragma unroll
  for (int j = 0; j < Q; ++j) lo[j] = 0.0;
  const int npro = nst < nt ? nst : nt;
  for (int t = 0; t < npro; ++t) {
    const size_t o = (size_t)(nt - 1 - t) * nx;
    pp.issue(t, lam + o, u + o, uh + o);
  }
  int s = 0, r3 = 0;
  for (int t = 0; t < nt; ++t) {
    const int k = nt - 1 - t;
    pp.wait(s);
    pp.out_reuse();
    const double* sy = pp.row(s, 0);
    const double* su = pp.row(s, 1);
    const double* sh = pp.row(s, 2);
    double* lc = pp.out(r3);
    const double* lp = pp.out(r3 == 0 ? 2 : r3 - 1);
    double* uo = pp.out(3 + (t & 1));
    double* lg = lam + (size_t)k * nx;
    double* ug = unew + (size_t)k * nx;
    double lsum = 0.0;
    if (KIND == KB) {
#pragma unroll
      for (int j = 0; j < Q; ++j) {
        const int i = lane + 32 * j;
        if (i < nx) {
          const int ip = (i + 1 == nx) ? 0 : i + 1;
          const int im = (i == 0) ? nx - 1 : i - 1;
          const double yv = sy[i], v = su[i], uhk = sh[i];
          double l = yv;
          if (t > 0)  // lam_k = y_k + A_k^T lam_{k+1}
            l = fma(fma(-P.bs_hs, v, P.bs_e), lp[im], fma(fma(P.bs_hs, v, P.bs_e), lp[ip], fma(P.bs_a0, lo[j], yv)));
          lc[i] = l;
          const double un = (mode == 0) ? (uhk - yv) : v;
          if (pp.tma) uo[i] = un; else { lg[i] = l; ug[i] = un; }
          const double w = v - uhk;
          wd = fma(w, (uhk - yv) - v, wd);
          linf = fmax(linf, fabs(l));
          lsum += l;
          lo[j] = l;
        }
      }
    } else {
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
      if (k > 0) {  // T_k lam_k = y_k + lam_{k+1}   (level 0: identity block)
        fisher_matrix<Q>(P, uk, lane, a, b, c);
        warp_tridiag<Q>(a, b, c, rhs, lane);
      }
#pragma unroll
      for (int j = 0; j < Q; ++j) {
        const int i = lane * Q + j;
        if (i < nx) {
          const double l = rhs[j];
          const double un = (mode == 0) ? (uhk[j] - yv[j]) : uk[j];
          if (pp.tma) { lc[i] = l; uo[i] = un; } else { lg[i] = l; ug[i] = un; }
          const double w = uk[j] - uhk[j];
          wd = fma(w, (uhk[j] - yv[j]) - uk[j], wd);
          linf = fmax(linf, fabs(l));
          lsum += l;
          lo[j] = l;
        }
      }
    }
    if (sig) {
      const double sk = warp_sum(lsum);
      if (lane == 0) sig[k] = sk;
    }
    if (pp.tma) fence_proxy_async_smem();
    __syncwarp();
    pp.store_row(lg, lc);
    pp.store_row(ug, uo);
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
  // fmax drops NaN: detect a non-finite multiplier through the sum as well
  linf_out = finite_d(wd) ? linf : __longlong_as_double(0x7ff8000000000000LL);
  wd_out = wd;
}

// Minimum-norm multiplier for the linearly dependent mass rows of kind 4 (streaming
// recipe): with level sums sigma_j of the basic solution (mass multipliers 0) and c = nx dx^2,
//   (D^T D + c I) t = -dx D^T sigma     [ <=> (I + c L1 L1^T) t = N lam_basic ; D = L1^{-1} first difference ]
//   lam_mass[k] = -t_k ;  lam_loc[j][.] += dx sum_{k>=j} t_k .
__device__ void min_norm_burgers_mass(const DevParams& P, int lane, double* __restrict__ lam, double* __restrict__ sig,
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
template <int KIND, int Q>
__global__ void __launch_bounds__(256) project1d_kernel(const __grid_constant__ Proj1dArgs A) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const DevParams& P = A.P;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int b = blockIdx.x * (blockDim.x >> 5) + warp;
  if (b >= A.batch) return;
  const int nx = P.nx, nt = P.nt;
  const size_t n = (size_t)P.n;

  unsigned char* base = smem_raw + (size_t)warp * A.warp_bytes;
  Pipe pp;
  pp.stage = reinterpret_cast<double*>(base);
  pp.srow = pp.stage + (size_t)A.nst * 3 * A.nxp;
  pp.bar0 = smem_u32(pp.srow + (size_t)5 * A.nxp);
  pp.phase = 0;
  pp.nst = A.nst; pp.nxp = A.nxp; pp.nx = nx; pp.tma = A.tma; pp.lane = lane;
  if (lane == 0) {
    for (int s = 0; s < A.nst; ++s) mbar_init(pp.bar0 + 8u * s, 1);
    mbar_fence_init();
    fence_proxy_async_smem();
  }
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
  double mu = 0.0;
  if (A.warm) {  // the incoming multipliers only seed the merit parameter for these kinds
    double li = 0.0;
    for (size_t i = lane; i < (size_t)P.m; i += 32) li = fmax(li, fabs(lam[i]));
    li = warp_max(li);
    if (finite_d(li)) mu = 1.1 * li + 1e-3;
  }

  const double* cur = uh;   // accepted iterate
  double* trial = bufA;     // where the next trial point goes
  bool have_trial = false, polishing = false;
  int polish_left = 0, steps = 0, solves = 0, tries = 0, status = 0;
  double alpha = 1.0, phi_cur = 0.0, Dphi = 0.0;
  SweepNorms nrm;
  const bool want_sig = (P.kind == SNAP_BURGERS1D_LF_MASS) && (P.lambda_mode == 0);

  while (true) {
    const double* pt = have_trial ? trial : cur;
    fwd_sweep<KIND, Q>(P, pp, pt, uh, u0, lam, M0, nrm);
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
    double linf, wd;
    if (final_solve) {
      bwd_sweep<KIND, Q>(P, pp, cur, uh, lam, ustar, 1, want_sig ? sig : nullptr, linf, wd);
      if (!finite_d(linf)) status = SNAP_ST_NONFINITE;
      break;
    }
    bwd_sweep<KIND, Q>(P, pp, cur, uh, lam, trial, 0, nullptr, linf, wd);
    if (!finite_d(linf)) { status = SNAP_ST_NONFINITE; break; }
    if (polishing) {
      --polish_left;
    } else {
      mu = fmax(mu, 1.1 * linf + 1e-3);
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
  if (lane == 0) A.iters[b] = (status == 0) ? solves : status;
}

}  // namespace snap
