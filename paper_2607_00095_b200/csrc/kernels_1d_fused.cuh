// Burgers family (kinds 1, 4), nx = 32 Q: fused Gauss-Newton sweeps, one persistent warp per sample.
//
// For these row sets J_loc is square, unit block lower-bidiagonal in time (diagonal blocks I, sub-diagonal
// blocks -A_{k-1}, A_k = dPhi/du at level k), so the Schur solve (J J^T) lam+ = r factors into the forward
// sweep L y = r and the backward sweep L^T lam+ = y with L = J_loc (oracle pin P6), and the
// Gauss-Newton step needs only the forward half:  J^T lam+ = y  =>  u+ = u_hat - y = u - q,  q = y + (u - u_hat):
//     q_0 = h_0 ,   q_k = h_k + A_{k-1} q_{k-1} ,   h_k = u[k] - Phi(u[k-1]).
// With the multiplier-free penalty parameter (R2) the multiplier half is postponed to the
// converged point.  Level k of iterate t+1 depends only on levels <= k of iterate t and level k-1 of
// iterate t+1, so ONE forward pass over the levels carries up to JT consecutive Gauss-Newton iterations
// (a1-a3, a5 forward half, a8): the u_hat row is read once, the last iterate written once, and the state of
// every iteration in flight (Phi(u[k-1]) and A_{k-1} q_{k-1}, 2 doubles per cell) stays in registers.  The
// Armijo tests of the fused steps are evaluated after the pass from per-iteration sums; if one fails the
// pass is discarded and the sample continues with one iteration per pass (classic back-tracking).
//
// Layout: lane l owns the Q contiguous cells l*Q .. l*Q+Q-1, neighbours are register-local except at the two
// ends (one shuffle each, periodic wrap for free).  Rows travel HBM <-> shared memory as 128-byte bulk (TMA)
// copies, one per lane, into rows padded by 16 bytes per 128 so that the lanes' 128-bit shared-memory
// accesses are bank-conflict free.
#pragma once
#include "device_utils.cuh"
#include "launch.h"
#include "snap_internal.h"

namespace snap {

template <int Q>
struct RowGeom {
  static constexpr int NX = 32 * Q;
  static constexpr int SEGS = NX / 16;   // 128-byte segments per row, one bulk copy (and one issuing lane) each
  static constexpr int RP = SEGS * 18;   // padded row pitch in doubles: 16 data + 2 pad per segment
};

// cell i of a row lives at double index i + 2 (i >> 4) of its padded shared-memory row
__device__ __forceinline__ int pad_idx(int i) { return i + 2 * (i >> 4); }

template <int Q>
__device__ __forceinline__ void load_cells(const double* row, int lane, double (&x)[Q]) {
  const double* p = row + pad_idx(Q * lane);
  if constexpr (Q == 1) {
    x[0] = p[0];
  } else {
#pragma unroll
    for (int c = 0; c < Q / 2; ++c) {
      const double2 t = reinterpret_cast<const double2*>(p)[c];
      x[2 * c] = t.x;
      x[2 * c + 1] = t.y;
    }
  }
}
template <int Q>
__device__ __forceinline__ void store_cells(double* row, int lane, const double (&x)[Q]) {
  double* p = row + pad_idx(Q * lane);
  if constexpr (Q == 1) {
    p[0] = x[0];
  } else {
#pragma unroll
    for (int c = 0; c < Q / 2; ++c) reinterpret_cast<double2*>(p)[c] = make_double2(x[2 * c], x[2 * c + 1]);
  }
}

__device__ __forceinline__ double shfl_prev(double v, int lane) { return __shfl_sync(SNAP_FULL, v, (lane + 31) & 31); }
__device__ __forceinline__ double shfl_next(double v, int lane) { return __shfl_sync(SNAP_FULL, v, (lane + 1) & 31); }

// ------------------------------------------------------------------------------------------------
// per-warp row pipeline: ring of `nst` stages x 2 input rows + 4 output rows, padded layout
// ------------------------------------------------------------------------------------------------
template <int Q>
struct RowPipe {
  using G = RowGeom<Q>;
  double* stage;   // [nst][2][RP]
  double* orow;    // [4][RP]
  uint32_t bar0, phase;
  int nst, lane;
  long long rows_rd, rows_wr;   // HBM rows requested (lane 0 counts): the traffic this variant needs

  __device__ __forceinline__ double* row(int s, int r) const { return stage + (size_t)(s * 2 + r) * G::RP; }
  __device__ __forceinline__ double* out(int r) const { return orow + (size_t)r * G::RP; }

  // every lane has finished reading stage s; load one or two global rows into it
  __device__ __forceinline__ void issue(int s, const double* g0, const double* g1) {
    __syncwarp();
    const uint32_t bar = bar0 + 8u * s;
    if (lane == 0) {
      mbar_expect_tx(bar, (uint32_t)G::NX * 8u * (g1 ? 2u : 1u));
      rows_rd += g1 ? 2 : 1;
    }
    __syncwarp();
    if (lane < G::SEGS) {
      bulk_g2s(smem_u32(row(s, 0) + 18 * lane), g0 + 16 * lane, 128u, bar);
      if (g1) bulk_g2s(smem_u32(row(s, 1) + 18 * lane), g1 + 16 * lane, 128u, bar);
    }
  }
  __device__ __forceinline__ void wait(int s) {
    mbar_wait(bar0 + 8u * s, (phase >> s) & 1u);
    phase ^= (1u << s);
  }
  // the output rows written two levels ago have been read by the bulk-store engine
  __device__ __forceinline__ void out_ready() {
    if (lane < G::SEGS) bulk_wait_read<1>();
    __syncwarp();
  }
  // lanes have filled output row(s) with generic stores: fence, then hand them to the bulk-store engine
  __device__ __forceinline__ void store_rows(double* g0, const double* s0, double* g1, const double* s1) {
    fence_proxy_async_smem();
    __syncwarp();
    if (lane < G::SEGS) {
      if (g0) bulk_s2g(g0 + 16 * lane, smem_u32(s0 + 18 * lane), 128u);
      if (g1) bulk_s2g(g1 + 16 * lane, smem_u32(s1 + 18 * lane), 128u);
      bulk_commit();
    }
    if (lane == 0) rows_wr += (g0 ? 1 : 0) + (g1 ? 1 : 0);
  }
  // all bulk stores of this warp are complete and visible to later (bulk or generic) loads
  __device__ __forceinline__ void drain() {
    if (lane < G::SEGS) bulk_wait_all<0>();
    fence_proxy_async_all();
    __syncwarp();
  }
};

// warp-uniform sums of one fused pass, index t = iteration within the pass (iterate x_t, step d_t = -q_t)
template <int JT>
struct FusedStats {
  double hinf[JT], h1[JT];   // ||h(x_t)||_inf, ||h(x_t)||_1   (local + mass rows)
  double wd[JT], dd[JT];     // (x_t - u_hat)^T d_t ,  ||d_t||^2
  double f0;                 // 1/2 ||x_0 - u_hat||^2
  bool bad[JT];              // something non-finite in iteration t
};

// ------------------------------------------------------------------------------------------------
// fused forward pass: iterations t = 0 .. T-1 at every level; iterations t < J update the iterate
// (x_{t+1} = x_t - q_t), iteration J (present iff T == J + 1) only emits y = q - (x_J - u_hat) into `yout`
// (the right-hand side of the multiplier solve at x_J).  Reads x_0 (and u_hat if different), writes x_J to
// `xout` when J > 0.
// ------------------------------------------------------------------------------------------------
template <int Q, int JT>
__device__ void fused_fwd(const DevParams& P, RowPipe<Q>& pp, const double* __restrict__ x0,
                          const double* __restrict__ uh, const double* __restrict__ u0, double* __restrict__ xout,
                          double* __restrict__ yout, const int J, const int T, const double M0, FusedStats<JT>& S) {
  constexpr int nx = RowGeom<Q>::NX;
  const int nt = P.nt, lane = pp.lane, nst = pp.nst;
  const double a0 = P.bs_a0, e = P.bs_e, qs = P.bs_qs, hs = P.bs_hs;
  const bool same = (x0 == uh);
  const bool has_mass = P.has_mass != 0;

  double phi[JT][Q], cc[JT][Q];              // Phi(x_t[k-1]) and (A_{k-1} q_{k-1}) of iteration t, own cells
  double hinf[JT], h1[JT], wd[JT], dd[JT];   // per-lane partial sums
  double minf[JT], m1[JT];                   // mass rows (warp-uniform)
  double f2 = 0.0;
  {
    double u0r[Q];
#pragma unroll
    for (int c = 0; c < Q; ++c) u0r[c] = u0[Q * lane + c];
#pragma unroll
    for (int t = 0; t < JT; ++t) {
#pragma unroll
      for (int c = 0; c < Q; ++c) {
        phi[t][c] = u0r[c];   // level 0: h_0 = x[0] - u0
        cc[t][c] = 0.0;
      }
      hinf[t] = 0.0; h1[t] = 0.0; wd[t] = 0.0; dd[t] = 0.0; minf[t] = 0.0; m1[t] = 0.0;
    }
  }
  const int npro = nst < nt ? nst : nt;
  for (int k = 0; k < npro; ++k) pp.issue(k, x0 + (size_t)k * nx, same ? nullptr : uh + (size_t)k * nx);

  int s = 0;
  for (int k = 0; k < nt; ++k) {
    pp.wait(s);
    double v[Q], uhr[Q];
    load_cells<Q>(pp.row(s, 0), lane, v);
    if (same) {
#pragma unroll
      for (int c = 0; c < Q; ++c) uhr[c] = v[c];
    } else {
      load_cells<Q>(pp.row(s, 1), lane, uhr);
    }
    pp.out_ready();
    double* so_u = pp.out(k & 1);
    double* so_y = pp.out(2 + (k & 1));
#pragma unroll
    for (int t = 0; t < JT; ++t) {
      if (t < T) {
        const double vL = shfl_prev(v[Q - 1], lane), vR = shfl_next(v[0], lane);
        double q[Q];
        double msum = 0.0;
#pragma unroll
        for (int c = 0; c < Q; ++c) {
          const double h = v[c] - phi[t][c];
          q[c] = h + cc[t][c];
          const double w = v[c] - uhr[c];
          const double ah = fabs(h);
          hinf[t] = fmax(hinf[t], ah);
          h1[t] += ah;
          wd[t] = fma(w, q[c], wd[t]);
          dd[t] = fma(q[c], q[c], dd[t]);
          if (t == 0) f2 = fma(w, w, f2);
          msum += v[c];
        }
        const double qL = shfl_prev(q[Q - 1], lane), qR = shfl_next(q[0], lane);
#pragma unroll
        for (int c = 0; c < Q; ++c) {
          const double up = (c < Q - 1) ? v[c + 1] : vR, um = (c > 0) ? v[c - 1] : vL;
          const double qr = (c < Q - 1) ? q[c + 1] : qR, ql = (c > 0) ? q[c - 1] : qL;
          phi[t][c] = fma(a0, v[c], (up + um) * fma(-qs, up - um, e));
          cc[t][c] = fma(fma(-hs, up, e), qr, fma(fma(hs, um, e), ql, a0 * q[c]));
        }
        if (has_mass) {
          const double hm = fabs(fma(P.dx, warp_sum(msum), -M0));
          minf[t] = fmax(minf[t], hm);
          m1[t] += hm;
        }
        if (t < J) {
#pragma unroll
          for (int c = 0; c < Q; ++c) v[c] -= q[c];
        } else {
          double yv[Q];
#pragma unroll
          for (int c = 0; c < Q; ++c) yv[c] = q[c] - (v[c] - uhr[c]);
          store_cells<Q>(so_y, lane, yv);
        }
      }
    }
    if (J > 0) store_cells<Q>(so_u, lane, v);
    pp.store_rows(J > 0 ? xout + (size_t)k * nx : nullptr, so_u, T > J ? yout + (size_t)k * nx : nullptr, so_y);
    if (k + nst < nt) pp.issue(s, x0 + (size_t)(k + nst) * nx, same ? nullptr : uh + (size_t)(k + nst) * nx);
    if (++s == nst) s = 0;
  }
  pp.drain();
  f2 = warp_sum(f2);
  S.f0 = 0.5 * f2;
#pragma unroll
  for (int t = 0; t < JT; ++t) {
    if (t < T) {
      double a = warp_max(hinf[t]), b = warp_sum(h1[t]);
      const double c1 = -warp_sum(wd[t]), c2 = warp_sum(dd[t]);
      if (has_mass) { a = fmax(a, minf[t]); b += m1[t]; }
      S.hinf[t] = a; S.h1[t] = b; S.wd[t] = c1; S.dd[t] = c2;
      // fmax drops NaN, the sums do not: a non-finite residual or direction shows up in h1 / dd
      S.bad[t] = !(finite_d(a) && finite_d(b) && finite_d(c1) && finite_d(c2) && finite_d(f2));
    }
  }
}

// ------------------------------------------------------------------------------------------------
// multiplier solve at the final iterate x (a5 backward half):  lam_{nt-1} = y_{nt-1} ,
//     lam_k = y_k + A_k^T lam_{k+1} ,  (A_k^T l)_i = a0 l_i + (e - hs x_i) l_{i-1} + (e + hs x_i) l_{i+1}.
// y is read from `lam`, which is overwritten in place; x is copied to `ucopy` when that is not null.
// sig != nullptr: level sums of lam (input of the min-norm correction).  Returns sum(lam) (finite check).
// ------------------------------------------------------------------------------------------------
template <int Q>
__device__ double fused_bwd(const DevParams& P, RowPipe<Q>& pp, const double* __restrict__ x, double* __restrict__ lam,
                            double* __restrict__ ucopy, double* __restrict__ sig) {
  constexpr int nx = RowGeom<Q>::NX;
  const int nt = P.nt, lane = pp.lane, nst = pp.nst;
  const double a0 = P.bs_a0, e = P.bs_e, hs = P.bs_hs;
  double lo[Q];
#pragma unroll
  for (int c = 0; c < Q; ++c) lo[c] = 0.0;
  double chk = 0.0;
  const int npro = nst < nt ? nst : nt;
  for (int t = 0; t < npro; ++t) {
    const size_t o = (size_t)(nt - 1 - t) * nx;
    pp.issue(t, lam + o, x + o);
  }
  int s = 0;
  for (int t = 0; t < nt; ++t) {
    const int k = nt - 1 - t;
    pp.wait(s);
    double yv[Q], v[Q], l[Q];
    load_cells<Q>(pp.row(s, 0), lane, yv);
    load_cells<Q>(pp.row(s, 1), lane, v);
    pp.out_ready();
    const double lL = shfl_prev(lo[Q - 1], lane), lR = shfl_next(lo[0], lane);
    double lsum = 0.0;
#pragma unroll
    for (int c = 0; c < Q; ++c) {
      const double ll = (c > 0) ? lo[c - 1] : lL, lr = (c < Q - 1) ? lo[c + 1] : lR;
      l[c] = fma(fma(-hs, v[c], e), ll, fma(fma(hs, v[c], e), lr, fma(a0, lo[c], yv[c])));
      lsum += l[c];
    }
#pragma unroll
    for (int c = 0; c < Q; ++c) lo[c] = l[c];
    chk += lsum;
    if (sig) {
      const double sk = warp_sum(lsum);
      if (lane == 0) sig[k] = sk;
    }
    double* so_l = pp.out(t & 1);
    double* so_u = pp.out(2 + (t & 1));
    store_cells<Q>(so_l, lane, l);
    if (ucopy) store_cells<Q>(so_u, lane, v);
    pp.store_rows(lam + (size_t)k * nx, so_l, ucopy ? ucopy + (size_t)k * nx : nullptr, so_u);
    if (t + nst < nt) {
      const size_t o = (size_t)(k - nst) * nx;
      pp.issue(s, lam + o, x + o);
    }
    if (++s == nst) s = 0;
  }
  pp.drain();
  return warp_sum(chk);
}

// Minimum-norm multiplier for the linearly dependent mass rows of kind 4 (streaming
// recipe): with level sums sigma_j of the basic solution (mass multipliers 0) and c = nx dx^2,
//   (D^T D + c I) t = -dx D^T sigma ,  lam_mass[k] = -t_k ,  lam_loc[j][.] += dx sum_{k>=j} t_k
// (D = first difference).  The rank-nt update of lam is one more streaming pass through the row pipe.
template <int Q>
__device__ void fused_min_norm(const DevParams& P, RowPipe<Q>& pp, double* __restrict__ lam, double* __restrict__ sig,
                               double* __restrict__ tt) {
  constexpr int nx = RowGeom<Q>::NX;
  const int nt = P.nt, lane = pp.lane, nst = pp.nst;
  const double c = (double)nx * P.dx * P.dx;
  __syncwarp();
  if (lane == 0) {
    // Thomas on the SPD tridiagonal diag (2+c, ..., 2+c, 1+c), off-diagonals -1
    double cp = 0.0, dp = 0.0;
    for (int k = 0; k < nt; ++k) {
      const double bk = -P.dx * (sig[k] - (k + 1 < nt ? sig[k + 1] : 0.0));
      const double diag = ((k == nt - 1) ? 1.0 : 2.0) + c;
      const double inv = 1.0 / (diag + cp);
      dp = (bk + dp) * inv;
      cp = -inv;
      tt[k] = dp;
      sig[k] = cp;
    }
    double x = tt[nt - 1], suf = x;
    sig[nt - 1] = suf;   // sig now holds the suffix sums of t
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
  const int npro = nst < nt ? nst : nt;
  for (int k = 0; k < npro; ++k) pp.issue(k, lam + (size_t)k * nx, nullptr);
  int s = 0;
  for (int k = 0; k < nt; ++k) {
    pp.wait(s);
    double l[Q];
    load_cells<Q>(pp.row(s, 0), lane, l);
    pp.out_ready();
    const double add = P.dx * sig[k];
#pragma unroll
    for (int cidx = 0; cidx < Q; ++cidx) l[cidx] += add;
    double* so = pp.out(k & 1);
    store_cells<Q>(so, lane, l);
    pp.store_rows(lam + (size_t)k * nx, so, nullptr, nullptr);
    if (k + nst < nt) pp.issue(s, lam + (size_t)(k + nst) * nx, nullptr);
    if (++s == nst) s = 0;
  }
  pp.drain();
}

// ------------------------------------------------------------------------------------------------
// the persistent Gauss-Newton driver (a8, a9)
// ------------------------------------------------------------------------------------------------
template <int Q, int JT>
__global__ void __launch_bounds__(256) project1d_fused_kernel(const __grid_constant__ Proj1dArgs A) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  using G = RowGeom<Q>;
  const DevParams& P = A.P;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int b = blockIdx.x * (blockDim.x >> 5) + warp;
  if (b >= A.batch) return;
  constexpr int nx = G::NX;
  const int nt = P.nt;
  const size_t n = (size_t)P.n;

  unsigned char* base = smem_raw + (size_t)warp * A.warp_bytes;
  RowPipe<Q> pp;
  pp.stage = reinterpret_cast<double*>(base);
  pp.orow = pp.stage + (size_t)A.nst * 2 * G::RP;
  pp.bar0 = smem_u32(pp.orow + (size_t)4 * G::RP);
  pp.phase = 0;
  pp.nst = A.nst; pp.lane = lane;
  pp.rows_rd = 0; pp.rows_wr = 0;
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
#pragma unroll
    for (int c = 0; c < Q; ++c) sm += u0[Q * lane + c];
    M0 = P.dx * warp_sum(sm);
  }
  // iterates ping-pong between two buffers; u_star itself serves as one of them unless it aliases u_hat
  double* const buf0 = bufA;
  double* const buf1 = (ustar != uh) ? ustar : bufB;

  int jcap = (A.fuse > 0 && A.fuse < JT) ? A.fuse : JT;   // updates per pass; drops to 1 after a failed Armijo test
  const double* cur = uh;        // accepted iterate
  double* trial = nullptr;       // pending trial point, awaiting its Armijo test by iteration 0 of the next pass
  bool pend = false;
  int pend_J = 0;                // updates of the pass that produced the pending trial (1: trial = cur + alpha d)
  bool conv = false;             // tol (or max_iter) reached at an accepted iterate: only polish steps remain
  int polish_left = 0, steps = 0, solves = 0, tries = 0, status = 0, sweeps = 0;
  double alpha = 1.0, mu = 0.0, phi_cur = 0.0, Dphi = 0.0;
  const double* xfin = nullptr;  // final iterate; its multiplier right-hand side y has been emitted into lam
  // snapshot of the driver state at the start of the last walked pass (restored when that pass is discarded)
  int steps0 = 0, solves0 = 0, polish0 = 0;
  bool conv0 = false;
  double mu0 = 0.0;
  FusedStats<JT> S;

  while (true) {
    const double* x0 = pend ? trial : cur;
    double* xo = (x0 == buf0) ? buf1 : buf0;
    // ---- plan this pass: J updates, then one y-emitting iteration if it fits (T = J + 1 <= JT) -------------
    int J;
    if (conv) {
      J = polish_left;
    } else if (pend && cur != uh) {
      J = 0;                                  // classic trial evaluation: `cur` lives in the other work buffer
    } else {
      J = jcap;
      if (sweeps > 0 && J > JT - 1) J = JT - 1;
      const int budget = P.max_iter - steps - (pend ? 1 : 0);
      if (J > budget) J = budget;
    }
    if (J > JT - 1 && (sweeps > 0 || conv)) J = JT - 1;
    if (J < 0) J = 0;
    const int T = (J < JT) ? J + 1 : J;
    fused_fwd<Q, JT>(P, pp, x0, uh, u0, xo, lam, J, T, M0, S);
    ++sweeps;

    // ---- a pending step is judged by iteration 0 of this pass ---------------------------------------------
    if (pend) {
      const double phi_t = S.f0 + mu * S.h1[0];
      const bool ok = !S.bad[0] && finite_d(phi_t) && (phi_t <= phi_cur + P.ls_c1 * alpha * Dphi);
      if (!ok) {
        if (pend_J > 1) {   // produced by a fused pass: discard it, redo from its x_0 one iteration per pass
          steps = steps0; solves = solves0; conv = conv0; polish_left = polish0; mu = mu0;
          pend = false; jcap = 1;
          continue;
        }
        if (++tries > P.ls_max) { status = SNAP_ST_LINESEARCH; break; }
        for (size_t i = lane; i < n; i += 32) trial[i] = fma(P.ls_shrink, trial[i] - cur[i], cur[i]);
        __threadfence();
        fence_proxy_async_all();
        __syncwarp();
        alpha *= P.ls_shrink;
        jcap = 1;
        continue;
      }
      ++steps;
      cur = trial;
      pend = false;
    } else if (S.bad[0]) {
      status = SNAP_ST_NONFINITE;   // non-finite residual or direction at an accepted iterate (R16)
      break;
    }

    // ---- walk the pass: x_0 = cur is accepted; judge the steps x_t -> x_{t+1} in order ---------------------
    steps0 = steps; solves0 = solves; conv0 = conv; polish0 = polish_left; mu0 = mu;
    bool discard = false, backtrack = false, fin0 = false, finJ = false;
    double f_t = S.f0;
    for (int t = 0; t < T; ++t) {
      if (!conv) {
        if (S.hinf[t] < P.tol) {
          conv = true;
          polish_left = (S.hinf[t] > kPolishSkip * P.tol) ? P.polish : 0;
        } else if (steps >= P.max_iter) {
          status = SNAP_ST_MAXITER;
          conv = true;
          polish_left = 0;
        }
      }
      if (conv && polish_left == 0) {   // x_t is final; at hand are only x_0 and x_J
        if (t == 0 && J > 0) fin0 = true;                   // final = x_0, y there still to be emitted
        else { finJ = true; solves += (J - t) + 1; }        // final = x_J (t < J: J - t extra polish steps)
        break;
      }
      if (t >= J) break;                // y-emitting iteration at a non-final x_J: y is not used
      if (S.bad[t]) { status = SNAP_ST_NONFINITE; break; }  // non-finite direction at an accepted iterate
      ++solves;
      if (conv) {
        --polish_left;                  // polish step: taken without a test (R4)
      } else {
        mu = merit_mu(mu, S.wd[t], S.dd[t], S.h1[t], kMuRho, kMuFloor);
        phi_cur = f_t + mu * S.h1[t];
        Dphi = S.wd[t] - mu * S.h1[t];
        alpha = 1.0;
        tries = 0;
        if (t + 1 < T) {
          const double phi_t = (f_t + S.wd[t] + 0.5 * S.dd[t]) + mu * S.h1[t + 1];
          const bool ok = !S.bad[t + 1] && finite_d(phi_t) && (phi_t <= phi_cur + P.ls_c1 * Dphi);
          if (!ok) {
            if (t == 0 && J == 1) backtrack = true;   // x_J = x_0 + d_0 is at hand: classic back-tracking
            else discard = true;
            break;
          }
          ++steps;
        } else {
          pend = true;                  // last update of a pass without y iteration: judged by the next pass
          pend_J = J;
        }
      }
      f_t = f_t + S.wd[t] + 0.5 * S.dd[t];
    }
    if (status == SNAP_ST_NONFINITE) break;
    if (discard) {        // an inner Armijo test failed: forget the pass, continue one iteration per pass
      steps = steps0; solves = solves0; conv = conv0; polish_left = polish0; mu = mu0;
      pend = false; jcap = 1;
      if (status == SNAP_ST_MAXITER) status = 0;
      continue;
    }
    if (backtrack) {      // first reduction of the step x_0 -> x_1 (mu, phi_cur, Dphi are those of this step)
      trial = xo;
      if (++tries > P.ls_max) { status = SNAP_ST_LINESEARCH; break; }
      for (size_t i = lane; i < n; i += 32) trial[i] = fma(P.ls_shrink, trial[i] - cur[i], cur[i]);
      __threadfence();
      fence_proxy_async_all();
      __syncwarp();
      alpha = P.ls_shrink;
      pend = true; pend_J = 1; jcap = 1;
      continue;
    }
    if (fin0) {           // e.g. feasible input: return x_0 itself; the speculative updates are dropped
      solves = solves0;
      pend = false;       // conv is set and polish_left == 0: the next pass has J = 0 and only emits y at x_0
      continue;
    }
    if (finJ) {
      if (T > J) { xfin = (J > 0) ? xo : cur; break; }
      cur = xo; pend = false; solves -= 1;          // y at x_J not emitted yet: next pass J = 0
      continue;
    }
    if (J > 0) {
      if (pend) trial = xo;
      else cur = xo;
    }
  }

  long long* stat = A.stats ? A.stats + (size_t)b * 4 : nullptr;
  if (status == SNAP_ST_NONFINITE) {  // R16: u* = u_hat, lam = 0
    if (ustar != uh)
      for (size_t i = lane; i < n; i += 32) ustar[i] = uh[i];
    for (size_t i = lane; i < (size_t)P.m; i += 32) lam[i] = 0.0;
  } else {
    if (status == SNAP_ST_LINESEARCH) {   // multiplier at the last accepted iterate (as the oracle returns it)
      fused_fwd<Q, JT>(P, pp, cur, uh, u0, nullptr, lam, 0, 1, M0, S);
      ++sweeps;
      xfin = cur;
    }
    const bool want_sig = (P.kind == SNAP_BURGERS1D_LF_MASS) && (P.lambda_mode == 0);
    const double chk = fused_bwd<Q>(P, pp, xfin, lam, (xfin != ustar) ? ustar : nullptr, want_sig ? sig : nullptr);
    if (!finite_d(chk)) {
      status = SNAP_ST_NONFINITE;
      __syncwarp();
      for (size_t i = lane; i < n; i += 32) ustar[i] = uh[i];
      for (size_t i = lane; i < (size_t)P.m; i += 32) lam[i] = 0.0;
    } else if (P.has_mass) {
      if (want_sig) fused_min_norm<Q>(P, pp, lam, sig, tt);
      else
        for (int k = lane; k < nt; k += 32) lam[n + k] = 0.0;
    }
  }
  if (lane == 0) {
    A.iters[b] = (status == 0) ? solves : status;
    if (stat) { stat[0] = solves; stat[1] = sweeps; stat[2] = pp.rows_rd; stat[3] = pp.rows_wr; }
  }
}

template <int Q, int JT>
inline int launch_fused_variant(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st) {
  auto kern = project1d_fused_kernel<Q, JT>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem) != cudaSuccess)
    return SNAP_ECUDA;
  kern<<<pl.grid, pl.wpc * 32, pl.smem, st>>>(a);
  return cudaGetLastError() == cudaSuccess ? SNAP_OK : SNAP_ECUDA;
}

}  // namespace snap
