// Burgers family (kinds 1, 4), nx = 32 W Q: fused Gauss-Newton passes, one persistent group of W warps per sample.
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
// Layout: warp w of the group, lane l owns the Q contiguous cells (32 w + l) Q ... + Q - 1; neighbours are
// register-local except at the two ends of a lane (one shuffle each) and of a warp (a shared-memory slot and one
// mbarrier exchange per level, fused_fwd_mw_body; W = 1 needs neither).  A row travels HBM <-> shared memory as ONE tiled TMA
// copy (tensor map [sample][line of 16 doubles][16], box = one row, issued by one elected lane) with the
// 128-byte swizzle, so that the lanes' 128-bit shared-memory accesses to their contiguous cells are
// bank-conflict free: the 16-byte chunk c of line r sits at chunk position c ^ (r & 7).
#pragma once
#include <stdio.h>
#include <stdlib.h>

#include "device_utils.cuh"
#include "launch.h"
#include "snap_internal.h"
#include "tridiag.cuh"

namespace snap {

template <int W, int Q>
struct RowGeom {
  static constexpr int NX = 32 * W * Q;
  static constexpr int LINES = NX / 16;       // 128-byte lines per row
  static constexpr int WLINES = LINES / W;    // lines owned (and stored) by one warp; one TMA box
  static constexpr int RP = (NX < 128 ? 128 : NX);   // row pitch in doubles: rows start 1024-byte aligned
  static constexpr int XCH = 2 * W * 8;       // doubles: exchange slots [parity][warp][8]
  static_assert(W == 1 || WLINES % 8 == 0, "a warp's part of a row must start on a 1024-byte boundary");
};

// cell i of a row lives at this double index of its swizzled shared-memory row (row base 1024-byte aligned)
__device__ __forceinline__ int swz_idx(int i) {
  const int r = i >> 4, c = (i & 15) >> 1;
  return (r << 4) + ((c ^ (r & 7)) << 1) + (i & 1);
}

// per-lane chunk offsets (in doubles) of its Q contiguous cells: Q/2 chunks of 2 doubles inside one line
template <int Q>
struct LaneOff {
  int o[(Q + 1) / 2];
  __device__ __forceinline__ void init(int first) {
#pragma unroll
    for (int c = 0; c < (Q + 1) / 2; ++c) o[c] = swz_idx(first + 2 * c);
  }
};

// Shared-memory rows are addressed in the .shared state space explicitly (LDS / STS): through the generic pointers of
// RowPipe the compiler emitted generic LD.E / ST.E, which resolve the address space per access and are tracked by the
// long scoreboard (profiles/r01d: the top stall of the fused passes).
__device__ __forceinline__ double2 lds_v2(uint32_t a) {
  double2 t;
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(t.x), "=d"(t.y) : "r"(a));
  return t;
}
__device__ __forceinline__ double lds_f64(uint32_t a) {
  double t;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(t) : "r"(a));
  return t;
}
__device__ __forceinline__ void sts_v2(uint32_t a, double x, double y) {
  asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(x), "d"(y) : "memory");
}
__device__ __forceinline__ void sts_f64(uint32_t a, double x) {
  asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(x) : "memory");
}

template <int Q>
__device__ __forceinline__ void load_cells(const double* row, const LaneOff<Q>& lo, double (&x)[Q]) {
  const uint32_t a = smem_u32(row);
  if constexpr (Q == 1) {
    x[0] = lds_f64(a + 8u * lo.o[0]);
  } else {
#pragma unroll
    for (int c = 0; c < Q / 2; ++c) {
      const double2 t = lds_v2(a + 8u * lo.o[c]);
      x[2 * c] = t.x;
      x[2 * c + 1] = t.y;
    }
  }
}
template <int Q>
__device__ __forceinline__ double cell_at(const double* row, const LaneOff<Q>& lo, int c) {
  return lds_f64(smem_u32(row) + 8u * (lo.o[c >> 1] + (c & 1)));
}
template <int Q>
__device__ __forceinline__ void store_cells(double* row, const LaneOff<Q>& lo, const double (&x)[Q]) {
  const uint32_t a = smem_u32(row);
  if constexpr (Q == 1) {
    sts_f64(a + 8u * lo.o[0], x[0]);
  } else {
#pragma unroll
    for (int c = 0; c < Q / 2; ++c) sts_v2(a + 8u * lo.o[c], x[2 * c], x[2 * c + 1]);
  }
}

// a lane's Q contiguous cells straight to global memory (128-bit stores)
template <int Q>
__device__ __forceinline__ void store_cells_global(double* __restrict__ g, const double (&x)[Q]) {
  if constexpr (Q == 1) {
    g[0] = x[0];
  } else {
#pragma unroll
    for (int c = 0; c < Q / 2; ++c) reinterpret_cast<double2*>(g)[c] = make_double2(x[2 * c], x[2 * c + 1]);
  }
}

// a lane's Q contiguous cells from global memory (128-bit loads)
template <int Q>
__device__ __forceinline__ void load_cells_global(const double* __restrict__ g, double (&x)[Q]) {
  if constexpr (Q == 1) {
    x[0] = g[0];
  } else {
#pragma unroll
    for (int c = 0; c < Q / 2; ++c) {
      const double2 t = reinterpret_cast<const double2*>(g)[c];
      x[2 * c] = t.x;
      x[2 * c + 1] = t.y;
    }
  }
}

__device__ __forceinline__ double shfl_prev(double v, int lane) { return __shfl_sync(SNAP_FULL, v, (lane + 31) & 31); }
__device__ __forceinline__ double shfl_next(double v, int lane) { return __shfl_sync(SNAP_FULL, v, (lane + 1) & 31); }

// balanced sum of a lane's Q values (dependency depth log2 Q instead of Q)
template <int Q>
__device__ __forceinline__ double tree_sum(const double (&x)[Q]) {
  if constexpr (Q == 1) return x[0];
  else if constexpr (Q == 2) return x[0] + x[1];
  else if constexpr (Q == 4) return (x[0] + x[1]) + (x[2] + x[3]);
  else if constexpr (Q == 8) return ((x[0] + x[1]) + (x[2] + x[3])) + ((x[4] + x[5]) + (x[6] + x[7]));
  else {
    double a = 0.0, b = 0.0, c = 0.0, d = 0.0;
#pragma unroll
    for (int i = 0; i < Q; i += 4) { a += x[i]; b += x[i + 1]; c += x[i + 2]; d += x[i + 3]; }
    return (a + b) + (c + d);
  }
}

#ifndef SNAP_INLINE_HOT
#define SNAP_INLINE_HOT 1
#endif

// ||h||_inf is only ever compared with two thresholds (tol, kPolishSkip tol).  The passes therefore keep, per lane,
// the maximum of the UPPER 32 bits of |h| (one integer max per cell on the ALU pipe instead of two FP64 compares;
// for non-negative doubles the upper word orders like the value, NaN/Inf sort above everything), and a residual
// counts as below a threshold only if its upper word is below the threshold's upper word.  That is the test
// "||h||_inf < threshold rounded down to 21 significant bits": conservative, it never accepts a residual >= tol.
// Returns 0: below kPolishSkip tol, 1: below tol, 2: not below tol.
__device__ __forceinline__ double hinf_level(int hmx_lane, double tol, double skip) {
  int m = hmx_lane;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(SNAP_FULL, m, o));
  return (m >= __double2hiint(tol)) ? 2.0 : ((m >= __double2hiint(skip)) ? 1.0 : 0.0);
}

constexpr int kMsbPitch = 34;   // doubles per level slot of RowPipe::msb (32 lanes + padding: conflict-free 128-bit reads)
constexpr int kRed = 24;   // doubles per warp in the reduction scratch (>= 4 JT + 1)

// a global buffer of the path: its tensor map (rows as TMA boxes) and the sample's base pointer (generic access)
struct Buf {
  const CUtensorMap* tm;
  double* p;
};

// ------------------------------------------------------------------------------------------------
// per-sample row pipeline shared by the W warps of a group: ring of `nst` stages x 2 input rows,
// 4 output rows, exchange slots, reduction scratch, mbarriers
// ------------------------------------------------------------------------------------------------
template <int W, int Q>
struct RowPipe {
  using G = RowGeom<W, Q>;
  double* stage;   // [nst][2][RP]   (1024-byte aligned)
  double* orow;    // [4][RP]
  double* xch;     // [2][W][8]
  double* red;     // [W][kRed] partial sums of a pass
  double* msb;     // W = 1: [JT][8 levels][kMsbPitch] per-lane cell sums of the iterates (mass rows, reduced every 8 levels)
  double* aux;     // W = 1: min(nt, 512) doubles (suffix sums of the min-norm correction)
  double* mxs;     // W > 1: [2][W][JT][8] level sums of the iterates per warp (mass rows)
  uint32_t bar0, phase;
  uint32_t xbar, xphase;   // W > 1: the group's exchange mbarrier (one arrive per warp and level) and its parity
  int nst, lane, w, bar_id, first, b;   // first = first cell owned by this lane, b = sample index (TMA coordinate)
  LaneOff<Q> lo;
  long long rows_rd, rows_wr;        // HBM rows requested (counted once per group): the traffic this variant needs
  // PCFM step (snap_flow_step): vel_tm != nullptr marks the pass that forms u_hat = u_tau + omt vel on the fly (Eq. 1);
  // unext != nullptr makes the pass that streams the final iterate also write u_0 + taun (u* - u_0) (Eq. 3)
  const CUtensorMap* vel_tm;
  double omt, taun;
  const double* uprior;
  double* unext;

  __device__ __forceinline__ double* row(int s, int r) const { return stage + (size_t)(s * 2 + r) * G::RP; }
  __device__ __forceinline__ double* out(int r) const { return orow + (size_t)r * G::RP; }

  __device__ __forceinline__ void gsync() const {
    if constexpr (W > 1) asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "n"(W * 32) : "memory");
    else __syncwarp();
  }
  // Every warp of the group has finished reading stage s (callers guarantee it through a gsync);
  // one lane of warp 0 loads level k of one or two buffers into it.
  __device__ __forceinline__ void issue(int s, int k, const CUtensorMap* t0, const CUtensorMap* t1) {
    if (w != 0) return;
    __syncwarp();
    if (lane == 0) {
      const uint32_t bar = bar0 + 8u * s;
      mbar_expect_tx(bar, (uint32_t)G::NX * 8u * (t1 ? 2u : 1u));
      rows_rd += t1 ? 2 : 1;
#pragma unroll
      for (int i = 0; i < W; ++i) {
        tma_load_3d(smem_u32(row(s, 0) + i * G::WLINES * 16), t0, 0, k * G::LINES + i * G::WLINES, b, bar);
        if (t1) tma_load_3d(smem_u32(row(s, 1) + i * G::WLINES * 16), t1, 0, k * G::LINES + i * G::WLINES, b, bar);
      }
    }
  }
  __device__ __forceinline__ void wait(int s) {
    mbar_wait(bar0 + 8u * s, (phase >> s) & 1u);
    phase ^= (1u << s);
  }
  // this warp's part of the output rows written two levels ago has been read by the TMA store engine
  __device__ __forceinline__ void out_ready() {
    if (lane == 0) bulk_wait_read<1>();
    __syncwarp();
  }
  // lanes have filled their part of the output row(s) with generic stores: fence, then store that part (level k)
  __device__ __forceinline__ void store_rows(int k, const CUtensorMap* t0, const double* s0, const CUtensorMap* t1,
                                             const double* s1) {
    fence_proxy_async_smem();
    __syncwarp();
    if (lane == 0) {
      const int line = k * G::LINES + w * G::WLINES;
      if (t0) tma_store_3d(t0, 0, line, b, smem_u32(s0 + w * G::WLINES * 16));
      if (t1) tma_store_3d(t1, 0, line, b, smem_u32(s1 + w * G::WLINES * 16));
      bulk_commit();
      rows_wr += (t0 ? 1 : 0) + (t1 ? 1 : 0);
    }
  }
  // all TMA stores of the group are complete and visible to later (TMA or generic) loads
  __device__ __forceinline__ void drain() {
    if (lane == 0) bulk_wait_all<0>();
    __threadfence();           // generic stores to global (direct row stores) are performed ...
    fence_proxy_async_all();   // ... and ordered before the async-proxy (TMA) loads of the next pass
    gsync();
  }
};

// group-uniform sums of one fused pass, index t = iteration within the pass (iterate x_t, step d_t = -q_t)
template <int JT>
struct FusedStats {
  double hlev[JT];           // ||h(x_t)||_inf against the two thresholds: 0: <= kPolishSkip tol, 1: < tol, 2: >= tol
  double h1[JT];             // ||h(x_t)||_1   (local + mass rows)
  double wd[JT], dd[JT];     // (x_t - u_hat)^T d_t ,  ||d_t||^2
  double f0;                 // 1/2 ||x_0 - u_hat||^2
  bool bad[JT];              // something non-finite in iteration t
};

// ------------------------------------------------------------------------------------------------
// fused forward pass, NU updates + (EMIT ? 1 : 0) y-emitting iteration, T = NU + EMIT iterations per level.
// Iteration t < NU:  x_{t+1} = x_t - q_t;  iteration NU (EMIT): y = q - (x_NU - u_hat) -> `yout`, the
// right-hand side of the multiplier solve at x_NU.  Reads x_0 (and u_hat if different), writes x_NU to
// `xout` when NU > 0.
// ------------------------------------------------------------------------------------------------
template <int W, int Q, int JT, int NU, bool EMIT>
__device__ __forceinline__ void fused_fwd_body(const DevParams& P, RowPipe<W, Q>& pp_ref, const Buf x0, const Buf uh,
                                       const double* __restrict__ u0, const Buf xout, const Buf yout, const double M0,
                                       FusedStats<JT>& S) {
  static_assert(W == 1, "one warp per sample (groups of W > 1 warps run fused_fwd_mw_body)");
  using G = RowGeom<W, Q>;
  constexpr int nx = G::NX;
  constexpr int T = NU + (EMIT ? 1 : 0);
  static_assert(T >= 1 && T <= JT, "iterations per pass");
  constexpr bool kFirstPass = (NU == JT && !EMIT);   // this shape is only planned as the first pass: x_0 == u_hat
  RowPipe<W, Q> pp = pp_ref;   // registers; the mutable fields are written back at the end
  const int nt = P.nt, lane = pp.lane, nst = pp.nst, first = pp.first;
  const double a0 = P.bs_a0, e = P.bs_e, qs = P.bs_qs, hs = P.bs_hs;
  const bool same = (x0.p == uh.p);
  const bool has_mass = P.has_mass != 0;
  const bool shoot = (pp.vel_tm != nullptr);   // x0 holds u_tau: this pass forms u_hat (Eq. 1) in place
  const CUtensorMap* const tm_uh = shoot ? pp.vel_tm : (same ? nullptr : uh.tm);

  double phi[T][Q], cc[T][Q];              // Phi(x_t[k-1]) and (A_{k-1} q_{k-1}) of iteration t, own cells
  double h1[T], wd[T], dd[T];              // per-lane partial sums (thread 0 of the group also takes the mass rows)
  int hmx[T];                              // max over the upper 32 bits of |h| (see hinf_level)
  const double tol = P.tol, skip = kPolishSkip * P.tol;
  double f2 = 0.0;
  {
    double u0r[Q];
#pragma unroll
    for (int c = 0; c < Q; ++c) u0r[c] = u0[first + c];
#pragma unroll
    for (int t = 0; t < T; ++t) {
#pragma unroll
      for (int c = 0; c < Q; ++c) {
        phi[t][c] = u0r[c];   // level 0: h_0 = x[0] - u0
        cc[t][c] = 0.0;
      }
      h1[t] = 0.0; wd[t] = 0.0; dd[t] = 0.0; hmx[t] = 0;
    }
  }
  const int npro = nst < nt ? nst : nt;
  for (int k = 0; k < npro; ++k) pp.issue(k, k, x0.tm, tm_uh);

  // W == 1, mass rows: every lane parks the sum of its cells of each iterate in shared memory ([t][k & 7][lane]);
  // after 8 levels the warp reduces the 8 T level sums at once (lane (j, p) adds 8 lanes' entries of level j, two
  // butterfly rounds join the 4 parts).  A butterfly per level and iterate (5 dependent shuffle rounds) was 12 % of
  // the instructions of a pass and sat on its critical path (profiles/r02_project1d_fused.md).
  const double dxm = P.dx;
  const uint32_t msb_a = smem_u32(pp.msb);
  auto mass_rows8 = [&](int nv) {
    __syncwarp();
    const int j = lane & 7, pq = lane >> 3;
#pragma unroll
    for (int t = 0; t < T; ++t) {
      const uint32_t a = msb_a + 8u * (uint32_t)((t * 8 + j) * kMsbPitch + pq * 8);
      const double2 x0 = lds_v2(a), x1 = lds_v2(a + 16u), x2 = lds_v2(a + 32u), x3 = lds_v2(a + 48u);
      double sacc = ((x0.x + x0.y) + (x1.x + x1.y)) + ((x2.x + x2.y) + (x3.x + x3.y));
      sacc += __shfl_xor_sync(SNAP_FULL, sacc, 8);
      sacc += __shfl_xor_sync(SNAP_FULL, sacc, 16);
      const double hm = fabs(fma(dxm, sacc, -M0));
      const bool on = (pq == 0) && (j < nv);
      hmx[t] = max(hmx[t], on ? __double2hiint(hm) : 0);
      h1[t] += on ? hm : 0.0;
    }
    __syncwarp();
  };

  int s = 0;
  for (int k = 0; k < nt; ++k) {
    pp.wait(s);
    double v[Q];
    const double* r0 = pp.row(s, 0);
    const double* ruh = same ? r0 : pp.row(s, 1);   // u_hat cells are re-read where needed
    load_cells<Q>(r0, pp.lo, v);
    if (shoot) {   // u_hat = u_tau + (1 - tau) v_theta: to global (in place over u_tau) and back into the stage row,
                   // which later iterations of this level re-read as the u_hat row
      double vv[Q];
      load_cells<Q>(pp.row(s, 1), pp.lo, vv);
#pragma unroll
      for (int c = 0; c < Q; ++c) v[c] = fma(pp.omt, vv[c], v[c]);
      store_cells<Q>(pp.row(s, 0), pp.lo, v);
      store_cells_global<Q>(uh.p + (size_t)k * nx + first, v);
      if (lane == 0) pp.rows_wr += 1;
    }
    double vL = shfl_prev(v[Q - 1], lane), vR = shfl_next(v[0], lane);
#pragma unroll
    for (int t = 0; t < T; ++t) {
      double q[Q], uhr[Q];
      const double msum = tree_sum<Q>(v);
      if (!(kFirstPass && t == 0)) load_cells<Q>(ruh, pp.lo, uhr);   // 128-bit conflict-free reads; not kept across iterations
#pragma unroll
      for (int c = 0; c < Q; ++c) {
        const double h = v[c] - phi[t][c];
        q[c] = h + cc[t][c];
        const double ah = fabs(h);
        hmx[t] = max(hmx[t], __double2hiint(ah));
        h1[t] += ah;
        dd[t] = fma(q[c], q[c], dd[t]);
        if (!(kFirstPass && t == 0)) {   // the first pass starts at x_0 = u_hat: w = 0 there
          const double wv = v[c] - uhr[c];
          wd[t] = fma(wv, q[c], wd[t]);
          if (t == 0) f2 = fma(wv, wv, f2);
        }
      }
      // The neighbours' end cells of the NEXT iterate need no exchange of their own: the neighbour forms x - q there, and
      // both operands are at hand (vL, qL / vR, qR): the same subtraction on the same values (t + 1 < T implies t < NU).
      const double qL = shfl_prev(q[Q - 1], lane), qR = shfl_next(q[0], lane);
      double vnL = 0.0, vnR = 0.0;
      if (t + 1 < T) { vnL = vL - qL; vnR = vR - qR; }
      if (has_mass) sts_f64(msb_a + 8u * (uint32_t)((t * 8 + (k & 7)) * kMsbPitch + lane), msum);
      // state for the next level (needs the old v and q with neighbours), then the update in place
      double um = vL, ql = qL;
#pragma unroll
      for (int c = 0; c < Q; ++c) {
        const double up = (c < Q - 1) ? v[c + 1] : vR;
        const double qr = (c < Q - 1) ? q[c + 1] : qR;
        const double vc = v[c], qc = q[c];
        phi[t][c] = fma(a0, vc, (up + um) * fma(-qs, up - um, e));
        cc[t][c] = fma(fma(-hs, up, e), qr, fma(fma(hs, um, e), ql, a0 * qc));
        um = vc; ql = qc;
        if (t < NU) v[c] = vc - qc;
        else if (EMIT) q[c] = qc - (vc - uhr[c]);   // y
      }
      if (t < NU) { vL = vnL; vR = vnR; }
      else if (yout.p) store_cells_global<Q>(yout.p + (size_t)k * nx + first, q);
    }
    if (has_mass && ((k & 7) == 7 || k == nt - 1)) mass_rows8((k & 7) + 1);
    // results go straight to global memory (no staging row, no proxy fence)
    if (NU > 0) store_cells_global<Q>(xout.p + (size_t)k * nx + first, v);
    if (lane == 0) pp.rows_wr += (NU > 0 ? 1 : 0) + ((EMIT && yout.p) ? 1 : 0);
    if (k + nst < nt) pp.issue(s, k + nst, x0.tm, tm_uh);   // the warp has read stage s
    if (++s == nst) s = 0;
  }
  pp.drain();
  // ---- reduce: lanes -> warp -> group (fixed order: identical in every warp, run-to-run deterministic) ----
  double part[4 * T + 1];
#pragma unroll
  for (int t = 0; t < T; ++t) {
    part[4 * t + 0] = hinf_level(hmx[t], tol, skip);
    part[4 * t + 1] = warp_sum(h1[t]);
    part[4 * t + 2] = warp_sum(wd[t]);
    part[4 * t + 3] = warp_sum(dd[t]);
  }
  part[4 * T] = warp_sum(f2);
  S.f0 = 0.5 * part[4 * T];
#pragma unroll
  for (int t = 0; t < T; ++t) {
    const double a = part[4 * t + 0], b = part[4 * t + 1];
    const double c1 = -part[4 * t + 2], c2 = part[4 * t + 3];
    S.hlev[t] = a; S.h1[t] = b; S.wd[t] = c1; S.dd[t] = c2;
    // fmax drops NaN, the sums do not: a non-finite residual or direction shows up in h1 / dd
    S.bad[t] = !(finite_d(a) && finite_d(b) && finite_d(c1) && finite_d(c2) && finite_d(part[4 * T]));
  }
  pp_ref.phase = pp.phase; pp_ref.rows_rd = pp.rows_rd; pp_ref.rows_wr = pp.rows_wr;
}

// ------------------------------------------------------------------------------------------------
// W > 1: the same fused pass with ONE exchange per level between the warps of a group.  The in-level chain
// x_t -> h -> q_t -> x_{t+1} is cell-local (it needs Phi and A q of the PREVIOUS level only), so a warp first runs all
// T iterations of the level on its own cells, publishes the end values (x_t, q_t of its first and last cell, every t)
// to a shared-memory slot, arrives on the group's mbarrier, does the work that needs no neighbour (sums, row stores,
// intra-warp shuffles), and only then waits for the other warps' slots and forms Phi / A q for the next level.
// The warps of a group therefore run at most one level apart and never wait inside an iteration (the per-iteration
// named barrier of the first W > 1 mapping cost 2.4x, profiles/r02_project1d_fused.md).  Rows leave through direct
// 128-bit global stores as for W = 1.
// ------------------------------------------------------------------------------------------------
template <int W, int Q, int JT, int NU, bool EMIT>
__device__ __forceinline__ void fused_fwd_mw_body(const DevParams& P, RowPipe<W, Q>& pp_ref, const Buf x0, const Buf uh,
                                                  const double* __restrict__ u0, const Buf xout, const Buf yout,
                                                  const double M0, FusedStats<JT>& S) {
  static_assert(W > 1, "multi-warp groups only");
  using G = RowGeom<W, Q>;
  constexpr int nx = G::NX;
  constexpr int T = NU + (EMIT ? 1 : 0);
  static_assert(T >= 1 && T <= JT, "iterations per pass");
  constexpr bool kFirstPass = (NU == JT && !EMIT);   // only planned as the first pass: x_0 == u_hat
  RowPipe<W, Q> pp = pp_ref;
  const int nt = P.nt, lane = pp.lane, nst = pp.nst, w = pp.w, first = pp.first;
  const double a0 = P.bs_a0, e = P.bs_e, qs = P.bs_qs, hs = P.bs_hs;
  const bool same = (x0.p == uh.p);
  const bool has_mass = P.has_mass != 0;
  const int wl = (w + W - 1) % W, wr = (w + 1) % W;
  const CUtensorMap* const tm_uh = same ? nullptr : uh.tm;

  double phi[T][Q], cc[T][Q];
  double h1[T], wd[T], dd[T];
  int hmx[T];
  const double tol = P.tol, skip = kPolishSkip * P.tol;
  double f2 = 0.0;
  {
    double u0r[Q];
#pragma unroll
    for (int c = 0; c < Q; ++c) u0r[c] = u0[first + c];
#pragma unroll
    for (int t = 0; t < T; ++t) {
#pragma unroll
      for (int c = 0; c < Q; ++c) { phi[t][c] = u0r[c]; cc[t][c] = 0.0; }
      h1[t] = 0.0; wd[t] = 0.0; dd[t] = 0.0; hmx[t] = 0;
    }
  }
  const int npro = nst < nt ? nst : nt;
  for (int k = 0; k < npro; ++k) pp.issue(k, k, x0.tm, tm_uh);

  const double dxm = P.dx;
  const uint32_t msb_a = smem_u32(pp.msb) + 8u * (uint32_t)(w * JT * 8 * kMsbPitch);   // this warp's cell sums
  const uint32_t mxs_a = smem_u32(pp.mxs);                                              // [2][W][JT][8] level sums per warp (buffer (k >> 3) & 1)
  const uint32_t xch_a = smem_u32(pp.xch);                                              // [2][W][JT][4] end values
  // the warp's part of the level sums of the last nv levels -> mxs (before this level's arrive)
  auto mass_part8 = [&](int mb) {
    __syncwarp();
    const int j = lane & 7, pq = lane >> 3;
#pragma unroll
    for (int t = 0; t < T; ++t) {
      const uint32_t a = msb_a + 8u * (uint32_t)((t * 8 + j) * kMsbPitch + pq * 8);
      const double2 y0 = lds_v2(a), y1 = lds_v2(a + 16u), y2 = lds_v2(a + 32u), y3 = lds_v2(a + 48u);
      double sacc = ((y0.x + y0.y) + (y1.x + y1.y)) + ((y2.x + y2.y) + (y3.x + y3.y));
      sacc += __shfl_xor_sync(SNAP_FULL, sacc, 8);
      sacc += __shfl_xor_sync(SNAP_FULL, sacc, 16);
      if (pq == 0) sts_f64(mxs_a + 8u * (uint32_t)(((mb * W + w) * JT + t) * 8 + j), sacc);
    }
  };
  // after the wait: warp 0 joins the W parts (fixed order) and takes the mass rows into its sums
  auto mass_join8 = [&](int mb, int nv) {
    const int j = lane & 7, pq = lane >> 3;
    if (w == 0) {
#pragma unroll
      for (int t = 0; t < T; ++t) {
        double sacc = 0.0;
#pragma unroll
        for (int i = 0; i < W; ++i) sacc += lds_f64(mxs_a + 8u * (uint32_t)(((mb * W + i) * JT + t) * 8 + j));
        const double hm = fabs(fma(dxm, sacc, -M0));
        const bool on = (pq == 0) && (j < nv);
        hmx[t] = max(hmx[t], on ? __double2hiint(hm) : 0);
        h1[t] += on ? hm : 0.0;
      }
    }
  };

  int s = 0;
  uint32_t xph = pp.xphase;
  for (int k = 0; k < nt; ++k) {
    pp.wait(s);
    double vt[T][Q], qt[T][Q], uhr[Q], vfin[Q];
    load_cells<Q>(pp.row(s, 0), pp.lo, vt[0]);
    if (!same) load_cells<Q>(pp.row(s, 1), pp.lo, uhr);
    else {
#pragma unroll
      for (int c = 0; c < Q; ++c) uhr[c] = vt[0][c];
    }
    // ---- the cell-local chain of the level: all T iterations --------------------------------------------
#pragma unroll
    for (int t = 0; t < T; ++t) {
      if (has_mass) sts_f64(msb_a + 8u * (uint32_t)((t * 8 + (k & 7)) * kMsbPitch + lane), tree_sum<Q>(vt[t]));
#pragma unroll
      for (int c = 0; c < Q; ++c) {
        const double v = vt[t][c];
        const double h = v - phi[t][c];
        const double q = h + cc[t][c];
        const double ah = fabs(h);
        hmx[t] = max(hmx[t], __double2hiint(ah));
        h1[t] += ah;
        dd[t] = fma(q, q, dd[t]);
        if (!(kFirstPass && t == 0)) {
          const double wv = v - uhr[c];
          wd[t] = fma(wv, q, wd[t]);
          if (t == 0) f2 = fma(wv, wv, f2);
        }
        qt[t][c] = q;
        if (t < NU) {
          const double vn = v - q;
          if (t + 1 < T) vt[t + 1][c] = vn;
          else vfin[c] = vn;
        }
      }
    }
    // ---- publish the end values, arrive -----------------------------------------------------------------
    {
      const uint32_t xs = xch_a + 8u * (uint32_t)(((k & 1) * W + w) * JT * 4);
      if (lane == 0) {
#pragma unroll
        for (int t = 0; t < T; ++t) { sts_f64(xs + 32u * t, vt[t][0]); sts_f64(xs + 32u * t + 16u, qt[t][0]); }
      }
      if (lane == 31) {
#pragma unroll
        for (int t = 0; t < T; ++t) { sts_f64(xs + 32u * t + 8u, vt[t][Q - 1]); sts_f64(xs + 32u * t + 24u, qt[t][Q - 1]); }
      }
    }
    const bool mass_now = has_mass && ((k & 7) == 7 || k == nt - 1);
    if (mass_now) mass_part8((k >> 3) & 1);
    __syncwarp();
    if (lane == 0) mbar_arrive(pp.xbar);
    // ---- work that needs no other warp ------------------------------------------------------------------
    double vL[T], vR[T], qL[T], qR[T];
#pragma unroll
    for (int t = 0; t < T; ++t) {
      vL[t] = shfl_prev(vt[t][Q - 1], lane); vR[t] = shfl_next(vt[t][0], lane);
      qL[t] = shfl_prev(qt[t][Q - 1], lane); qR[t] = shfl_next(qt[t][0], lane);
    }
    if (NU > 0) {
      if constexpr (EMIT) store_cells_global<Q>(xout.p + (size_t)k * nx + first, vt[T - 1]);
      else store_cells_global<Q>(xout.p + (size_t)k * nx + first, vfin);
    }
    if constexpr (EMIT) {
      if (yout.p) {
        double y[Q];
#pragma unroll
        for (int c = 0; c < Q; ++c) y[c] = qt[T - 1][c] - (vt[T - 1][c] - uhr[c]);
        store_cells_global<Q>(yout.p + (size_t)k * nx + first, y);
      }
    }
    if (w == 0 && lane == 0) pp.rows_wr += (NU > 0 ? 1 : 0) + ((EMIT && yout.p) ? 1 : 0);
    // ---- the other warps' end values --------------------------------------------------------------------
    mbar_wait(pp.xbar, xph);
    xph ^= 1u;
    {
      const uint32_t xl = xch_a + 8u * (uint32_t)(((k & 1) * W + wl) * JT * 4);
      const uint32_t xr = xch_a + 8u * (uint32_t)(((k & 1) * W + wr) * JT * 4);
      if (lane == 0) {
#pragma unroll
        for (int t = 0; t < T; ++t) { vL[t] = lds_f64(xl + 32u * t + 8u); qL[t] = lds_f64(xl + 32u * t + 24u); }
      }
      if (lane == 31) {
#pragma unroll
        for (int t = 0; t < T; ++t) { vR[t] = lds_f64(xr + 32u * t); qR[t] = lds_f64(xr + 32u * t + 16u); }
      }
    }
    if (mass_now) mass_join8((k >> 3) & 1, (k & 7) + 1);
    // every warp of the group has read stage s (its reads precede its arrive): refill it
    if (k + nst < nt) pp.issue(s, k + nst, x0.tm, tm_uh);
    // ---- Phi and A q of this level, the state of the next one -------------------------------------------
#pragma unroll
    for (int t = 0; t < T; ++t) {
#pragma unroll
      for (int c = 0; c < Q; ++c) {
        const double um = (c > 0) ? vt[t][c - 1] : vL[t], up = (c < Q - 1) ? vt[t][c + 1] : vR[t];
        const double ql = (c > 0) ? qt[t][c - 1] : qL[t], qr = (c < Q - 1) ? qt[t][c + 1] : qR[t];
        const double vc = vt[t][c], qc = qt[t][c];
        phi[t][c] = fma(a0, vc, (up + um) * fma(-qs, up - um, e));
        cc[t][c] = fma(fma(-hs, up, e), qr, fma(fma(hs, um, e), ql, a0 * qc));
      }
    }
    if (++s == nst) s = 0;
  }
  pp.xphase = xph;
  pp.drain();
  // ---- reduce: lanes -> warp -> group (fixed order) ----------------------------------------------------------
  double part[4 * T + 1];
#pragma unroll
  for (int t = 0; t < T; ++t) {
    part[4 * t + 0] = hinf_level(hmx[t], tol, skip);
    part[4 * t + 1] = warp_sum(h1[t]);
    part[4 * t + 2] = warp_sum(wd[t]);
    part[4 * t + 3] = warp_sum(dd[t]);
  }
  part[4 * T] = warp_sum(f2);
  if (lane == 0) {
#pragma unroll
    for (int i = 0; i < 4 * T + 1; ++i) pp.red[w * kRed + i] = part[i];
  }
  pp.gsync();
#pragma unroll
  for (int i = 0; i < 4 * T + 1; ++i) {
    double acc = pp.red[i];
#pragma unroll
    for (int ww = 1; ww < W; ++ww) {
      const double o = pp.red[ww * kRed + i];
      acc = ((i & 3) == 0 && i < 4 * T) ? fmax(acc, o) : acc + o;
    }
    part[i] = acc;
  }
  pp.gsync();
  S.f0 = 0.5 * part[4 * T];
#pragma unroll
  for (int t = 0; t < T; ++t) {
    const double a = part[4 * t + 0], b = part[4 * t + 1];
    const double c1 = -part[4 * t + 2], c2 = part[4 * t + 3];
    S.hlev[t] = a; S.h1[t] = b; S.wd[t] = c1; S.dd[t] = c2;
    S.bad[t] = !(finite_d(a) && finite_d(b) && finite_d(c1) && finite_d(c2) && finite_d(part[4 * T]));
  }
  pp_ref.phase = pp.phase; pp_ref.xphase = pp.xphase; pp_ref.rows_rd = pp.rows_rd; pp_ref.rows_wr = pp.rows_wr;
}

// ------------------------------------------------------------------------------------------------
// Fisher-KPP (kind 2, W = 1): the same fused pass with the implicit level operator,
//     q_0 = h_0 ,   T_k q_k = h_k + q_{k-1} ,   T_k = I - dt D Lap_h - dt rho diag(1 - 2 x[k])   (symmetric tridiagonal),
//     h_k = x[k] - x[k-1] - dt (D Lap_h x[k] + rho x[k] (1 - x[k]))   with ghost-cell Neumann ends (R10).
// State per iteration in flight: q_{k-1} and x_t[k-1] of the own cells.  The tridiagonal solve is the warp-level
// partition + cyclic-reduction solver of tridiag.cuh; the level matrix depends on the current level only.
// ------------------------------------------------------------------------------------------------
template <int Q, int JT, int NU, bool EMIT>
__device__ __forceinline__ void fused_fwd_f_body(const DevParams& P, RowPipe<1, Q>& pp_ref, const Buf x0, const Buf uh,
                                         const double* __restrict__ u0, const Buf xout, const Buf yout,
                                         FusedStats<JT>& S) {
  constexpr int T = NU + (EMIT ? 1 : 0);
  static_assert(T >= 1 && T <= JT, "iterations per pass");
  RowPipe<1, Q> pp = pp_ref;
  constexpr int nx = 32 * Q;
  const int nt = P.nt, lane = pp.lane, nst = pp.nst, first = pp.first;
  const double fa = P.fi_a, fr = P.fi_dtrho;
  const bool same = (x0.p == uh.p);
  const bool shoot = (pp.vel_tm != nullptr);   // see fused_fwd_body
  const CUtensorMap* const tm_uh = shoot ? pp.vel_tm : (same ? nullptr : uh.tm);
  const double tol = P.tol, skip = kPolishSkip * P.tol;

  double qo[T][Q], xp[T][Q];   // q_{k-1} and x_t[k-1] of iteration t, own cells
  double h1[T], wd[T], dd[T];
  int hmx[T];
  double f2 = 0.0;
  double u0r[Q];
#pragma unroll
  for (int c = 0; c < Q; ++c) u0r[c] = u0[first + c];
#pragma unroll
  for (int t = 0; t < T; ++t) {
#pragma unroll
    for (int c = 0; c < Q; ++c) { qo[t][c] = 0.0; xp[t][c] = 0.0; }
    h1[t] = 0.0; wd[t] = 0.0; dd[t] = 0.0; hmx[t] = 0;
  }
  const int npro = nst < nt ? nst : nt;
  for (int k = 0; k < npro; ++k) pp.issue(k, k, x0.tm, tm_uh);

  int s = 0;
  for (int k = 0; k < nt; ++k) {
    pp.wait(s);
    double v[Q];
    const double* r0 = pp.row(s, 0);
    const double* ruh = same ? r0 : pp.row(s, 1);
    load_cells<Q>(r0, pp.lo, v);
    if (shoot) {
      double vv[Q];
      load_cells<Q>(pp.row(s, 1), pp.lo, vv);
#pragma unroll
      for (int c = 0; c < Q; ++c) v[c] = fma(pp.omt, vv[c], v[c]);
      store_cells<Q>(pp.row(s, 0), pp.lo, v);
      store_cells_global<Q>(uh.p + (size_t)k * nx + first, v);
      if (lane == 0) pp.rows_wr += 1;
    }
#pragma unroll
    for (int t = 0; t < T; ++t) {
      double q[Q], uhr[Q], hv[Q];
      load_cells<Q>(ruh, pp.lo, uhr);
      if (k == 0) {
#pragma unroll
        for (int c = 0; c < Q; ++c) { hv[c] = v[c] - u0r[c]; q[c] = hv[c]; }
      } else {
        double vL = shfl_prev(v[Q - 1], lane), vR = shfl_next(v[0], lane);
        if (lane == 0) vL = v[0];          // mirrored ghost cells (Neumann)
        if (lane == 31) vR = v[Q - 1];
        double b[Q];
#pragma unroll
        for (int c = 0; c < Q; ++c) {
          const double um = (c > 0) ? v[c - 1] : vL, up = (c < Q - 1) ? v[c + 1] : vR;
          hv[c] = v[c] - xp[t][c] - fa * ((um - v[c]) + (up - v[c])) - fr * v[c] * (1.0 - v[c]);
          q[c] = hv[c] + qo[t][c];
        }
        // T_k = I - dt D Lap_h - dt rho diag(1 - 2 x): off-diagonals -fa, rows fill the warp exactly (nx = 32 Q): the
        // two-scalar form of the warp solve (12 % faster per call on config 3 than the general one: 32 registers less)
        fisher_diag<Q>(fa, fr, v, lane, b);
        warp_tridiag_sym<Q>(-fa, b, q, lane);
      }
#pragma unroll
      for (int c = 0; c < Q; ++c) {
        const double wv = v[c] - uhr[c];
        const double ah = fabs(hv[c]);
        hmx[t] = max(hmx[t], __double2hiint(ah));
        h1[t] += ah;
        wd[t] = fma(wv, q[c], wd[t]);
        dd[t] = fma(q[c], q[c], dd[t]);
        if (t == 0) f2 = fma(wv, wv, f2);
        qo[t][c] = q[c];
        xp[t][c] = v[c];
        if (t < NU) v[c] -= q[c];
        else if (EMIT) q[c] = q[c] - wv;   // y
      }
      if (t >= NU && yout.p) store_cells_global<Q>(yout.p + (size_t)k * nx + first, q);
    }
    if (NU > 0) store_cells_global<Q>(xout.p + (size_t)k * nx + first, v);
    if (lane == 0) pp.rows_wr += (NU > 0 ? 1 : 0) + ((EMIT && yout.p) ? 1 : 0);
    if (k + nst < nt) pp.issue(s, k + nst, x0.tm, tm_uh);
    if (++s == nst) s = 0;
  }
  pp.drain();
  const double f2s = warp_sum(f2);
  S.f0 = 0.5 * f2s;
#pragma unroll
  for (int t = 0; t < T; ++t) {
    const double a = hinf_level(hmx[t], tol, skip);
    const double b = warp_sum(h1[t]), c1 = -warp_sum(wd[t]), c2 = warp_sum(dd[t]);
    S.hlev[t] = a; S.h1[t] = b; S.wd[t] = c1; S.dd[t] = c2;
    S.bad[t] = !(finite_d(b) && finite_d(c1) && finite_d(c2) && finite_d(f2s));
  }
  pp_ref.phase = pp.phase; pp_ref.rows_rd = pp.rows_rd; pp_ref.rows_wr = pp.rows_wr;
}

template <int Q, int JT, int NU, bool EMIT>
__device__ __noinline__ void fused_fwd_f(const DevParams& P, RowPipe<1, Q>& pp_ref, const Buf x0, const Buf uh,
                                         const double* __restrict__ u0, const Buf xout, const Buf yout,
                                         FusedStats<JT>& S) {
  fused_fwd_f_body<Q, JT, NU, EMIT>(P, pp_ref, x0, uh, u0, xout, yout, S);
}

// Fisher multiplier solve at the final iterate:  T_k lam_k = y_k + lam_{k+1} (k >= 1) ,  lam_0 = y_0 + lam_1.
template <int Q>
__device__ __noinline__ double fused_bwd_f(const DevParams& P, RowPipe<1, Q>& pp_ref, const Buf x, const Buf lam,
                                           double* __restrict__ ucopy) {
  RowPipe<1, Q> pp = pp_ref;
  constexpr int nx = 32 * Q;
  const int nt = P.nt, lane = pp.lane, nst = pp.nst, first = pp.first;
  double lo[Q];
#pragma unroll
  for (int c = 0; c < Q; ++c) lo[c] = 0.0;
  double chk = 0.0;
  const int npro = nst < nt ? nst : nt;
  for (int t = 0; t < npro; ++t) pp.issue(t, nt - 1 - t, lam.tm, x.tm);
  // OT pull-back fused into this sweep (Eq. 3): the prior row of the next level travels while this one is computed
  const bool pull = pp.unext != nullptr;
  double upc[Q], upn[Q];
  if (pull) load_cells_global<Q>(pp.uprior + (size_t)(nt - 1) * nx + first, upc);
  int s = 0;
  for (int t = 0; t < nt; ++t) {
    const int k = nt - 1 - t;
    if (pull && k > 0) load_cells_global<Q>(pp.uprior + (size_t)(k - 1) * nx + first, upn);
    pp.wait(s);
    double l[Q], v[Q];
    load_cells<Q>(pp.row(s, 0), pp.lo, l);
    load_cells<Q>(pp.row(s, 1), pp.lo, v);
#pragma unroll
    for (int c = 0; c < Q; ++c) l[c] += lo[c];
    if (k > 0) {
      double b[Q];
      fisher_diag<Q>(P.fi_a, P.fi_dtrho, v, lane, b);
      warp_tridiag_sym<Q>(-P.fi_a, b, l, lane);
    }
#pragma unroll
    for (int c = 0; c < Q; ++c) { lo[c] = l[c]; chk += l[c]; }
    store_cells_global<Q>(lam.p + (size_t)k * nx + first, l);
    if (ucopy) store_cells_global<Q>(ucopy + (size_t)k * nx + first, v);
    if (lane == 0) pp.rows_wr += ucopy ? 2 : 1;
    if (pull) {
#pragma unroll
      for (int c = 0; c < Q; ++c) { upc[c] = fma(pp.taun, v[c] - upc[c], upc[c]); }
      store_cells_global<Q>(pp.unext + (size_t)k * nx + first, upc);
#pragma unroll
      for (int c = 0; c < Q; ++c) upc[c] = upn[c];
      if (lane == 0) { pp.rows_rd += 1; pp.rows_wr += 1; }
    }
    if (t + nst < nt) pp.issue(s, k - nst, lam.tm, x.tm);
    if (++s == nst) s = 0;
  }
  pp.drain();
  pp_ref.phase = pp.phase; pp_ref.rows_rd = pp.rows_rd; pp_ref.rows_wr = pp.rows_wr;
  return warp_sum(chk);
}

// runtime (J, T) -> static instantiation; KIND: KB_FUSED (Burgers family) or KF_FUSED (Fisher, W = 1)
constexpr int KB_FUSED = 1, KF_FUSED = 2;

// out-of-line copy for the rarely used pass shapes; the two shapes every projection runs (JT updates; JT - 1 updates
// + y) are inlined into the kernel so that the grid constants stay constant-bank operands instead of registers
template <int W, int Q, int JT, int NU, bool EMIT>
__device__ __noinline__ void fused_fwd(const DevParams& P, RowPipe<W, Q>& pp_ref, const Buf x0, const Buf uh,
                                       const double* __restrict__ u0, const Buf xout, const Buf yout, const double M0,
                                       FusedStats<JT>& S) {
  if constexpr (W > 1) fused_fwd_mw_body<W, Q, JT, NU, EMIT>(P, pp_ref, x0, uh, u0, xout, yout, M0, S);
  else fused_fwd_body<W, Q, JT, NU, EMIT>(P, pp_ref, x0, uh, u0, xout, yout, M0, S);
}

template <int KIND, int W, int Q, int JT, int NU, bool EMIT>
__device__ __forceinline__ void fused_fwd_kind(const DevParams& P, RowPipe<W, Q>& pp, const Buf x0, const Buf uh,
                                               const double* u0, const Buf xout, const Buf yout, double M0,
                                               FusedStats<JT>& S) {
  if constexpr (KIND == KF_FUSED) {
    if constexpr (SNAP_INLINE_HOT && ((NU == JT && !EMIT) || (NU == JT - 1 && EMIT)))
      fused_fwd_f_body<Q, JT, NU, EMIT>(P, pp, x0, uh, u0, xout, yout, S);
    else fused_fwd_f<Q, JT, NU, EMIT>(P, pp, x0, uh, u0, xout, yout, S);
  }
  else if constexpr (SNAP_INLINE_HOT && W == 1 && ((NU == JT && !EMIT) || (NU == JT - 1 && EMIT)))
    fused_fwd_body<W, Q, JT, NU, EMIT>(P, pp, x0, uh, u0, xout, yout, M0, S);
  else fused_fwd<W, Q, JT, NU, EMIT>(P, pp, x0, uh, u0, xout, yout, M0, S);
}

template <int KIND, int W, int Q, int JT>
__device__ __forceinline__ void fused_fwd_dispatch(const DevParams& P, RowPipe<W, Q>& pp, const Buf x0, const Buf uh,
                                                   const double* u0, const Buf xout, const Buf yout, int J, int T,
                                                   double M0, FusedStats<JT>& S) {
  if (T == J) {   // only the first pass: JT updates, no y
    fused_fwd_kind<KIND, W, Q, JT, JT, false>(P, pp, x0, uh, u0, xout, yout, M0, S);
    return;
  }
  if (J == 0) fused_fwd_kind<KIND, W, Q, JT, 0, true>(P, pp, x0, uh, u0, xout, yout, M0, S);
  else if (J == 1) fused_fwd_kind<KIND, W, Q, JT, 1, true>(P, pp, x0, uh, u0, xout, yout, M0, S);
  else if (J == 2) {
    if constexpr (JT >= 3) fused_fwd_kind<KIND, W, Q, JT, 2, true>(P, pp, x0, uh, u0, xout, yout, M0, S);
  } else if (J == 3) {
    if constexpr (JT >= 4) fused_fwd_kind<KIND, W, Q, JT, 3, true>(P, pp, x0, uh, u0, xout, yout, M0, S);
  }
}

// ------------------------------------------------------------------------------------------------
// multiplier solve at the final iterate x (a5 backward half):  lam_{nt-1} = y_{nt-1} ,
//     lam_k = y_k + A_k^T lam_{k+1} ,  (A_k^T l)_i = a0 l_i + (e - hs x_i) l_{i-1} + (e + hs x_i) l_{i+1}.
// y is read from `lam`, which is overwritten in place; x is copied to `ucopy` when that is not null.
// sig != nullptr: level sums of lam (input of the min-norm correction).  Returns sum(lam) (finite check).
// ------------------------------------------------------------------------------------------------
template <int W, int Q>
__device__ __noinline__ double fused_bwd(const DevParams& P, RowPipe<W, Q>& pp_ref, const Buf x, const Buf lam,
                                         const CUtensorMap* ucopy, double* __restrict__ ucopy_p,
                                         double* __restrict__ sig) {
  using G = RowGeom<W, Q>;
  constexpr int nx = G::NX;
  RowPipe<W, Q> pp = pp_ref;

  const int nt = P.nt, lane = pp.lane, nst = pp.nst, w = pp.w, first = pp.first;
  const double a0 = P.bs_a0, e = P.bs_e, hs = P.bs_hs;
  const int wl = (w + W - 1) % W, wr = (w + 1) % W;
  double lo[Q];
#pragma unroll
  for (int c = 0; c < Q; ++c) lo[c] = 0.0;
  double lL = 0.0, lR = 0.0, chk = 0.0, lsum_prev = 0.0;
  const int npro = nst < nt ? nst : nt;
  for (int t = 0; t < npro; ++t) pp.issue(t, nt - 1 - t, lam.tm, x.tm);
  // OT pull-back fused into this sweep (Eq. 3; W = 1): the prior row of the next level travels while this one is computed
  bool pull = false;
  if constexpr (W == 1) pull = pp.unext != nullptr;
  double upc[Q], upn[Q];
  if (pull) load_cells_global<Q>(pp.uprior + (size_t)(nt - 1) * nx + first, upc);
  int s = 0, par = 0;
  for (int t = 0; t < nt; ++t) {
    const int k = nt - 1 - t;
    if (pull && k > 0) load_cells_global<Q>(pp.uprior + (size_t)(k - 1) * nx + first, upn);
    pp.wait(s);
    double yv[Q], v[Q], l[Q];
    load_cells<Q>(pp.row(s, 0), pp.lo, yv);
    load_cells<Q>(pp.row(s, 1), pp.lo, v);
    if constexpr (W > 1) pp.out_ready();
    if constexpr (W == 1) {   // level sum of the previous step: the butterfly overlaps this level's arithmetic
      if (sig) {
        const double sp = warp_sum(lsum_prev);
        if (lane == 0 && t > 0) sig[k + 1] = sp;
      }
    }
    double lsum = 0.0;
#pragma unroll
    for (int c = 0; c < Q; ++c) {
      const double ll = (c > 0) ? lo[c - 1] : lL, lr = (c < Q - 1) ? lo[c + 1] : lR;
      l[c] = fma(fma(-hs, v[c], e), ll, fma(fma(hs, v[c], e), lr, fma(a0, lo[c], yv[c])));
      lsum += l[c];
    }
#pragma unroll
    for (int c = 0; c < Q; ++c) lo[c] = l[c];
    lL = shfl_prev(l[Q - 1], lane);
    lR = shfl_next(l[0], lane);
    double stot = 0.0;
    if constexpr (W > 1) {
      stot = warp_sum(lsum);
      double* xs = pp.xch + (size_t)par * (W * 8);
      if (lane == 0) { xs[w * 8 + 0] = l[0]; xs[w * 8 + 4] = stot; }
      if (lane == 31) xs[w * 8 + 1] = l[Q - 1];
      pp.gsync();
      if (lane == 0) lL = xs[wl * 8 + 1];
      if (lane == 31) lR = xs[wr * 8 + 0];
      stot = 0.0;
#pragma unroll
      for (int i = 0; i < W; ++i) stot += xs[i * 8 + 4];
      par ^= 1;
      chk += stot;
      if (sig && w == 0 && lane == 0) sig[k] = stot;
    } else {
      chk += lsum;
      lsum_prev = lsum;
    }
    if constexpr (W == 1) {   // straight to global memory (see fused_fwd)
      store_cells_global<Q>(lam.p + (size_t)k * nx + first, l);
      if (ucopy_p) store_cells_global<Q>(ucopy_p + (size_t)k * nx + first, v);
      if (lane == 0) pp.rows_wr += ucopy_p ? 2 : 1;
      if (pull) {
#pragma unroll
        for (int c = 0; c < Q; ++c) upc[c] = fma(pp.taun, v[c] - upc[c], upc[c]);
        store_cells_global<Q>(pp.unext + (size_t)k * nx + first, upc);
#pragma unroll
        for (int c = 0; c < Q; ++c) upc[c] = upn[c];
        if (lane == 0) { pp.rows_rd += 1; pp.rows_wr += 1; }
      }
    } else {
      double* so_l = pp.out(t & 1);
      double* so_u = pp.out(2 + (t & 1));
      store_cells<Q>(so_l, pp.lo, l);
      if (ucopy) store_cells<Q>(so_u, pp.lo, v);
      pp.store_rows(k, lam.tm, so_l, ucopy, so_u);
    }
    if (t + nst < nt) pp.issue(s, k - nst, lam.tm, x.tm);
    if (++s == nst) s = 0;
  }
  if constexpr (W == 1) {
    if (sig) {
      const double sp = warp_sum(lsum_prev);
      if (lane == 0) sig[0] = sp;
    }
  }
  pp.drain();
  pp_ref.phase = pp.phase; pp_ref.rows_rd = pp.rows_rd; pp_ref.rows_wr = pp.rows_wr;
  return (W > 1) ? chk : warp_sum(chk);
}

// W = 1 version of the min-norm correction below.  The nt x nt SPD tridiagonal system is solved by the whole warp
// (QT contiguous rows per lane, partition + cyclic reduction, tridiag.cuh) instead of one lane running Thomas, the
// suffix sums go to shared memory, and the rank-nt update lam_loc[j][.] += dx S_j is a plain coalesced
// read-add-write stream (it is elementwise, so it needs neither the lane-contiguous layout nor TMA staging).
template <int QT>
__device__ __forceinline__ void min_norm_coeffs(const DevParams& P, int lane, const double* __restrict__ sig,
                                                double* __restrict__ ssuf, double* __restrict__ lmass) {
  const int nt = P.nt;
  const double cdiag = (double)P.nx * P.dx * P.dx;
  double a[QT], b[QT], c[QT], d[QT];
#pragma unroll
  for (int j = 0; j < QT; ++j) {
    const int r = lane * QT + j;
    const bool valid = r < nt;
    const double s0 = valid ? sig[r] : 0.0, s1 = (r + 1 < nt) ? sig[r + 1] : 0.0;
    a[j] = (valid && r > 0) ? -1.0 : 0.0;
    c[j] = (r + 1 < nt) ? -1.0 : 0.0;
    b[j] = valid ? ((r == nt - 1) ? 1.0 : 2.0) + cdiag : 1.0;
    d[j] = valid ? -P.dx * (s0 - s1) : 0.0;
  }
  warp_tridiag<QT>(a, b, c, d, lane);   // d = t
  // suffix sums S_r = sum_{k >= r} t_k : inside the lane, then over the lanes above
  double suf[QT];
  double run = 0.0;
#pragma unroll
  for (int j = QT - 1; j >= 0; --j) { run += d[j]; suf[j] = run; }
  double incl = run;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const double v = __shfl_down_sync(SNAP_FULL, incl, o);
    if (lane + o < 32) incl += v;
  }
  const double above = incl - run;
#pragma unroll
  for (int j = 0; j < QT; ++j) {
    const int r = lane * QT + j;
    if (r < nt) { ssuf[r] = suf[j] + above; lmass[r] = -d[j]; }
  }
}

template <int Q>
__device__ __noinline__ void fused_min_norm_w1(const DevParams& P, RowPipe<1, Q>& pp_ref, const Buf lamb,
                                               const double* __restrict__ sig) {
  constexpr int nx = 32 * Q;
  RowPipe<1, Q>& pp = pp_ref;
  const int nt = P.nt, lane = pp.lane;
  double* ssuf = pp.aux;
  double* lmass = lamb.p + (size_t)nt * nx;
  __syncwarp();
  if (nt <= 32) min_norm_coeffs<1>(P, lane, sig, ssuf, lmass);
  else if (nt <= 64) min_norm_coeffs<2>(P, lane, sig, ssuf, lmass);
  else if (nt <= 128) min_norm_coeffs<4>(P, lane, sig, ssuf, lmass);
  else if (nt <= 256) min_norm_coeffs<8>(P, lane, sig, ssuf, lmass);
  else min_norm_coeffs<16>(P, lane, sig, ssuf, lmass);
  __syncwarp();
  // lam_loc[k][.] += dx S_k, four levels in flight per lane
  constexpr int V = (nx >= 64) ? nx / 64 : 1;   // double2 per lane and level (nx = 32: lanes 16..31 idle)
  const double dxm = P.dx;
  double2* base = reinterpret_cast<double2*>(lamb.p);
  const bool act = (nx >= 64) || lane < 16;
  int k = 0;
  for (; k + 4 <= nt; k += 4) {
    double2 x[4][V];
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int j = 0; j < V; ++j)
        if (act) x[u][j] = base[(size_t)(k + u) * (nx / 2) + lane + 32 * j];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const double add = dxm * ssuf[k + u];
#pragma unroll
      for (int j = 0; j < V; ++j)
        if (act) base[(size_t)(k + u) * (nx / 2) + lane + 32 * j] = make_double2(x[u][j].x + add, x[u][j].y + add);
    }
  }
  for (; k < nt; ++k) {
    const double add = dxm * ssuf[k];
#pragma unroll
    for (int j = 0; j < V; ++j)
      if (act) {
        double2 x = base[(size_t)k * (nx / 2) + lane + 32 * j];
        base[(size_t)k * (nx / 2) + lane + 32 * j] = make_double2(x.x + add, x.y + add);
      }
  }
  if (lane == 0) { pp.rows_rd += nt; pp.rows_wr += nt; }
  __threadfence();
  __syncwarp();
}

// Minimum-norm multiplier for the linearly dependent mass rows of kind 4 (streaming
// recipe): with level sums sigma_j of the basic solution (mass multipliers 0) and c = nx dx^2,
//   (D^T D + c I) t = -dx D^T sigma ,  lam_mass[k] = -t_k ,  lam_loc[j][.] += dx sum_{k>=j} t_k
// (D = first difference).  The rank-nt update of lam is one more streaming pass through the row pipe.
template <int W, int Q>
__device__ __noinline__ void fused_min_norm(const DevParams& P, RowPipe<W, Q>& pp_ref, const Buf lamb,
                                            double* __restrict__ sig, double* __restrict__ tt) {
  using G = RowGeom<W, Q>;
  RowPipe<W, Q> pp = pp_ref;
  constexpr int nx = G::NX;
  const int nt = P.nt, lane = pp.lane, nst = pp.nst, first = pp.first;
  const double c = (double)nx * P.dx * P.dx;
  __threadfence_block();
  pp.gsync();
  if (pp.w == 0 && lane == 0) {
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
    __threadfence_block();
  }
  pp.gsync();
  double* lmass = lamb.p + (size_t)nt * nx;
  for (int k = pp.w * 32 + lane; k < nt; k += W * 32) lmass[k] = -tt[k];
  const int npro = nst < nt ? nst : nt;
  for (int k = 0; k < npro; ++k) pp.issue(k, k, lamb.tm, nullptr);
  int s = 0;
  for (int k = 0; k < nt; ++k) {
    pp.wait(s);
    double l[Q];
    load_cells<Q>(pp.row(s, 0), pp.lo, l);
    if constexpr (W > 1) pp.out_ready();
    const double add = P.dx * sig[k];
#pragma unroll
    for (int cidx = 0; cidx < Q; ++cidx) l[cidx] += add;
    if constexpr (W == 1) {
      store_cells_global<Q>(lamb.p + (size_t)k * nx + first, l);
      if (lane == 0) pp.rows_wr += 1;
    } else {
      double* so = pp.out(k & 1);
      store_cells<Q>(so, pp.lo, l);
      pp.store_rows(k, lamb.tm, so, nullptr, nullptr);
    }
    if constexpr (W > 1) pp.gsync();   // every warp has read stage s
    if (k + nst < nt) pp.issue(s, k + nst, lamb.tm, nullptr);
    if (++s == nst) s = 0;
  }
  pp.drain();
  pp_ref.phase = pp.phase; pp_ref.rows_rd = pp.rows_rd; pp_ref.rows_wr = pp.rows_wr;
}

// Streaming epilogue of a group of GT threads over one sample (n doubles, n % 2 == 0, 16-byte aligned rows):
//   ucopy != nullptr:  ucopy = x ;   unext != nullptr:  unext = uprior + taun (x - uprior)     (Eq. 3)
// 128-bit accesses, kU independent iterations in flight per thread (a scalar loop of one warp is latency-bound).
template <int GT>
__device__ __forceinline__ void stream_epilogue(int gtid, size_t n, const double* __restrict__ x, double* __restrict__ ucopy,
                                                const double* __restrict__ uprior, double* __restrict__ unext, double taun) {
  constexpr int kU = 8;
  const size_t n2 = n >> 1;
  const double2* x2 = reinterpret_cast<const double2*>(x);
  const double2* p2 = reinterpret_cast<const double2*>(uprior);
  double2* c2 = reinterpret_cast<double2*>(ucopy);
  double2* o2 = reinterpret_cast<double2*>(unext);
  size_t i = gtid;
  for (; i + (size_t)(kU - 1) * GT < n2; i += (size_t)kU * GT) {
    double2 xv[kU], pv[kU];
#pragma unroll
    for (int u = 0; u < kU; ++u) xv[u] = x2[i + (size_t)u * GT];
    if (unext) {
#pragma unroll
      for (int u = 0; u < kU; ++u) pv[u] = p2[i + (size_t)u * GT];
    }
#pragma unroll
    for (int u = 0; u < kU; ++u) {
      if (ucopy) c2[i + (size_t)u * GT] = xv[u];
      if (unext)
        o2[i + (size_t)u * GT] = make_double2(fma(taun, xv[u].x - pv[u].x, pv[u].x), fma(taun, xv[u].y - pv[u].y, pv[u].y));
    }
  }
  for (; i < n2; i += GT) {
    const double2 xv = x2[i];
    if (ucopy) c2[i] = xv;
    if (unext) {
      const double2 pv = p2[i];
      o2[i] = make_double2(fma(taun, xv.x - pv.x, pv.x), fma(taun, xv.y - pv.y, pv.y));
    }
  }
}

// ------------------------------------------------------------------------------------------------
// the persistent Gauss-Newton driver (a8, a9); every warp of a group runs it with identical values
// ------------------------------------------------------------------------------------------------
template <int KIND, int W, int Q, int JT, int MAXT>
__global__ void __launch_bounds__(MAXT) project1d_fused_kernel(const __grid_constant__ Proj1dArgs A) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  using G = RowGeom<W, Q>;
  const DevParams& P = A.P;
  const int gwarp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int slot = gwarp / W, w = gwarp % W;
  const int b = blockIdx.x * (blockDim.x / (32 * W)) + slot;
  if (b >= A.batch) return;   // whole groups leave together: the named barriers of the others are unaffected
  constexpr int nx = G::NX;
  const int nt = P.nt;
  const size_t n = (size_t)P.n;
  const int gtid = w * 32 + lane;
  constexpr int GT = W * 32;

  // swizzled rows need 1024-byte aligned bases: align the CTA's window, per-sample strides are multiples of 1024
  unsigned char* base = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u) + (size_t)slot * A.warp_bytes;
  RowPipe<W, Q> pp;
  pp.stage = reinterpret_cast<double*>(base);
  pp.orow = pp.stage + (size_t)A.nst * 2 * G::RP;           // output staging rows: only W > 1 uses them
  pp.xch = pp.orow + (size_t)(W > 1 ? 4 : 0) * G::RP;
  pp.red = pp.xch + fused_xch_doubles(W, JT);
  pp.msb = pp.red + W * kRed;
  pp.aux = pp.msb + W * JT * 8 * kMsbPitch;
  pp.mxs = pp.aux + (W == 1 ? (nt < 512 ? nt : 512) : 0);
  pp.bar0 = smem_u32(pp.mxs + (W > 1 ? 2 * W * JT * 8 : 0));
  pp.xbar = pp.bar0 + 8u * A.nst;
  pp.phase = 0; pp.xphase = 0;
  pp.nst = A.nst; pp.lane = lane; pp.w = w; pp.bar_id = 1 + slot;
  pp.first = (w * 32 + lane) * Q;
  pp.b = b;
  pp.lo.init(pp.first);
  pp.rows_rd = 0; pp.rows_wr = 0;
  pp.vel_tm = nullptr; pp.omt = A.omt; pp.taun = A.taun;
  pp.uprior = nullptr; pp.unext = nullptr;    // armed below, around the pass that streams the final iterate
  if (gtid == 0) {
    for (int s = 0; s < A.nst; ++s) mbar_init(pp.bar0 + 8u * s, 1);
    if (W > 1) mbar_init(pp.xbar, W);
    mbar_fence_init();
    fence_proxy_async_smem();
  }
  pp.gsync();

  const double* uh = A.u_hat + (size_t)b * n;
  const double* u0 = A.cdata + (size_t)b * nx;
  double* ustar = A.u_star + (size_t)b * n;
  double* lam = A.lam ? A.lam + (size_t)b * P.m : nullptr;   // nullptr: multiplier-free call (include/snap.h)
  double* bufA = A.bufA + (size_t)b * n;
  double* bufB = A.bufB + (size_t)b * n;
  double* sig = A.aux + (size_t)b * 2 * nt;
  double* tt = sig + nt;
  // sample base pointer -> (tensor map, pointer); u_star may alias u_hat (same map contents)
  auto mk = [&](const double* q) -> Buf {
    const CUtensorMap* t = nullptr;
    if (q == uh) t = &A.tm[TM_UHAT];
    else if (q == bufA) t = &A.tm[TM_BUFA];
    else if (q == bufB) t = &A.tm[TM_BUFB];
    else if (q == ustar) t = &A.tm[TM_USTAR];
    else if (q == lam) t = &A.tm[TM_LAM];
    return Buf{t, const_cast<double*>(q)};
  };

  double M0 = 0.0;
  if (P.has_mass) {   // every warp sums the whole u0 row in the same order: identical M0 in the group
    double sm = 0.0;
    for (int i = lane; i < nx; i += 32) sm += u0[i];
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
  int polish_left = 0, steps = 0, solves = 0, tries = 0, status = 0, sweeps = 0, nback = 0;
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
      const int budget = P.max_iter - steps - (pend ? 1 : 0);
      if (J > budget) J = budget;
    }
    if (J > JT - 1 && (sweeps > 0 || conv || jcap < JT || x0 != uh)) J = JT - 1;   // the JT-update shape assumes x_0 == u_hat
    if (J < 0) J = 0;
    const int T = (J < JT) ? J + 1 : J;
    if (A.vel && sweeps == 0) pp.vel_tm = &A.tm[TM_VEL];   // PCFM step: the first pass reads u_tau and forms u_hat (Eq. 1)
    fused_fwd_dispatch<KIND, W, Q, JT>(P, pp, mk(x0), mk(uh), u0, mk(xo), mk(lam), J, T, M0, S);
    pp.vel_tm = nullptr;
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
        for (size_t i = gtid; i < n; i += GT) trial[i] = fma(P.ls_shrink, trial[i] - cur[i], cur[i]);
        __threadfence();
        fence_proxy_async_all();
        pp.gsync();
        alpha *= P.ls_shrink;
        ++nback;
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
        if (S.hlev[t] < 2.0) {              // ||h(x_t)||_inf < tol
          conv = true;
          polish_left = (S.hlev[t] > 0.0) ? P.polish : 0;   // polish unless already <= kPolishSkip tol
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
      for (size_t i = gtid; i < n; i += GT) trial[i] = fma(P.ls_shrink, trial[i] - cur[i], cur[i]);
      __threadfence();
      fence_proxy_async_all();
      pp.gsync();
      alpha = P.ls_shrink;
      ++nback;
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

  long long* stat = A.stats ? A.stats + (size_t)b * SNAP_STAT_COUNT : nullptr;
  const double* const up_b = A.u_next ? A.u_prior + (size_t)b * n : nullptr;   // PCFM pull-back (Eq. 3) wanted
  double* const un_b = A.u_next ? A.u_next + (size_t)b * n : nullptr;
  bool pulled = false;
  if (status == SNAP_ST_NONFINITE) {  // R16: u* = u_hat, lam = 0
    if (ustar != uh)
      for (size_t i = gtid; i < n; i += GT) ustar[i] = uh[i];
    if (lam)
      for (size_t i = gtid; i < (size_t)P.m; i += GT) lam[i] = 0.0;
  } else if (!lam) {
    // multiplier-free call: no y emission, no multiplier sweep, no min-norm correction; u* = the final iterate
    const double* xf = (status == SNAP_ST_LINESEARCH) ? cur : xfin;
    if (un_b) {          // one stream: u* (if it is not in place already) and the pull-back
      stream_epilogue<GT>(gtid, n, xf, xf != ustar ? ustar : nullptr, up_b, un_b, A.taun);
      pulled = true;
      if (gtid == 0) { pp.rows_rd += 2 * nt; pp.rows_wr += nt + (xf != ustar ? nt : 0); }
    } else if (xf != ustar) {
      stream_epilogue<GT>(gtid, n, xf, ustar, nullptr, nullptr, 0.0);
      if (gtid == 0) { pp.rows_rd += nt; pp.rows_wr += nt; }
    }
  } else {
    if (status == SNAP_ST_LINESEARCH) {   // multiplier at the last accepted iterate (as the oracle returns it)
      fused_fwd_dispatch<KIND, W, Q, JT>(P, pp, mk(cur), mk(uh), u0, Buf{nullptr, nullptr}, mk(lam), 0, 1, M0, S);
      ++sweeps;
      xfin = cur;
    }
    const bool want_sig = (P.kind == SNAP_BURGERS1D_LF_MASS) && (P.lambda_mode == 0);
    // in place (u_star aliases u_hat) the final iterate is copied out only after the multiplier sweep proved finite:
    // status -3 must leave u* = u_hat (include/snap.h)
    const bool late_copy = (ustar == uh) && (xfin != ustar);
    const CUtensorMap* const tm_copy = (xfin != ustar && !late_copy) ? &A.tm[TM_USTAR] : nullptr;
    double chk;
    if (un_b && W == 1 && !late_copy && status == 0) { pp.uprior = up_b; pp.unext = un_b; pulled = true; }
    if constexpr (KIND == KF_FUSED) chk = fused_bwd_f<Q>(P, pp, mk(xfin), mk(lam), tm_copy ? ustar : nullptr);
    else chk = fused_bwd<W, Q>(P, pp, mk(xfin), mk(lam), tm_copy, tm_copy ? ustar : nullptr, want_sig ? sig : nullptr);
    pp.uprior = nullptr; pp.unext = nullptr;
    ++sweeps;
    if (finite_d(chk) && late_copy) {
      for (size_t i = gtid; i < n; i += GT) ustar[i] = xfin[i];
      if (gtid == 0) { pp.rows_rd += nt; pp.rows_wr += nt; }
    }
    if (!finite_d(chk)) {
      status = SNAP_ST_NONFINITE;
      pulled = false;
      pp.gsync();
      if (ustar != uh)
        for (size_t i = gtid; i < n; i += GT) ustar[i] = uh[i];
      for (size_t i = gtid; i < (size_t)P.m; i += GT) lam[i] = 0.0;
    } else if (P.has_mass) {
      if (want_sig) {
        if constexpr (KIND == KB_FUSED) {
          if constexpr (W == 1) {
            if (nt <= 512) fused_min_norm_w1<Q>(P, pp, mk(lam), sig);
            else fused_min_norm<W, Q>(P, pp, mk(lam), sig, tt);
          } else {
            fused_min_norm<W, Q>(P, pp, mk(lam), sig, tt);
          }
        }
        ++sweeps;
      } else {
        for (int k = gtid; k < nt; k += GT) lam[n + k] = 0.0;
      }
    }
  }
  if (un_b && !pulled) {   // pull-back of whatever u* holds (statuses that did not stream the final iterate)
    pp.gsync();
    __threadfence_block();
    stream_epilogue<GT>(gtid, n, ustar, nullptr, up_b, un_b, A.taun);
    if (gtid == 0) { pp.rows_rd += 2 * nt; pp.rows_wr += nt; }
  }
  if (gtid == 0) {
    A.iters[b] = (status == 0) ? solves : status;
    if (stat) {
      stat[SNAP_STAT_LINEARISATIONS] = solves; stat[SNAP_STAT_PASSES] = sweeps;
      stat[SNAP_STAT_ROWS_READ] = pp.rows_rd; stat[SNAP_STAT_ROWS_WRITTEN] = pp.rows_wr;
      stat[SNAP_STAT_VARIANT] = A.variant; stat[SNAP_STAT_INNER] = 0; stat[SNAP_STAT_ROW_DOUBLES] = nx;
      stat[SNAP_STAT_BACKTRACKS] = nback;
    }
  }
}

template <int KIND, int W, int Q, int JT, int MAXT>
inline int launch_fused_variant(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st) {
  auto kern = project1d_fused_kernel<KIND, W, Q, JT, MAXT>;
  if (pl.wpc * W * 32 > MAXT) return SNAP_EINVAL;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem) != cudaSuccess)
    return SNAP_ECUDA;
  kern<<<pl.grid, pl.wpc * W * 32, pl.smem, st>>>(a);
  const cudaError_t err = cudaGetLastError();
  if (err != cudaSuccess && getenv("SNAP_DEBUG")) {
    cudaFuncAttributes fa;
    cudaFuncGetAttributes(&fa, kern);
    fprintf(stderr, "snap: fused<%d,%d,%d,%d,%d> launch failed: %s; grid %d block %d smem %zu; regs %d maxThreads %d local %zu\n",
            KIND, W, Q, JT, MAXT, cudaGetErrorString(err), pl.grid, pl.wpc * W * 32, pl.smem, fa.numRegs, fa.maxThreadsPerBlock,
            fa.localSizeBytes);
  }
  return err == cudaSuccess ? SNAP_OK : SNAP_ECUDA;
}

}  // namespace snap
