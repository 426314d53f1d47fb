// 2D kind (Allen-Cahn, implicit Euler, 5-point periodic), product-form path ("making
// Tt^{-1} exact ... turns M into S"): J_loc is square and block lower-bidiagonal in time (diagonal blocks
// T_k = I - ax dxx - ay dyy + dt diag(3 u_k^2 - 1), sub-diagonal blocks -I), so J J^T is its own block Cholesky
// factorisation and the Schur solve is a forward sweep  T_k q_k = h_k + q_{k-1}  and a backward sweep
// T_k lam_k = y_k + lam_{k+1}.  The level systems (nx ny <= 4096 unknowns, strictly diagonally
// dominant M-matrices) are solved ON CHIP: the level lives in shared memory in two colour planes and is relaxed
// by red-black Gauss-Seidel, whose error contracts by rho^2 per full sweep in the max norm, rho =
// (2ax+2ay)/(1+2ax+2ay-dt) (0.039 on config 4: six sweeps reach fp64 rounding).  One persistent CTA per sample
// runs the whole Gauss-Newton loop; because J^T lam+ = y the step needs only the forward half (u+ = u - q,
// q = J^-1 h), the multiplier sweep runs once at the final point (as in kernels_1d_fused.cuh).
//
// Mapping: thread (pj, pi) owns the PR x 4 patch of cells rows PR pj .., columns 4 pi ..; its own values stay in
// registers across the sweeps, only the patch halo travels through shared memory.  Colour of cell (j, i) is
// (i + j) & 1; plane c stores the cells of colour c of row j contiguously ([ny][nx/2]), so the halo above/below a
// patch is one 128-bit load per colour and the updated cells of a patch row are one 128-bit store.
// Level rows arrive by one bulk (TMA) copy per field into a two-stage mbarrier ring, issued one level ahead.
#pragma once
#include <stdlib.h>

#include "device_utils.cuh"
#include "launch.h"
#include "snap_internal.h"

namespace snap {

struct Dir2dArgs {
  DevParams P;
  int batch;
  const double* u_hat;
  const double* cdata;
  double* u_star;
  double* lam;
  int* iters;
  double* ws;        // [batch][kPcgVectors][n]; vectors 0..2 are the iterate / trial buffers
  long long* stats;  // [batch][SNAP_STAT_COUNT]
  // PCFM step fused around the projection (snap_flow_step; Eq. 1, 3): null / 0 for a plain projection
  const double* vel;      // [batch][n]: the first pass forms u_hat = u_tau + omt vel, in place in u_hat
  const double* u_prior;  // [batch][n] prior sample u_0
  double* u_next;         // [batch][n] out: u_0 + taun (u* - u_0)
  double omt, taun;
  int npx, nthr;     // patches per row, patches per level
  int ns_exact;      // full red-black sweeps that bring a level solve to fp64 rounding
  double log_rho2;   // log(rho^2) < 0: contraction per full sweep
};

struct Geo2d {
  int nx, hx, L, psz;         // psz = doubles per colour plane = L / 2
  int own;                    // plane offset of this thread's patch row 0: j0 hx + p0
  int offN, offS;             // plane offsets of the halo rows above / below (same columns)
  int rowW, rowE;             // plane offsets of the halo columns left / right of patch row 0
  int nat;                    // natural-layout offset of patch row 0: j0 nx + i0
  bool swap;                  // this lane fetches its east halo first (see gs_half)
};

struct Ring2d {
  double* stage;              // [2 stages][2 rows][L]
  uint32_t bar0;              // two mbarriers
  uint32_t phase;             // parity bits of the two stages
  int L;
  __device__ __forceinline__ double* row(int s, int which) const { return stage + (size_t)(2 * s + which) * L; }
  __device__ __forceinline__ void issue(int s, const double* a, const double* b) const {   // one thread
    const uint32_t bytes = (uint32_t)L * 8u;
    const uint32_t bar = bar0 + 8u * s;
    mbar_expect_tx(bar, 2u * bytes);
    bulk_g2s(smem_u32(row(s, 0)), a, bytes, bar);
    bulk_g2s(smem_u32(row(s, 1)), b, bytes, bar);
  }
  __device__ __forceinline__ void wait(int s) {
    mbar_wait(bar0 + 8u * s, (phase >> s) & 1u);
    phase ^= (1u << s);
  }
};

// sums a pass returns (block-reduced, identical in every thread)
struct Pass2d {
  double hinf, h1, f, wd, dd;
  int bad;
};

template <int PR>
__device__ __forceinline__ void load_nat(const double* __restrict__ base, int nx, double (&v)[PR][4]) {
#pragma unroll
  for (int r = 0; r < PR; ++r) {
    const double2 a = *reinterpret_cast<const double2*>(base + r * nx);
    const double2 b = *reinterpret_cast<const double2*>(base + r * nx + 2);
    v[r][0] = a.x; v[r][1] = a.y; v[r][2] = b.x; v[r][3] = b.y;
  }
}
template <int PR>
__device__ __forceinline__ void store_nat(double* __restrict__ base, int nx, const double (&v)[PR][4]) {
#pragma unroll
  for (int r = 0; r < PR; ++r) {
    *reinterpret_cast<double2*>(base + r * nx) = make_double2(v[r][0], v[r][1]);
    *reinterpret_cast<double2*>(base + r * nx + 2) = make_double2(v[r][2], v[r][3]);
  }
}
// own patch <-> colour planes: row r keeps cells e = 0, 2 in plane (r & 1) and e = 1, 3 in the other one
template <int PR>
__device__ __forceinline__ void store_planes(double* __restrict__ pl, const Geo2d& g, const double (&v)[PR][4]) {
#pragma unroll
  for (int r = 0; r < PR; ++r) {
    *reinterpret_cast<double2*>(pl + (r & 1) * g.psz + g.own + r * g.hx) = make_double2(v[r][0], v[r][2]);
    *reinterpret_cast<double2*>(pl + (1 - (r & 1)) * g.psz + g.own + r * g.hx) = make_double2(v[r][1], v[r][3]);
  }
}
template <int PR>
__device__ __forceinline__ void load_planes(const double* __restrict__ pl, const Geo2d& g, double (&v)[PR][4]) {
#pragma unroll
  for (int r = 0; r < PR; ++r) {
    const double2 a = *reinterpret_cast<const double2*>(pl + (r & 1) * g.psz + g.own + r * g.hx);
    const double2 b = *reinterpret_cast<const double2*>(pl + (1 - (r & 1)) * g.psz + g.own + r * g.hx);
    v[r][0] = a.x; v[r][2] = a.y; v[r][1] = b.x; v[r][3] = b.y;
  }
}

// One red-black half sweep: the cells of colour C take (rhs + ax (W + E) + ay (N + S)) / D from their neighbours of
// the other colour (own registers inside the patch, the halo from the other colour's plane).
template <int PR, int C>
__device__ __forceinline__ void gs_half(double* __restrict__ pl, const Geo2d& g, double (&q)[PR][4],
                                        const double (&rhs)[PR][4], const double (&invD)[PR][4], double ax, double ay,
                                        bool store) {
  const double* po = pl + (1 - C) * g.psz;
  const double2 nN = *reinterpret_cast<const double2*>(po + g.offN);
  const double2 nS = *reinterpret_cast<const double2*>(po + g.offS);
  // row r needs its west halo if (r & 1) == C, else its east halo: PR/2 of each.  A 64-bit load of 16 lanes at a
  // 16-byte stride is a 2-way bank conflict; pairing a west row with an east row and letting every other group of 8
  // lanes fetch the east one first puts the 16 lanes of a phase on 16 different bank pairs (odd / even 8-byte slots).
  double hWE[PR];
#pragma unroll
  for (int rp = 0; rp < PR; rp += 2) {
    const int rw = rp + C, re = rp + 1 - C;          // west row, east row of this pair
    const int ow = g.rowW + rw * g.hx, oe = g.rowE + re * g.hx;
    const double first = po[g.swap ? oe : ow];
    const double second = po[g.swap ? ow : oe];
    hWE[rw] = g.swap ? second : first;
    hWE[re] = g.swap ? first : second;
  }
#pragma unroll
  for (int r = 0; r < PR; ++r) {
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      if (((r + e) & 1) != C) continue;
      const double W = (e == 0) ? hWE[r] : q[r][e == 0 ? 0 : e - 1];
      const double E = (e == 3) ? hWE[r] : q[r][e == 3 ? 3 : e + 1];
      const double N = (r == 0) ? ((e >> 1) ? nN.y : nN.x) : q[r == 0 ? 0 : r - 1][e];
      const double S = (r == PR - 1) ? ((e >> 1) ? nS.y : nS.x) : q[r == PR - 1 ? r : r + 1][e];
      q[r][e] = fma(ax, W + E, fma(ay, N + S, rhs[r][e])) * invD[r][e];
    }
  }
  if (store) {
    double* pc = pl + C * g.psz;
#pragma unroll
    for (int r = 0; r < PR; ++r) {
      const int c0 = (r + C) & 1;
      *reinterpret_cast<double2*>(pc + g.own + r * g.hx) = make_double2(q[r][c0], q[r][c0 + 2]);
    }
  }
}

// Solve T q = rhs on the level: initial guess rhs / D, then `ns` full red-black sweeps.  q leaves in registers.
template <int PR>
__device__ __forceinline__ void level_solve(double* __restrict__ qpl, const Geo2d& g, double (&q)[PR][4],
                                            const double (&rhs)[PR][4], const double (&invD)[PR][4], double ax,
                                            double ay, int ns) {
#pragma unroll
  for (int r = 0; r < PR; ++r)
#pragma unroll
    for (int e = 0; e < 4; ++e) q[r][e] = rhs[r][e] * invD[r][e];
  if (ns <= 0) { __syncthreads(); return; }   // the barrier also separates the x-plane halo reads from the next level's stores
  store_planes<PR>(qpl, g, q);
  __syncthreads();
  for (int s = 0; s < ns; ++s) {
    gs_half<PR, 0>(qpl, g, q, rhs, invD, ax, ay, true);
    __syncthreads();
    const bool more = (s + 1 < ns);
    gs_half<PR, 1>(qpl, g, q, rhs, invD, ax, ay, more);
    if (more) __syncthreads();
  }
}

__device__ __forceinline__ double blk_sum2(double* red, double v, int nwarp) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  v = warp_sum(v);
  __syncthreads();
  if (lane == 0) red[warp] = v;
  __syncthreads();
  double r = 0.0;
  for (int w = 0; w < nwarp; ++w) r += red[w];   // fixed order: run-to-run deterministic
  return r;
}
__device__ __forceinline__ double blk_max2(double* red, double v, int nwarp) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  v = warp_max(v);
  __syncthreads();
  if (lane == 0) red[warp] = v;
  __syncthreads();
  double r = 0.0;
  for (int w = 0; w < nwarp; ++w) r = fmax(r, red[w]);
  return r;
}

// ---- forward pass at the point x (a1-a3, forward half of a5, a8 sums) --------------------------------------------
//   h_0 = x_0 - u0,  h_k = x_k - x_{k-1} - ax dxx x_k - ay dyy x_k + dt (x_k^3 - x_k)
//   q_0 = h_0,       T(x_k) q_k = h_k + q_{k-1}                       (q = J^-1 h: the Newton direction is -q)
//   trial_k = x_k - q_k  (full Gauss-Newton step),  y_k = q_k - (x_k - uh_k)  (right-hand side of J^T lam = y)
template <int PR>
__device__ void fwd_pass2d(const DevParams& P, const Geo2d& g, Ring2d& ring, double* __restrict__ xpl,
                           double* __restrict__ qpl, double* red, const double* __restrict__ x,
                           const double* __restrict__ uh, const double* __restrict__ u0, double* __restrict__ trial,
                           double* __restrict__ yout, double* __restrict__ ost, int ns, bool active, int nwarp,
                           Pass2d& out, const double* __restrict__ vel = nullptr, double omt = 0.0,
                           double* __restrict__ uh_out = nullptr) {
  const int nt = P.nt, L = g.L;
  const double ax = P.ac_ax, ay = P.ac_ay, dt = P.dt;
  const double c0 = 1.0 + 2.0 * ax + 2.0 * ay - dt, dt3 = 3.0 * dt, c1 = 2.0 * ax + 2.0 * ay - dt;
  double a_inf = 0.0, a_1 = 0.0, a_f = 0.0, a_wd = 0.0, a_dd = 0.0;
  double q[PR][4], rhs[PR][4], invD[PR][4];
  // PCFM step: x holds u_tau and the second row of a stage carries the velocity; the pass forms u_hat (Eq. 1) per level,
  // writes it to `uh_out` (in place over u_tau) and into both stage rows, so the rest of the level sees x = u_hat
  const double* __restrict__ second = vel ? vel : uh;
  const bool all_active = __syncthreads_and(active ? 1 : 0) != 0;
  if (threadIdx.x == 0) ring.issue(0, x, second);
  for (int k = 0; k < nt; ++k) {
    const int s = k & 1;
    ring.wait(s);
    double xv[PR][4];
    load_nat<PR>(ring.row(s, 0) + g.nat, g.nx, xv);
    if (vel) {
      double vv[PR][4];
      load_nat<PR>(ring.row(s, 1) + g.nat, g.nx, vv);
      // the spare threads of the last warp shadow patch 0: they must have read its velocity cells before thread 0 (another
      // warp) overwrites them with u_hat, or one of the two forms u_tau + omt u_hat (found at 96 x 42, 504 of 512 threads)
      if (!all_active) __syncthreads();
#pragma unroll
      for (int r = 0; r < PR; ++r)
#pragma unroll
        for (int e = 0; e < 4; ++e) xv[r][e] = fma(omt, vv[r][e], xv[r][e]);
      store_nat<PR>(ring.row(s, 1) + g.nat, g.nx, xv);
      if (active) store_nat<PR>(uh_out + (size_t)k * L + g.nat, g.nx, xv);
    }
    if (k == 0) {
      double u0v[PR][4];
      load_nat<PR>(u0 + g.nat, g.nx, u0v);
#pragma unroll
      for (int r = 0; r < PR; ++r)
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const double h = xv[r][e] - u0v[r][e];
          q[r][e] = h;
          const double ah = fabs(h);
          a_inf = fmax(a_inf, ah);
          a_1 += ah;
        }
      store_planes<PR>(xpl, g, xv);
      __syncthreads();
      if (threadIdx.x == 0 && nt > 1) ring.issue(1, x + L, second + L);
    } else {
      // rhs still holds x_{k-1} (own cells, left there by the end of the previous level); the planes take x_k
      store_planes<PR>(xpl, g, xv);
      if (threadIdx.x == 0) bulk_wait_read<0>();   // the previous level's trial row has left the staging row
      __syncthreads();
      if (threadIdx.x == 0 && k + 1 < nt) ring.issue(s ^ 1, x + (size_t)(k + 1) * L, second + (size_t)(k + 1) * L);
      // halo of x_k in both colours
      const double2 n1 = *reinterpret_cast<const double2*>(xpl + g.psz + g.offN);   // (-1, e = 0, 2): colour 1
      const double2 n0 = *reinterpret_cast<const double2*>(xpl + g.offN);           // (-1, e = 1, 3): colour 0
      const double2 s0 = *reinterpret_cast<const double2*>(xpl + g.offS);           // (PR, e = 0, 2): colour 0
      const double2 s1 = *reinterpret_cast<const double2*>(xpl + g.psz + g.offS);   // (PR, e = 1, 3): colour 1
      const double hN[4] = {n1.x, n0.x, n1.y, n0.y};
      const double hS[4] = {s0.x, s1.x, s0.y, s1.y};
      double hW[PR], hE[PR];
#pragma unroll
      for (int r = 0; r < PR; ++r) {
        hW[r] = xpl[((r + 1) & 1) * g.psz + g.rowW + r * g.hx];
        hE[r] = xpl[(r & 1) * g.psz + g.rowE + r * g.hx];
      }
#pragma unroll
      for (int r = 0; r < PR; ++r)
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const double v = xv[r][e];
          const double W = (e == 0) ? hW[r] : xv[r][e == 0 ? 0 : e - 1];
          const double E = (e == 3) ? hE[r] : xv[r][e == 3 ? 3 : e + 1];
          const double N = (r == 0) ? hN[e] : xv[r == 0 ? 0 : r - 1][e];
          const double S = (r == PR - 1) ? hS[e] : xv[r == PR - 1 ? r : r + 1][e];
          // h = (v - x_{k-1}) - ax (W + E - 2v) - ay (N + S - 2v) + dt (v^3 - v), grouped as
          //     (v - x_{k-1}) + v (2ax + 2ay - dt + dt v^2) - ax (W + E) - ay (N + S):  9 instead of 16 FP64 operations with D
          const double v2 = v * v;
          double h = fma(fma(dt, v2, c1), v, v - rhs[r][e]);
          h = fma(-ax, W + E, h);
          h = fma(-ay, N + S, h);
          const double ah = fabs(h);
          a_inf = fmax(a_inf, ah);
          a_1 += ah;
          rhs[r][e] = h + q[r][e];
          invD[r][e] = rcp_pos(fma(dt3, v2, c0));
        }
      level_solve<PR>(qpl, g, q, rhs, invD, ax, ay, ns);
    }
    // level end: own x_k (planes), own uh_k (stage); sums, outputs
    double uv[PR][4];
    load_nat<PR>(ring.row(s, 1) + g.nat, g.nx, uv);
    if (k > 0) load_planes<PR>(xpl, g, xv);
    double tv[PR][4], yv[PR][4];
#pragma unroll
    for (int r = 0; r < PR; ++r)
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const double w = xv[r][e] - uv[r][e], qq = q[r][e];
        a_f = fma(w, w, a_f);
        a_wd = fma(-w, qq, a_wd);
        a_dd = fma(qq, qq, a_dd);
        tv[r][e] = xv[r][e] - qq;
        yv[r][e] = qq - w;
        rhs[r][e] = xv[r][e];          // x_k for the next level's residual (not live across the sweeps)
      }
    // the trial row leaves through the staging row as one bulk (TMA) store: 16 STG.128 per thread back to back
    // filled the load/store queue and stalled the start of the next level (profiles/r02_direct2d.md)
    if (yout && active) store_nat<PR>(yout + (size_t)k * L + g.nat, g.nx, yv);
    if (trial) {
      store_nat<PR>(ost + g.nat, g.nx, tv);
      fence_proxy_async_smem();
      __syncthreads();
      if (threadIdx.x == 0) {
        bulk_s2g(trial + (size_t)k * L, smem_u32(ost), (uint32_t)L * 8u);
        bulk_commit();
      }
    }
  }
  if (threadIdx.x == 0) bulk_wait_all<0>();
  if (!active) { a_inf = 0.0; a_1 = 0.0; a_f = 0.0; a_wd = 0.0; a_dd = 0.0; }
  out.hinf = blk_max2(red, a_inf, nwarp);
  out.h1 = blk_sum2(red, a_1, nwarp);
  out.f = 0.5 * blk_sum2(red, a_f, nwarp);
  out.wd = blk_sum2(red, a_wd, nwarp);
  out.dd = blk_sum2(red, a_dd, nwarp);
  out.bad = !(finite_d(out.h1) && finite_d(out.f));
  // the rows just written are read by the next pass's bulk copies (async proxy)
  __threadfence();
  fence_proxy_async_all();
  __syncthreads();
}

// ---- multiplier sweep  J^T lam = y  at the final point x:  lam_k = T(x_k)^-1 (y_k + lam_{k+1}), lam_0 = y_0 + lam_1 ----
// y is read from and lam written to `lam` (in place, level by level); optionally copies x into ucopy.  Returns sum lam^2.
template <int PR>
__device__ double bwd_pass2d(const DevParams& P, const Geo2d& g, Ring2d& ring, double* __restrict__ qpl, double* red,
                             const double* __restrict__ x, double* __restrict__ lam, double* __restrict__ ucopy, int ns,
                             bool active, int nwarp, const double* __restrict__ uprior = nullptr,
                             double* __restrict__ unext = nullptr, double taun = 0.0) {
  const int nt = P.nt, L = g.L;
  const double ax = P.ac_ax, ay = P.ac_ay, dt = P.dt;
  const double c0 = 1.0 + 2.0 * ax + 2.0 * ay - dt, dt3 = 3.0 * dt;
  double q[PR][4], rhs[PR][4], invD[PR][4];
#pragma unroll
  for (int r = 0; r < PR; ++r)
#pragma unroll
    for (int e = 0; e < 4; ++e) q[r][e] = 0.0;
  double chk = 0.0;
  if (threadIdx.x == 0) ring.issue(0, lam + (size_t)(nt - 1) * L, x + (size_t)(nt - 1) * L);
  for (int k = nt - 1, idx = 0; k >= 0; --k, ++idx) {
    const int s = idx & 1;
    ring.wait(s);
    double yv[PR][4], xv[PR][4];
    load_nat<PR>(ring.row(s, 0) + g.nat, g.nx, yv);
    load_nat<PR>(ring.row(s, 1) + g.nat, g.nx, xv);
    if (unext) {   // OT pull-back of this level (Eq. 3): x is the final iterate, the prior row comes straight from HBM
      double up[PR][4];
      load_nat<PR>(uprior + (size_t)k * L + g.nat, g.nx, up);
#pragma unroll
      for (int r = 0; r < PR; ++r)
#pragma unroll
        for (int e = 0; e < 4; ++e) up[r][e] = fma(taun, xv[r][e] - up[r][e], up[r][e]);
      if (active) store_nat<PR>(unext + (size_t)k * L + g.nat, g.nx, up);
    }
    __syncthreads();   // every thread is done with the other stage (read one level ago) and with the q planes
    if (threadIdx.x == 0 && k > 0) ring.issue(s ^ 1, lam + (size_t)(k - 1) * L, x + (size_t)(k - 1) * L);
#pragma unroll
    for (int r = 0; r < PR; ++r)
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        rhs[r][e] = yv[r][e] + q[r][e];
        invD[r][e] = rcp_pos(fma(dt3, xv[r][e] * xv[r][e], c0));
      }
    if (k > 0) {
      level_solve<PR>(qpl, g, q, rhs, invD, ax, ay, ns);
    } else {
#pragma unroll
      for (int r = 0; r < PR; ++r)
#pragma unroll
        for (int e = 0; e < 4; ++e) q[r][e] = rhs[r][e];
    }
#pragma unroll
    for (int r = 0; r < PR; ++r)
#pragma unroll
      for (int e = 0; e < 4; ++e) chk = fma(q[r][e], q[r][e], chk);
    if (active) {
      store_nat<PR>(lam + (size_t)k * L + g.nat, g.nx, q);
      if (ucopy) store_nat<PR>(ucopy + (size_t)k * L + g.nat, g.nx, xv);
    }
  }
  if (!active) chk = 0.0;
  chk = blk_sum2(red, chk, nwarp);
  __threadfence();
  fence_proxy_async_all();
  __syncthreads();
  return chk;
}

template <int PR, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) project2d_direct_kernel(const __grid_constant__ Dir2dArgs A) {
  extern __shared__ __align__(128) unsigned char smem_d2[];
  const DevParams& P = A.P;
  const int b = blockIdx.x;
  if (b >= A.batch) return;
  const int tid = threadIdx.x;
  const bool active = tid < A.nthr;
  const int t = active ? tid : 0;     // spare threads of the last warp shadow patch 0 (same values, no stores, no sums)
  const int nwarp = (blockDim.x + 31) >> 5;
  const int L = P.lvl, nt = P.nt;
  const size_t n = (size_t)P.n;

  Geo2d g;
  g.nx = P.nx; g.hx = P.nx >> 1; g.L = L; g.psz = L >> 1;
  {
    const int pj = t / A.npx, pi = t % A.npx;
    const int j0 = PR * pj, p0 = 2 * pi;
    const int jn = (j0 == 0) ? P.ny - 1 : j0 - 1, js = (j0 + PR == P.ny) ? 0 : j0 + PR;
    const int pw = (p0 == 0) ? g.hx - 1 : p0 - 1, pe = (p0 + 2 == g.hx) ? 0 : p0 + 2;
    g.own = j0 * g.hx + p0;
    g.offN = jn * g.hx + p0;
    g.offS = js * g.hx + p0;
    g.rowW = j0 * g.hx + pw;
    g.rowE = j0 * g.hx + pe;
    g.nat = j0 * P.nx + 4 * pi;
    g.swap = (pi & 8) != 0;
  }
  double* sm = reinterpret_cast<double*>(smem_d2);
  Ring2d ring;
  ring.stage = sm;
  ring.L = L;
  double* xpl = sm + (size_t)4 * L;
  double* qpl = xpl + L;
  double* ost = qpl + L;         // staging row of the trial point (natural layout), leaves by bulk store
  double* red = ost + L;
  ring.bar0 = smem_u32(red + 32);
  ring.phase = 0;
  if (tid == 0) {
    mbar_init(ring.bar0, 1);
    mbar_init(ring.bar0 + 8u, 1);
    mbar_fence_init();
    fence_proxy_async_smem();
  }
  __syncthreads();

  const double* uh = A.u_hat + (size_t)b * n;
  const double* u0 = A.cdata + (size_t)b * L;
  double* ustar = A.u_star + (size_t)b * n;
  double* lam = A.lam ? A.lam + (size_t)b * n : nullptr;   // nullptr: multiplier-free call
  double* ws = A.ws + (size_t)b * kPcgVectors * n;
  double* const buf[3] = {ws, ws + n, ws + 2 * n};

  // sweeps of a pass whose input had ||h||_inf = hprev: the step only has to beat the quadratic term of the next
  // residual (inexact Newton; the residual itself is always evaluated exactly); eta = 1e-2 hprev^2 in [1e-16, 1e-6]
  const double* vel_b = A.vel ? A.vel + (size_t)b * n : nullptr;
  const double* up_b = A.u_next ? A.u_prior + (size_t)b * n : nullptr;
  double* un_b = A.u_next ? A.u_next + (size_t)b * n : nullptr;
  bool pulled = false;

  auto sweeps_for = [&](double hprev) -> int {
    double eta = 1e-2 * hprev * hprev;
    if (!(eta < 1e-6)) eta = 1e-6;
    if (eta <= 2.2e-16) return A.ns_exact;
    int s = (int)ceil(log(eta) / A.log_rho2);
    if (s < 1) s = 1;
    return s < A.ns_exact ? s : A.ns_exact;
  };

  const double* cur = uh;
  double* trial = nullptr;
  bool have_trial = false, polishing = false, have_y = false;
  int polish_left = 0, steps = 0, solves = 0, tries = 0, status = 0, nback = 0, passes = 0;
  long long inner = 0, rows_rd = 0, rows_wr = 0;
  double alpha = 1.0, mu = 0.0, phi_cur = 0.0, Dphi = 0.0, hprev = 1e300;
  Pass2d S;

  while (true) {
    if (!lam && have_trial && polishing && polish_left == 0) {
      // multiplier-free call: the last polish step is accepted without a test (R4) and nothing is computed at the
      // polished point (no y, no multiplier), so its pass is not run: `iters` is one linearisation short of a call with lam
      cur = trial;
      have_trial = false;
      break;
    }
    const double* pt = have_trial ? trial : cur;
    double* out = buf[0];
    if (out == pt || out == cur) out = buf[1];
    if (out == pt || out == cur) out = buf[2];
    // A pass writes the full-step trial point; the right-hand side y of the multiplier solve only when the point it
    // evaluates is final (last polish step done) or may turn out to be (quadratic convergence: ||h|| ~ hprev^2 < tol),
    // and then the level solves run to rounding.
    const bool last = polishing && polish_left == 0;
    const bool emit_y = lam && (last || hprev * hprev < 100.0 * P.tol);
    const int ns = (polishing || emit_y) ? A.ns_exact : sweeps_for(hprev);
    const bool shoot = vel_b && passes == 0;     // PCFM step: the first pass reads u_tau + velocity and forms u_hat
    fwd_pass2d<PR>(P, g, ring, xpl, qpl, red, pt, uh, u0, last ? nullptr : out, emit_y ? lam : nullptr, ost, ns, active,
                   nwarp, S, shoot ? vel_b : nullptr, A.omt, const_cast<double*>(uh));
    ++passes; inner += (long long)ns * (nt - 1);
    rows_rd += 2 * nt; rows_wr += (last ? 0 : nt) + (emit_y ? nt : 0) + (shoot ? nt : 0);
    have_y = emit_y;
    if (have_trial) {
      if (!polishing) {
        const double phi_t = S.f + mu * S.h1;
        const bool ok = !S.bad && finite_d(phi_t) && (phi_t <= phi_cur + P.ls_c1 * alpha * Dphi);
        if (!ok) {
          if (++tries > P.ls_max) { status = SNAP_ST_LINESEARCH; break; }
          for (size_t i = tid; i < n; i += blockDim.x) trial[i] = fma(P.ls_shrink, trial[i] - cur[i], cur[i]);
          __threadfence();
          fence_proxy_async_all();
          __syncthreads();
          alpha *= P.ls_shrink;
          rows_rd += 2 * nt; rows_wr += nt; ++nback;
          continue;
        }
        ++steps;
      }
      cur = trial;
      have_trial = false;
    } else if (S.bad) {
      status = SNAP_ST_NONFINITE;
      break;
    }
    ++solves;
    if (!finite_d(S.wd) || !finite_d(S.dd)) { status = SNAP_ST_NONFINITE; break; }   // non-finite direction (R16)
    hprev = S.hinf;
    bool final_pt = false;
    if (polishing) {
      final_pt = (polish_left == 0);
    } else if (S.hinf < P.tol) {
      polishing = true;
      polish_left = (S.hinf > kPolishSkip * P.tol) ? P.polish : 0;
      final_pt = (polish_left == 0);
    } else if (steps >= P.max_iter) {
      status = SNAP_ST_MAXITER;
      final_pt = true;
    }
    if (final_pt) break;
    if (polishing) {
      --polish_left;
    } else {
      mu = merit_mu(mu, S.wd, S.dd, S.h1, kMuRho, kMuFloor);
      phi_cur = S.f + mu * S.h1;
      Dphi = S.wd - mu * S.h1;
      alpha = 1.0;
      tries = 0;
    }
    trial = out;
    have_trial = true;
  }

  if (!lam) {
    // multiplier-free call: u* = the returned iterate, nothing else to do
    if (status != SNAP_ST_NONFINITE && cur != ustar) {
      __syncthreads();
      // one stream: u* and (PCFM step) its pull-back; 128-bit accesses, 4 independent iterations per thread
      const double2* x2 = reinterpret_cast<const double2*>(cur);
      const double2* p2 = reinterpret_cast<const double2*>(up_b);
      double2* c2 = reinterpret_cast<double2*>(ustar);
      double2* o2 = reinterpret_cast<double2*>(un_b);
      const size_t n2 = n >> 1, T4 = 4 * (size_t)blockDim.x;
      for (size_t i0 = tid; i0 < n2; i0 += T4) {
        double2 xv[4], pv[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const size_t i = i0 + (size_t)u * blockDim.x;
          if (i < n2) { xv[u] = x2[i]; if (un_b) pv[u] = p2[i]; }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const size_t i = i0 + (size_t)u * blockDim.x;
          if (i < n2) {
            c2[i] = xv[u];
            if (un_b) o2[i] = make_double2(fma(A.taun, xv[u].x - pv[u].x, pv[u].x), fma(A.taun, xv[u].y - pv[u].y, pv[u].y));
          }
        }
      }
      if (un_b) pulled = true;
      rows_rd += nt + (un_b ? nt : 0); rows_wr += nt + (un_b ? nt : 0);
    }
  } else if (status == SNAP_ST_LINESEARCH || (status != SNAP_ST_NONFINITE && !have_y)) {
    // the returned point was not known to be final when its pass ran (feasible input, polish skipped or 0, max_iter,
    // line search): right-hand side of the multiplier solve there, level solves to rounding
    fwd_pass2d<PR>(P, g, ring, xpl, qpl, red, cur, uh, u0, nullptr, lam, ost, A.ns_exact, active, nwarp, S);
    ++passes; inner += (long long)A.ns_exact * (nt - 1);
    rows_rd += 2 * nt; rows_wr += nt;
    if (S.bad || !finite_d(S.dd)) status = SNAP_ST_NONFINITE;
  }
  if (lam && status != SNAP_ST_NONFINITE) {
    const bool late_copy = (ustar == uh) && (cur != ustar);   // in place: u_hat survives until lam is known finite
    double* ucopy = (cur != ustar && !late_copy) ? ustar : nullptr;
    const bool pull = un_b && !late_copy && status == 0;
    const double chk = bwd_pass2d<PR>(P, g, ring, qpl, red, cur, lam, ucopy, A.ns_exact, active, nwarp,
                                      pull ? up_b : nullptr, pull ? un_b : nullptr, A.taun);
    ++passes; inner += (long long)A.ns_exact * (nt - 1);
    rows_rd += 2 * nt + (pull ? nt : 0); rows_wr += nt + (ucopy ? nt : 0) + (pull ? nt : 0);
    pulled = pull;
    if (!finite_d(chk)) {
      status = SNAP_ST_NONFINITE;
      pulled = false;
    } else if (late_copy) {
      for (size_t i = tid; i < n; i += blockDim.x) ustar[i] = cur[i];
      rows_rd += nt; rows_wr += nt;
    }
  }
  if (status == SNAP_ST_NONFINITE) {   // R16: u* = u_hat, lam = 0
    __syncthreads();
    if (ustar != uh)
      for (size_t i = tid; i < n; i += blockDim.x) ustar[i] = uh[i];
    if (lam)
      for (size_t i = tid; i < n; i += blockDim.x) lam[i] = 0.0;
  }
  if (un_b && !pulled) {   // pull-back of whatever u* holds (statuses that did not stream the final iterate)
    __syncthreads();
    for (size_t i = tid; i < n; i += blockDim.x) {
      const double u0p = up_b[i];
      un_b[i] = fma(A.taun, ustar[i] - u0p, u0p);
    }
    rows_rd += 2 * nt; rows_wr += nt;
  }
  if (tid == 0) {
    A.iters[b] = (status == 0) ? solves : status;
    if (A.stats) {
      long long* stat = A.stats + (size_t)b * SNAP_STAT_COUNT;
      stat[SNAP_STAT_LINEARISATIONS] = solves; stat[SNAP_STAT_PASSES] = passes;
      stat[SNAP_STAT_ROWS_READ] = rows_rd; stat[SNAP_STAT_ROWS_WRITTEN] = rows_wr;
      stat[SNAP_STAT_VARIANT] = SNAP_VAR_DIRECT2D; stat[SNAP_STAT_INNER] = inner;
      stat[SNAP_STAT_ROW_DOUBLES] = L; stat[SNAP_STAT_BACKTRACKS] = nback;
    }
  }
}

// Eligibility and launch.  Returns SNAP_OK, an error, or +1 when the shape / parameters are outside this path
// (the caller then takes the PCG kernel).
int launch_project2d_direct(snap_problem* p, int batch, const double* u_hat, const double* cdata,
                                   double* u_star, double* lambda, int* iters, void* workspace, long long* stats,
                                   const FlowArgs* flow, cudaStream_t st) {
  const DevParams& d = p->dp;
  if (d.nx % 4 != 0 || d.ny % 2 != 0) return 1;
  const int PR = (d.ny % 4 == 0) ? 4 : 2;
  const int npx = d.nx / 4, nthr = npx * (d.ny / PR);
  if (nthr > (PR == 4 ? 256 : 512)) return 1;
  const double off = 2.0 * d.ac_ax + 2.0 * d.ac_ay, dmin = 1.0 + off - d.dt;
  if (!(dmin > 0.0) || !(off >= 0.0)) return 1;
  const double rho = off / dmin;
  if (!(rho < 0.7)) return 1;                       // slow relaxation: the ADI-preconditioned PCG path serves it
  auto al16 = [](const void* q) { return (reinterpret_cast<uintptr_t>(q) & 15u) == 0; };
  if (!(al16(u_hat) && al16(cdata) && al16(u_star) && al16(lambda) && al16(workspace))) return 1;
  Dir2dArgs a;
  a.P = d;
  a.batch = batch;
  a.u_hat = u_hat; a.cdata = cdata; a.u_star = u_star; a.lam = lambda; a.iters = iters;
  a.ws = reinterpret_cast<double*>(workspace);
  a.stats = stats;
  a.npx = npx; a.nthr = nthr;
  a.vel = flow ? flow->vel : nullptr;
  a.u_prior = flow ? flow->u_prior : nullptr;
  a.u_next = flow ? flow->u_next : nullptr;
  a.omt = flow ? flow->omt : 0.0;
  a.taun = flow ? flow->taun : 0.0;
  if (flow && !(al16(flow->vel) && al16(flow->u_prior) && al16(flow->u_next))) return 1;
  // error after s full sweeps <= rho^(2 s) ||q||_inf (initial guess rhs / D is already within rho); 2.2e-16 is rounding
  a.log_rho2 = (rho > 0.0) ? 2.0 * log(rho) : -1e30;
  a.ns_exact = (rho > 0.0) ? (int)ceil(log(2.2e-16) / a.log_rho2) : 0;
  if (a.ns_exact < 1) a.ns_exact = (rho > 0.0) ? 1 : 0;
  const size_t smem = ((size_t)7 * d.lvl + 32 + 4) * sizeof(double);
  if (smem > (size_t)p->max_smem_optin) return 1;
  const int threads = (nthr + 31) / 32 * 32;
  cudaError_t err;
  if (PR == 4) {
    auto k = project2d_direct_kernel<4, 256>;
    if (cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return SNAP_ECUDA;
    k<<<batch, threads, smem, st>>>(a);
  } else {
    auto k = project2d_direct_kernel<2, 512>;
    if (cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return SNAP_ECUDA;
    k<<<batch, threads, smem, st>>>(a);
  }
  err = cudaGetLastError();
  p->launches++;
  return err == cudaSuccess ? SNAP_OK : SNAP_ECUDA;
}

}  // namespace snap
