// Residual + per-type norms (a1, Eq. 27), matrix-free Schur operator J J^T x (a2 + a4) for
// every kind, and the affine heat kind (closed-form block solve with the dense mass border rows, a7).
// These are plain global-memory kernels: one CTA per sample, warps take time levels round-robin.
#pragma once
#include "device_utils.cuh"
#include "snap_internal.h"

namespace snap {

constexpr int kMiscThreads = 256;

// one-step scheme residual of cell c of level k >= 1 (needs levels k-1 and k)
__device__ __forceinline__ double pde_residual(const DevParams& P, const double* __restrict__ up /*u[k-1]*/,
                                               const double* __restrict__ uk /*u[k]*/, int c) {
  const int nx = P.nx;
  if (P.kind == SNAP_BURGERS1D_LF || P.kind == SNAP_BURGERS1D_LF_MASS) {
    const int ip = (c + 1 == nx) ? 0 : c + 1, im = (c == 0) ? nx - 1 : c - 1;
    const double v = up[c], vp = up[ip], vm = up[im];
    const double phi = fma(P.bs_a0, v, (vp + vm) * fma(-P.bs_qs, vp - vm, P.bs_e));
    return uk[c] - phi;
  } else if (P.kind == SNAP_FISHER1D_IE) {
    const double w = uk[c];
    const double wl = (c > 0) ? uk[c - 1] : w, wr = (c < nx - 1) ? uk[c + 1] : w;
    return w - up[c] - P.fi_a * ((wl - w) + (wr - w)) - P.fi_dtrho * w * (1.0 - w);
  } else {  // Allen-Cahn 2D
    const int ny = P.ny;
    const int j = c / nx, i = c - j * nx;
    const int xp = j * nx + ((i + 1 == nx) ? 0 : i + 1), xm = j * nx + ((i == 0) ? nx - 1 : i - 1);
    const int yp = ((j + 1 == ny) ? 0 : j + 1) * nx + i, ym = ((j == 0) ? ny - 1 : j - 1) * nx + i;
    const double w = uk[c];
    const double lapx = (uk[xp] - w) + (uk[xm] - w), lapy = (uk[yp] - w) + (uk[ym] - w);
    return w - up[c] - P.ac_ax * lapx - P.ac_ay * lapy + P.dt * (w * w * w - w);
  }
}

// (T_k x)_c for the implicit kinds / (A_k x)_c for Burgers, with coefficients from the level row `uk`.
__device__ __forceinline__ double level_op(const DevParams& P, const double* __restrict__ uk,
                                           const double* __restrict__ x, int c, bool transpose) {
  const int nx = P.nx;
  if (P.kind == SNAP_BURGERS1D_LF || P.kind == SNAP_BURGERS1D_LF_MASS) {
    const int ip = (c + 1 == nx) ? 0 : c + 1, im = (c == 0) ? nx - 1 : c - 1;
    if (!transpose)  // (A x)_i = a0 x_i + (e - hs v_{i+1}) x_{i+1} + (e + hs v_{i-1}) x_{i-1}
      return fma(fma(-P.bs_hs, uk[ip], P.bs_e), x[ip], fma(fma(P.bs_hs, uk[im], P.bs_e), x[im], P.bs_a0 * x[c]));
    return fma(fma(-P.bs_hs, uk[c], P.bs_e), x[im], fma(fma(P.bs_hs, uk[c], P.bs_e), x[ip], P.bs_a0 * x[c]));
  } else if (P.kind == SNAP_FISHER1D_IE) {
    const double w = uk[c], xc = x[c];
    const double xl = (c > 0) ? x[c - 1] : xc, xr = (c < nx - 1) ? x[c + 1] : xc;
    return xc - P.fi_a * ((xl - xc) + (xr - xc)) - P.fi_dtrho * (1.0 - 2.0 * w) * xc;
  } else {
    const int ny = P.ny;
    const int j = c / nx, i = c - j * nx;
    const int xp = j * nx + ((i + 1 == nx) ? 0 : i + 1), xm = j * nx + ((i == 0) ? nx - 1 : i - 1);
    const int yp = ((j + 1 == ny) ? 0 : j + 1) * nx + i, ym = ((j == 0) ? ny - 1 : j - 1) * nx + i;
    const double w = uk[c], xc = x[c];
    return xc - P.ac_ax * ((x[xp] - xc) + (x[xm] - xc)) - P.ac_ay * ((x[yp] - xc) + (x[ym] - xc)) +
           P.dt * (3.0 * w * w - 1.0) * xc;
  }
}

__device__ __forceinline__ bool is_burgers(const DevParams& P) {
  return P.kind == SNAP_BURGERS1D_LF || P.kind == SNAP_BURGERS1D_LF_MASS;
}

// block-wide reductions of per-thread partials (fixed order): warp shuffle, then warp 0 over the partials
__device__ __forceinline__ double block_reduce(double v, double* red, bool is_max) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  v = is_max ? warp_max(v) : warp_sum(v);
  __syncthreads();
  if (lane == 0) red[warp] = v;
  __syncthreads();
  double r = (lane < nw) ? red[lane] : 0.0;
  r = is_max ? warp_max(r) : warp_sum(r);
  return r;  // valid in every lane of every warp
}

__device__ __forceinline__ double sample_mass0(const DevParams& P, const double* __restrict__ u0, double* red) {
  double s = 0.0;
  for (int i = threadIdx.x; i < P.nx; i += blockDim.x) s += u0[i];
  return P.dx * block_reduce(s, red, false);
}

// h(u) and [||h||_inf, ||h_IC||_2, ||h_PDE||_2, ||h_mass||_2] per sample.
__global__ void __launch_bounds__(kMiscThreads) residual_kernel(const __grid_constant__ DevParams P, int batch,
                                                                const double* __restrict__ u,
                                                                const double* __restrict__ cdata,
                                                                double* __restrict__ h, double* __restrict__ norms) {
  __shared__ double red[32];
  const int b = blockIdx.x;
  if (b >= batch) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const double* ub = u + (size_t)b * P.n;
  const double* u0 = cdata + (size_t)b * P.lvl;
  double* hb = h ? h + (size_t)b * P.m : nullptr;
  const int loc_levels = (P.kind == SNAP_HEAT1D_IC_MASS) ? 1 : P.nt;
  const size_t mass_off = (size_t)loc_levels * P.lvl;
  double M0 = 0.0;
  if (P.has_mass) M0 = sample_mass0(P, u0, red);
  double hinf = 0.0, s_ic = 0.0, s_pde = 0.0, s_mass = 0.0;
  for (int k = warp; k < P.nt; k += nw) {
    const double* uk = ub + (size_t)k * P.lvl;
    double msum = 0.0;
    for (int c = lane; c < P.lvl; c += 32) {
      if (P.has_mass) msum += uk[c];
      if (k < loc_levels) {
        double r;
        if (k == 0) {
          r = uk[c] - u0[c];
          s_ic = fma(r, r, s_ic);
        } else {
          r = pde_residual(P, uk - P.lvl, uk, c);
          s_pde = fma(r, r, s_pde);
        }
        hinf = fmax(hinf, finite_d(r) ? fabs(r) : 1.7976931348623157e308);
        if (hb) hb[(size_t)k * P.lvl + c] = r;
      }
    }
    if (P.has_mass) {
      const double hm = P.dx * warp_sum(msum) - M0;
      if (lane == 0) {
        s_mass = fma(hm, hm, s_mass);
        hinf = fmax(hinf, finite_d(hm) ? fabs(hm) : 1.7976931348623157e308);
        if (hb) hb[mass_off + k] = hm;
      }
    }
  }
  hinf = block_reduce(hinf, red, true);
  s_ic = block_reduce(s_ic, red, false);
  s_pde = block_reduce(s_pde, red, false);
  s_mass = block_reduce(s_mass, red, false);
  if (norms && threadIdx.x == 0) {
    double* nb = norms + (size_t)b * 5;
    nb[0] = hinf;
    nb[1] = sqrt(s_ic);
    nb[2] = sqrt(s_pde);
    nb[3] = sqrt(s_mass);
    nb[4] = 0.0;
  }
}

// g = J(u)^T x   (n-vector per sample).  x in the multiplier layout.
__global__ void __launch_bounds__(kMiscThreads) jt_apply_kernel(const __grid_constant__ DevParams P, int batch,
                                                                const double* __restrict__ u,
                                                                const double* __restrict__ x,
                                                                double* __restrict__ g) {
  const int b = blockIdx.x;
  if (b >= batch) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const double* ub = u + (size_t)b * P.n;
  const double* xb = x + (size_t)b * P.m;
  double* gb = g + (size_t)b * P.n;
  const int loc_levels = (P.kind == SNAP_HEAT1D_IC_MASS) ? 1 : P.nt;
  const double* xmass = xb + (size_t)loc_levels * P.lvl;
  for (int k = warp; k < P.nt; k += nw) {
    const double* uk = ub + (size_t)k * P.lvl;
    const double* xk = xb + (size_t)k * P.lvl;
    const double madd = P.has_mass ? P.dx * xmass[k] : 0.0;
    for (int c = lane; c < P.lvl; c += 32) {
      double v = 0.0;
      if (k < loc_levels) {
        if (is_burgers(P)) {  // (J^T x)_k = x_k - A_k^T x_{k+1}
          v = xk[c];
          if (k + 1 < P.nt) v -= level_op(P, uk, xk + P.lvl, c, true);
        } else if (P.kind == SNAP_HEAT1D_IC_MASS) {
          v = xk[c];
        } else {              // level 0: x_0 - x_1 ; level k: T_k x_k - x_{k+1}
          v = (k == 0) ? xk[c] : level_op(P, uk, xk, c, true);
          if (k + 1 < P.nt) v -= xk[P.lvl + c];
        }
      }
      gb[(size_t)k * P.lvl + c] = v + madd;
    }
  }
}

// out = J(u) g   (multiplier layout)
__global__ void __launch_bounds__(kMiscThreads) j_apply_kernel(const __grid_constant__ DevParams P, int batch,
                                                               const double* __restrict__ u,
                                                               const double* __restrict__ g,
                                                               double* __restrict__ out) {
  const int b = blockIdx.x;
  if (b >= batch) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const double* ub = u + (size_t)b * P.n;
  const double* gb = g + (size_t)b * P.n;
  double* ob = out + (size_t)b * P.m;
  const int loc_levels = (P.kind == SNAP_HEAT1D_IC_MASS) ? 1 : P.nt;
  double* omass = ob + (size_t)loc_levels * P.lvl;
  for (int k = warp; k < P.nt; k += nw) {
    const double* uk = ub + (size_t)k * P.lvl;
    const double* gk = gb + (size_t)k * P.lvl;
    double msum = 0.0;
    for (int c = lane; c < P.lvl; c += 32) {
      if (P.has_mass) msum += gk[c];
      if (k < loc_levels) {
        double v;
        if (k == 0) v = gk[c];
        else if (is_burgers(P)) v = gk[c] - level_op(P, uk - P.lvl, gk - P.lvl, c, false);
        else v = level_op(P, uk, gk, c, false) - gk[c - P.lvl];
        ob[(size_t)k * P.lvl + c] = v;
      }
    }
    if (P.has_mass) {
      msum = warp_sum(msum);
      if (lane == 0) omass[k] = P.dx * msum;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// HEAT1D_IC_MASS (affine): IC rows A = J_ic J_ic^T = I, border rows C = J_mass J_ic^T (only level 0 couples),
// D = J_mass J_mass^T = nx dx^2 I.  Border Schur complement S_b = D - C A^{-1} C^T = nx dx^2 (I - e_0 e_0^T):
// singular in row 0 (that mass row is implied by the IC rows), diagonal elsewhere.
//   basic solution : lam_mass,0 = 0 ; lam_mass,k = r_mass,k / (nx dx^2) ; lam_ic = r_ic
//   minimum norm   : lam -= N^T (N lam) / (N N^T),  N = (dx 1 on IC rows, -1 on mass row 0),  N N^T = 1 + nx dx^2
// r = h - J (u - u_hat) = J u_hat - b does not depend on u, so one Gauss-Newton step is exact;
// the full step satisfies the Armijo condition identically (1/2 |d|^2 = 1/2 lam^T h <= mu |h|_1 / 2.2).
// One CTA per sample; iters = 2 (step + the solve at the projected point) or 1 if u_hat is already feasible.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kMiscThreads) heat_project_kernel(const __grid_constant__ DevParams P, int batch,
                                                                    const double* __restrict__ u_hat,
                                                                    const double* __restrict__ cdata,
                                                                    double* __restrict__ u_star,
                                                                    double* __restrict__ lam, int* __restrict__ iters,
                                                                    long long* __restrict__ stats) {
  // One CTA per sample: the levels are independent (every non-redundant mass row has its own multiplier), so the
  // warps of the CTA take the levels round-robin; only ||h||_inf and the non-finite flag are reduced over the CTA.
  __shared__ double s_max[kMiscThreads / 32];
  __shared__ int s_bad[kMiscThreads / 32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  const int b = blockIdx.x;
  if (b >= batch) return;
  const int nx = P.nx, nt = P.nt;
  const double* uh = u_hat + (size_t)b * P.n;
  const double* u0 = cdata + (size_t)b * nx;
  double* us = u_star + (size_t)b * P.n;
  double* lb = lam + (size_t)b * P.m;
  if (threadIdx.x == 0 && stats) {   // one pass: reads u_hat twice at most (the second time from cache), writes u*
    long long* stat = stats + (size_t)b * SNAP_STAT_COUNT;
    stat[SNAP_STAT_LINEARISATIONS] = 2; stat[SNAP_STAT_PASSES] = 2;
    stat[SNAP_STAT_ROWS_READ] = 2 * nt; stat[SNAP_STAT_ROWS_WRITTEN] = nt;
    stat[SNAP_STAT_VARIANT] = SNAP_VAR_HEAT_CLOSED_FORM; stat[SNAP_STAT_INNER] = 0;
    stat[SNAP_STAT_ROW_DOUBLES] = nx; stat[SNAP_STAT_BACKTRACKS] = 0;
  }
  const double c = (double)nx * P.dx * P.dx;
  double s0 = 0.0;
  for (int i = lane; i < nx; i += 32) s0 += u0[i];
  const double M0 = P.dx * warp_sum(s0);   // same order in every warp: identical value

  auto block_max = [&](double v, int flag, int& flag_out) {
    __syncthreads();
    if (lane == 0) { s_max[warp] = v; s_bad[warp] = flag; }
    __syncthreads();
    double m = 0.0;
    int f = 0;
    for (int w2 = 0; w2 < nwarp; ++w2) { m = fmax(m, s_max[w2]); f |= s_bad[w2]; }
    flag_out = f;
    return m;
  };

  // solve 1 at u = u_hat: residual norms and the mass multipliers
  double hinf = 0.0;
  int bad = 0;
  for (int k = warp; k < nt; k += nwarp) {
    double sk = 0.0, dmax = 0.0;
    for (int i = lane; i < nx; i += 32) {
      const double v = uh[(size_t)k * nx + i];
      sk += v;
      if (k == 0) {
        const double d = v - u0[i];
        bad |= !finite_d(d);
        dmax = fmax(dmax, fabs(d));
      }
    }
    const double rm = P.dx * warp_sum(sk) - M0;
    bad |= !finite_d(rm);
    hinf = fmax(hinf, fmax(fabs(rm), warp_max(dmax)));
    if (lane == 0) lb[nx + k] = (k == 0) ? 0.0 : rm / c;
  }
  bad = warp_or(bad);
  hinf = block_max(hinf, bad, bad);
  if (bad) {  // R16
    if (us != uh)
      for (size_t i = threadIdx.x; i < (size_t)P.n; i += blockDim.x) us[i] = uh[i];
    __syncthreads();
    for (int i = threadIdx.x; i < P.m; i += blockDim.x) lb[i] = 0.0;
    if (threadIdx.x == 0) iters[b] = SNAP_ST_NONFINITE;
    return;
  }

  double dsum = 0.0;
  for (int i = lane; i < nx; i += 32) dsum += uh[i] - u0[i];
  dsum = warp_sum(dsum);
  const double lm0 = (P.lambda_mode == 0) ? P.dx * dsum / (1.0 + c) : 0.0;  // minimum-norm correction
  const bool feasible = hinf <= kPolishSkip * P.tol;
  int solves = 1;
  // IC multipliers need u_hat[0]: computed before level 0 of u_star (which may alias u_hat) is overwritten
  if (warp == 0) {
    for (int i = lane; i < nx; i += 32) lb[i] = (uh[i] - u0[i]) - P.dx * lm0;
    if (lane == 0) lb[nx] = lm0;
  }
  __syncthreads();
  if (feasible) {
    if (us != uh)
      for (size_t i = threadIdx.x; i < (size_t)P.n; i += blockDim.x) us[i] = uh[i];
  } else {
    // full step u = u_hat - J^T lam:  level 0 -> u0 ; level k -> u_hat[k] - dx lam_mass,k ; then solve 2 at the
    // projected point: the residual there decides convergence; r (hence lam) is unchanged
    double h2 = 0.0;
    for (int k = warp; k < nt; k += nwarp) {
      const double sh = (k == 0) ? 0.0 : P.dx * lb[nx + k];
      double sk = 0.0, dmax = 0.0;
      for (int i = lane; i < nx; i += 32) {
        const double v = (k == 0) ? u0[i] : uh[(size_t)k * nx + i] - sh;
        us[(size_t)k * nx + i] = v;
        sk += v;
        if (k == 0) dmax = fmax(dmax, fabs(v - u0[i]));
      }
      h2 = fmax(h2, fmax(fabs(P.dx * warp_sum(sk) - M0), warp_max(dmax)));
    }
    int dummy;
    h2 = block_max(h2, 0, dummy);
    solves = 2;
    if (!(h2 < P.tol)) solves = SNAP_ST_MAXITER;
  }
  if (threadIdx.x == 0) iters[b] = solves;
}

// ---- PCFM step, unfused parts (paths whose projection kernel does not fuse them): Eq. 1 and Eq. 3 ----
__global__ void __launch_bounds__(kMiscThreads) flow_shoot_kernel(size_t total, double* __restrict__ u, const double* __restrict__ vel,
                                                                 double omt) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x)
    u[i] = fma(omt, vel[i], u[i]);                 // u_hat = u_tau + (1 - tau) v, in place
}
__global__ void __launch_bounds__(kMiscThreads) flow_pullback_kernel(size_t total, const double* __restrict__ u1,
                                                                    const double* __restrict__ u_prior,
                                                                    double* __restrict__ u_next, double taun) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    const double u0p = u_prior[i];
    u_next[i] = fma(taun, u1[i] - u0p, u0p);       // u_tau' = u_0 + tau' (u_1 - u_0)
  }
}

}  // namespace snap
