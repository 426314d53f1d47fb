// Kind 6, NS2D_VORT_ENST: the paper's Navier-Stokes constraint set (Eq. 20: initial vorticity, total vorticity
// and enstrophy of every later level).  There are no local PDE rows: level k >= 1 is constrained only by its two global
// rows, the levels decouple, and the Newton-KKT fixed point of one level has a closed form -- the projection onto a sphere
// inside a hyperplane (as the heat kind has one, a7):
//     w*_k = m + (w_hat_k - mean(w_hat_k)) / s ,   m = mean(w_IC),  r = ||w_IC - m||_2,  s = ||w_hat_k - mean(w_hat_k)||_2 / r
//     lam_Z,k = (s - 1) / (2 a) ,  lam_V,k = (mean(w_hat_k) - s m) / a ,  a = dx dy         (stationarity split into mean / deviation)
//     w*_0 = w_IC ,  lam_IC = w_hat_0 - w_IC.
// One CTA per sample; the warps take the levels round-robin.  Phase 1 reads w_hat and keeps (mean, s) per level in shared
// memory, phase 2 writes the outputs (so that a non-finite level leaves u* = u_hat even in place, R16).
#pragma once
#include "device_utils.cuh"
#include "kernels_misc.cuh"
#include "snap_internal.h"

namespace snap {

constexpr int kNsMaxLevels = 2048;   // (mean, s) per level live in shared memory

__global__ void __launch_bounds__(kMiscThreads) ns_project_kernel(const __grid_constant__ DevParams P, int batch,
                                                                 const double* __restrict__ u_hat,
                                                                 const double* __restrict__ cdata, double* u_star,
                                                                 double* lam, int* __restrict__ iters,
                                                                 long long* __restrict__ stats) {
  __shared__ double red[32];
  __shared__ double s_mean[kNsMaxLevels], s_scale[kNsMaxLevels];
  __shared__ int s_bad;
  const int b = blockIdx.x;
  if (b >= batch) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int L = P.lvl, nt = P.nt;
  const double a = P.dx * P.dy;
  const double* uh = u_hat + (size_t)b * P.n;
  const double* w0 = cdata + (size_t)b * L;
  double* us = u_star + (size_t)b * P.n;
  double* lb = lam ? lam + (size_t)b * P.m : nullptr;
  if (threadIdx.x == 0) s_bad = 0;
  // mean and radius of the initial vorticity (two passes: the radius from the deviations, not from sum w^2 - N m^2)
  double acc = 0.0;
  for (int c = threadIdx.x; c < L; c += blockDim.x) acc += w0[c];
  const double m = block_reduce(acc, red, false) / (double)L;
  acc = 0.0;
  for (int c = threadIdx.x; c < L; c += blockDim.x) { const double d = w0[c] - m; acc = fma(d, d, acc); }
  const double r = sqrt(block_reduce(acc, red, false));
  // ---- phase 1: mean and deviation norm of every level of w_hat ----
  for (int k = 1 + warp; k < nt; k += nw) {
    const double* row = uh + (size_t)k * L;
    double s1 = 0.0;
    for (int c = lane; c < L; c += 32) s1 += row[c];
    const double mh = warp_sum(s1) / (double)L;
    double s2 = 0.0;
    for (int c = lane; c < L; c += 32) { const double d = row[c] - mh; s2 = fma(d, d, s2); }
    const double nd = sqrt(warp_sum(s2));
    // r = 0: the level is pinned to the constant m (scale 0 marks it); nd = 0 with r > 0: no direction to project along
    const double sc = (r > 0.0) ? nd / r : 0.0;
    if (lane == 0) {
      s_mean[k] = mh;
      s_scale[k] = sc;
      if (!finite_d(mh) || !finite_d(nd) || (r > 0.0 && !(nd > 0.0))) s_bad = 1;
    }
  }
  {
    double chk = 0.0;
    for (int c = threadIdx.x; c < L; c += blockDim.x) chk += uh[c];
    chk = block_reduce(chk, red, false);          // also the barrier between the phases
    if (threadIdx.x == 0 && !(finite_d(chk) && finite_d(m) && finite_d(r))) s_bad = 1;
  }
  __syncthreads();
  const bool bad = s_bad != 0;
  // ---- phase 2: outputs ----
  if (bad) {
    if (us != uh)
      for (size_t i = threadIdx.x; i < (size_t)P.n; i += blockDim.x) us[i] = uh[i];
    if (lb)
      for (int i = threadIdx.x; i < P.m; i += blockDim.x) lb[i] = 0.0;
  } else {
    for (int c = threadIdx.x; c < L; c += blockDim.x) {
      const double t = uh[c], ic = w0[c];
      if (lb) lb[c] = t - ic;
      us[c] = ic;
    }
    for (int k = 1 + warp; k < nt; k += nw) {
      const double mh = s_mean[k], sc = s_scale[k];
      const double inv = (sc > 0.0) ? 1.0 / sc : 0.0;
      const double* row = uh + (size_t)k * L;
      double* out = us + (size_t)k * L;
      for (int c = lane; c < L; c += 32) out[c] = fma(row[c] - mh, inv, m);
      if (lb && lane == 0) {
        lb[L + (k - 1)] = (sc > 0.0) ? (mh - sc * m) / a : (mh - m) / a;
        lb[L + (nt - 1) + (k - 1)] = (sc > 0.0) ? (sc - 1.0) / (2.0 * a) : 0.0;
      }
    }
  }
  if (threadIdx.x == 0) {
    iters[b] = bad ? SNAP_ST_NONFINITE : 1;
    if (stats) {
      long long* st = stats + (size_t)b * SNAP_STAT_COUNT;
      st[SNAP_STAT_LINEARISATIONS] = 1; st[SNAP_STAT_PASSES] = 2;
      st[SNAP_STAT_ROWS_READ] = 2 * nt; st[SNAP_STAT_ROWS_WRITTEN] = nt;      // w_hat twice (second time from L2), u* once
      st[SNAP_STAT_VARIANT] = SNAP_VAR_NS_CLOSED_FORM; st[SNAP_STAT_INNER] = 0;
      st[SNAP_STAT_ROW_DOUBLES] = L; st[SNAP_STAT_BACKTRACKS] = 0;
    }
  }
}

// h(w) in the row layout [IC ny nx][total vorticity nt-1][enstrophy nt-1] and the norms
// [||h||_inf, ||h_IC||_2, 0, ||h_vorticity||_2, ||h_enstrophy||_2]  (the mass / energy slots of snap_residual)
__global__ void __launch_bounds__(kMiscThreads) ns_residual_kernel(const __grid_constant__ DevParams P, int batch,
                                                                  const double* __restrict__ u,
                                                                  const double* __restrict__ cdata, double* __restrict__ h,
                                                                  double* __restrict__ norms) {
  __shared__ double red[32];
  const int b = blockIdx.x;
  if (b >= batch) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int L = P.lvl, nt = P.nt;
  const double a = P.dx * P.dy;
  const double* ub = u + (size_t)b * P.n;
  const double* w0 = cdata + (size_t)b * L;
  double* hb = h ? h + (size_t)b * P.m : nullptr;
  double s1 = 0.0, s2 = 0.0;
  for (int c = threadIdx.x; c < L; c += blockDim.x) { s1 += w0[c]; s2 = fma(w0[c], w0[c], s2); }
  const double S1 = block_reduce(s1, red, false), S2 = block_reduce(s2, red, false);
  double hinf = 0.0, n_ic = 0.0, n_v = 0.0, n_z = 0.0;
  for (int c = threadIdx.x; c < L; c += blockDim.x) {
    const double rr = ub[c] - w0[c];
    if (hb) hb[c] = rr;
    n_ic = fma(rr, rr, n_ic);
    hinf = fmax(hinf, finite_d(rr) ? fabs(rr) : 1.7976931348623157e308);
  }
  for (int k = 1 + warp; k < nt; k += nw) {
    const double* row = ub + (size_t)k * L;
    double t1 = 0.0, t2 = 0.0;
    for (int c = lane; c < L; c += 32) { t1 += row[c]; t2 = fma(row[c], row[c], t2); }
    const double hv = a * (warp_sum(t1) - S1), hz = a * (warp_sum(t2) - S2);
    if (lane == 0) {
      if (hb) { hb[L + (k - 1)] = hv; hb[L + (nt - 1) + (k - 1)] = hz; }
      n_v = fma(hv, hv, n_v);
      n_z = fma(hz, hz, n_z);
      hinf = fmax(hinf, finite_d(hv) ? fabs(hv) : 1.7976931348623157e308);
      hinf = fmax(hinf, finite_d(hz) ? fabs(hz) : 1.7976931348623157e308);
    }
  }
  hinf = block_reduce(hinf, red, true);
  n_ic = block_reduce(n_ic, red, false);
  n_v = block_reduce(n_v, red, false);
  n_z = block_reduce(n_z, red, false);
  if (norms && threadIdx.x == 0) {
    double* nb = norms + (size_t)b * 5;
    nb[0] = hinf; nb[1] = sqrt(n_ic); nb[2] = 0.0; nb[3] = sqrt(n_v); nb[4] = sqrt(n_z);
  }
}

}  // namespace snap
