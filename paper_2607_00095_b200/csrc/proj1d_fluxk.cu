// Kind 5 (BURGERS1D_FLUXK) kernel instantiations: nx = 32 Q, Lax-Friedrichs or Godunov flux rows.
#include "kernels_1d_fluxk.cuh"

namespace snap {

// h(u) of kind 5 and [||h||_inf, ||h_IC||_2, ||h_flux||_2, ||h_mass||_2, ||h_energy||_2] (Eq. 27);
// one CTA per sample, warps take the levels round-robin, plain global loads.
template <int FLUX>
__global__ void __launch_bounds__(256) residual_fluxk_kernel(const __grid_constant__ DevParams P, int batch,
                                                             const double* __restrict__ u,
                                                             const double* __restrict__ cdata, double* __restrict__ h,
                                                             double* __restrict__ norms) {
  __shared__ double sE[512], sD[512], red[32];
  const int b = blockIdx.x;
  if (b >= batch) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int nx = P.nx, nt = P.nt, K = P.fk_K, F = nt - 1 - K;
  const double* ub = u + (size_t)b * P.n;
  const double* u0 = cdata + (size_t)b * nx;
  double* hb = h ? h + (size_t)b * P.m : nullptr;
  const size_t loc = (size_t)(K + 1) * nx;
  auto bsum = [&](double v) {
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    double r = (lane < nw) ? red[lane] : 0.0;
    return warp_sum(r);
  };
  auto bmax = [&](double v) {
    v = warp_max(v);
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    double r = (lane < nw) ? red[lane] : 0.0;
    return warp_max(r);
  };
  double s0 = 0.0;
  for (int i = threadIdx.x; i < nx; i += blockDim.x) s0 += u0[i];
  const double M0 = P.dx * bsum(s0);
  double hinf = 0.0, s_ic = 0.0, s_pde = 0.0, s_mass = 0.0, s_en = 0.0;
  auto track = [&](double r) { hinf = fmax(hinf, finite_d(r) ? fabs(r) : 1.7976931348623157e308); };
  for (int k = warp; k < nt; k += nw) {
    const double* uk = ub + (size_t)k * nx;
    double sm = 0.0, s2 = 0.0, sd = 0.0;
    for (int c = lane; c < nx; c += 32) {
      const int ip = (c + 1 == nx) ? 0 : c + 1, im = (c == 0) ? nx - 1 : c - 1;
      const double v = uk[c];
      sm += v;
      s2 = fma(v, v, s2);
      const double dv = uk[ip] - v;
      sd = fma(dv, dv, sd);
      if (k == 0) {
        const double r = v - u0[c];
        s_ic = fma(r, r, s_ic);
        track(r);
        if (hb) hb[c] = r;
      } else if (k <= K) {
        const double* up = uk - nx;
        const double a = up[c], ar = up[ip], al = up[im];
        double Fr, Fl, G;
        flux_lin<FLUX>(a, ar, 0.0, 0.0, P.fk_alpha, Fr, G);
        flux_lin<FLUX>(al, a, 0.0, 0.0, P.fk_alpha, Fl, G);
        const double r = v - (a - P.fk_s * (Fr - Fl) + P.fk_c * ((ar - a) + (al - a)));
        s_pde = fma(r, r, s_pde);
        track(r);
        if (hb) hb[(size_t)k * nx + c] = r;
      }
    }
    sm = warp_sum(sm); s2 = warp_sum(s2); sd = warp_sum(sd);
    if (lane == 0) { sE[k] = 0.5 * P.dx * s2; sD[k] = sd / P.dx; }
    if (k > K && lane == 0) {
      const double hm = P.dx * sm - M0;
      s_mass = fma(hm, hm, s_mass);
      track(hm);
      if (hb) hb[loc + (k - K - 1)] = hm;
    }
  }
  __syncthreads();
  if (P.fk_energy) {
    for (int f = threadIdx.x; f < F; f += blockDim.x) {
      const int k = K + f;
      const double he = (sE[k + 1] - sE[k]) + P.fk_dtnu * sD[k];
      s_en = fma(he, he, s_en);
      track(he);
      if (hb) hb[loc + F + f] = he;
    }
  }
  hinf = bmax(hinf);
  s_ic = bsum(s_ic); s_pde = bsum(s_pde); s_mass = bsum(s_mass); s_en = bsum(s_en);
  if (norms && threadIdx.x == 0) {
    double* nb = norms + (size_t)b * 5;
    nb[0] = hinf; nb[1] = sqrt(s_ic); nb[2] = sqrt(s_pde); nb[3] = sqrt(s_mass); nb[4] = sqrt(s_en);
  }
}

int launch_residual_fluxk(const DevParams& P, int batch, const double* u, const double* cdata, double* h, double* norms,
                          cudaStream_t st) {
  if (P.fk_flux == FLUX_GODUNOV) residual_fluxk_kernel<FLUX_GODUNOV><<<batch, 256, 0, st>>>(P, batch, u, cdata, h, norms);
  else residual_fluxk_kernel<FLUX_LF><<<batch, 256, 0, st>>>(P, batch, u, cdata, h, norms);
  return cudaGetLastError() == cudaSuccess ? SNAP_OK : SNAP_ECUDA;
}

template <int Q>
static int launch_fluxk_q(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st) {
  const bool god = a.P.fk_flux == FLUX_GODUNOV;
  if (a.P.fk_hess) {   // exact Lagrangian Hessian on the free levels (only meaningful with energy rows)
    return god ? launch_fluxk_variant<Q, FLUX_GODUNOV, true>(a, pl, st) : launch_fluxk_variant<Q, FLUX_LF, true>(a, pl, st);
  }
  return god ? launch_fluxk_variant<Q, FLUX_GODUNOV, false>(a, pl, st) : launch_fluxk_variant<Q, FLUX_LF, false>(a, pl, st);
}

int launch_project1d_fluxk(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st) {
  switch (a.P.nx) {
    case 32: return launch_fluxk_q<1>(a, pl, st);
    case 64: return launch_fluxk_q<2>(a, pl, st);
    case 128: return launch_fluxk_q<4>(a, pl, st);
    case 256: return launch_fluxk_q<8>(a, pl, st);
  }
  return SNAP_EINVAL;
}

}  // namespace snap
