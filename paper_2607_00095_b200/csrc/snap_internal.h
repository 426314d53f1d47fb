// Internal declarations shared by the translation units of libsnap (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/snap.h"

namespace snap {

constexpr int kWarp = 32;
constexpr int kHostChunksMax = 16;   // snap_project_host pipelines the batch in at most this many chunks
constexpr double kPolishSkip = 1e-3;  // polish skipped when ||h||_inf <= kPolishSkip * tol
// l1-merit penalty parameter (R2; Nocedal-Wright Eq. 18.36 with sigma = 1, Hessian of f = I):
//   mu <- max(mu, kMuFloor, (w^T d + 1/2 ||d||^2) / ((1 - kMuRho) ||h||_1))   -- needs no multiplier
constexpr double kMuRho = 0.5;
constexpr double kMuFloor = 1e-3;

// Plain-old-data copy of everything a kernel needs; passed by value as a __grid_constant__.
struct DevParams {
  int kind, nx, ny, nt;
  int lvl;        // nx * ny cells per level
  int n;          // unknowns per sample
  int m;          // constraint rows per sample
  int has_mass;   // kinds 0 and 4
  double dx, dy, dt;
  // Burgers (kinds 1, 4):  Phi(v)_i = a0 v_i + (v_{i+1}+v_{i-1}) (e - qs (v_{i+1}-v_{i-1}))
  double bs_e, bs_a0, bs_qs, bs_hs;   // e = s alpha/2 + nu dt/dx^2 ; a0 = 1-2e ; qs = s/4 ; hs = s/2
  // Fisher (kind 2): T = I - dt D Lap_h - dt rho diag(1-2u)
  double fi_a, fi_dtrho;              // a = dt D / dx^2
  // Allen-Cahn (kind 3): T = I - dt eps^2 Lap_h + dt diag(3u^2-1)
  double ac_ax, ac_ay;                // dt eps^2 / dx^2 , dt eps^2 / dy^2
  // kind 5 (BURGERS1D_FLUXK): K flux steps, energy rows on/off, flux kind; s = dt/dx, c = nu dt/dx^2,
  // cD = 2 dt nu / dx, dtnu = dt nu
  int fk_K, fk_energy, fk_flux, fk_hess;   // fk_hess: exact Lagrangian Hessian on the free levels (snap_params::hessian)
  double fk_s, fk_c, fk_cD, fk_dtnu, fk_alpha;
  // solver knobs
  double tol, ls_c1, ls_shrink, pcg_rtol;
  int max_iter, polish, ls_max, pcg_max, precond, lambda_mode;
  // 2D ADI line operator (I - a delta_xx): truncated circulant Green's functions
  int gx_K, gy_K;
  const double* gx;   // device, gx_K+1 taps
  const double* gy;
};

}  // namespace snap

struct snap_problem {
  snap::DevParams dp;
  snap_params params;
  double* d_green;       // device: gx taps then gy taps (2D kind), else nullptr
  // staging for snap_project_host
  void* stage;
  size_t stage_bytes;
  cudaStream_t s_in, s_out;                        // copy streams of snap_project_host (created on first use)
  cudaEvent_t ev_in[snap::kHostChunksMax], ev_k[snap::kHostChunksMax], ev_done;
  long long launches;
  int sm_count;
  int max_smem_optin;
};
