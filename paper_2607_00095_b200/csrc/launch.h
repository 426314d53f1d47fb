// Host-side launch interfaces between the translation units of libsnap (not part of the C ABI).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include "snap_internal.h"

namespace snap {

// doubles of the exchange slots of a fused group: [parity][warp][8] (sweeps) or [parity][warp][JT][4] (forward passes)
#ifdef __CUDACC__
__host__ __device__
#endif
constexpr int fused_xch_doubles(int W, int JT) { return 2 * W * (4 * JT > 8 ? 4 * JT : 8); }

// PCFM step arguments handed through the launch layers (null = plain projection)
struct FlowArgs {
  const double* vel;
  const double* u_prior;
  double* u_next;
  double omt, taun;
};


// buffers of the fused path addressed through tensor maps (one row = one box)
enum { TM_UHAT = 0, TM_BUFA = 1, TM_BUFB = 2, TM_USTAR = 3, TM_LAM = 4, TM_VEL = 5, TM_COUNT = 6 };

struct Proj1dArgs {
  alignas(64) CUtensorMap tm[TM_COUNT];   // fused path only: [sample][line of 16 doubles][16], 128-byte swizzle
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
  long long* stats;  // [batch][SNAP_STAT_COUNT]  work counters (snap_project_stats)
  int variant;       // SNAP_VAR_* recorded in the stats
  // PCFM step fused around the projection (snap_flow_step; Eq. 1, 3): all null / 0 for a plain projection
  const double* vel;      // [batch][n] velocity values: the first pass forms u_hat = u_tau + omt * vel (in place in u_hat)
  const double* u_prior;  // [batch][n] prior sample u_0 of the OT interpolant
  double* u_next;         // [batch][n] out: u_0 + taun (u* - u_0)
  double omt, taun;       // 1 - tau, tau'
  int fuse;      // cap on Gauss-Newton iterations per forward pass (0 = as many as the kernel supports)
  int nst;       // ring depth (levels in flight per warp)
  int rp;        // shared-memory row pitch in doubles (even; nx + halo + padding)
  int warp_bytes;
};

struct Plan1d {
  int q, wpc, nst, rp, warp_bytes, grid;
  int wps;       // fused path: warps per sample
  bool full;  // nx == 32 q: no bounds checks in the sweeps
  bool tma;   // every row start is 16-byte aligned: bulk (TMA) copies; otherwise plain loads/stores
  size_t smem;
};

constexpr int kPcgVectors = 8;  // 2D workspace n-vectors per sample: bufA bufB b r z p q y

// proj1d_burgers.cu / proj1d_fisher.cu / proj2d.cu (separate translation units, compiled in parallel)
int launch_project1d_burgers(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st);
int launch_project1d_fisher(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st);
// proj1d_burgers_fused.cu: nx = 32 q, bulk-copy alignment required; pl.rp / pl.warp_bytes follow plan_fused()
int launch_project1d_burgers_fused(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st);
int fused_row_pitch(int nx);   // padded shared-memory row pitch in doubles
// (warps per sample, cells per lane, iterations per pass, max threads per CTA) of the instantiation for nx
bool fused_variant(int nx, int& W, int& Q, int& JT, int& maxt);
// proj1d_fisher_fused.cu: same for kind 2
int launch_project1d_fisher_fused(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st);
bool fused_variant_fisher(int nx, int& W, int& Q, int& JT, int& maxt);
// proj1d_fluxk.cu: kind 5
int launch_project1d_fluxk(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st);
int launch_residual_fluxk(const DevParams& P, int batch, const double* u, const double* cdata, double* h, double* norms,
                          cudaStream_t st);
int launch_project2d(snap_problem* p, int batch, const double* u_hat, const double* cdata, double* u_star,
                     double* lambda, int* iters, int warm, void* workspace, long long* stats, cudaStream_t st);

// proj1d_f32.cu: Float32 mode of the Burgers kinds (multiplier-free)
int launch_project1d_f32(snap_problem* p, int batch, const float* u_hat, const float* cdata, float* u_star, int* iters,
                         float tol, void* workspace, cudaStream_t st);
// proj2d_direct.cu: product-form path of kind 3; returns +1 when the shape / parameters / alignment are outside it
int launch_project2d_direct(snap_problem* p, int batch, const double* u_hat, const double* cdata, double* u_star,
                            double* lambda, int* iters, void* workspace, long long* stats, const FlowArgs* flow,
                            cudaStream_t st);

}  // namespace snap
