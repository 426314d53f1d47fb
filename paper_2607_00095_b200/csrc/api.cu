// C ABI of libsnap (include/snap.h): validation, handle management, launch configuration.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <new>
#include <vector>

#include "kernels_misc.cuh"
#include "kernels_ns.cuh"
#include "launch.h"
#include "snap_internal.h"

using namespace snap;

namespace {

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

bool is_1d(int kind) { return kind != SNAP_ALLENCAHN2D_IE && kind != SNAP_NS2D_VORT_ENST; }

// Green's function of the cyclic tridiagonal (-a, 1+2a, -a) of size N, truncated where it drops below
// kGreenTol of its peak; g[t], t = 0..K, applied symmetrically (t = -K..K).
// taps of the ADI line solve below this fraction of the peak are dropped: the operator only preconditions,
// and M^{-1} = Jt^{-T} Jt^{-1} stays symmetric positive definite because both sweeps use the same taps
constexpr double kGreenTol = 1e-8;
void circulant_green(double a, int N, std::vector<double>& g) {
  g.clear();
  if (a <= 0.0) { g.push_back(1.0); return; }
  const double b = 1.0 + 2.0 * a;
  const double disc = sqrt(b * b - 4.0 * a * a);
  const double rho = (b - disc) / (2.0 * a);
  const double rhoN = pow(rho, (double)N);
  const int Kmax = N / 2;
  for (int t = 0; t <= Kmax; ++t) {
    const double v = (pow(rho, (double)t) + pow(rho, (double)(N - t))) / ((1.0 - rhoN) * disc);
    g.push_back(v);
    if (t > 0 && v < kGreenTol * g[0]) break;
  }
  const int K = (int)g.size() - 1;
  if (2 * K == N) g[K] *= 0.5;  // offset +K and -K are the same point on an even ring
}

int check_launch(snap_problem* p) {
  p->launches++;
  return cudaGetLastError() == cudaSuccess ? SNAP_OK : SNAP_ECUDA;
}

bool plan_1d(const snap_problem* p, int batch, Plan1d& pl) {
  const int nx = p->dp.nx;
  pl.q = 1;
  while (pl.q * 32 < nx) pl.q *= 2;
  if (pl.q > 16) return false;
  pl.full = (pl.q * 32 == nx);
  pl.rp = ((nx + 1) & ~1) + 4;  // [pad, halo, data(nx), halo, pad], data start 16-byte aligned
  const int sms = p->sm_count > 0 ? p->sm_count : 148;
  int wpc = (batch + sms - 1) / sms;
  if (wpc < 1) wpc = 1;
  if (wpc > 8) wpc = 8;
  const size_t limit = (size_t)p->max_smem_optin;
  for (;; --wpc) {
    for (int nst = 4; nst >= 2; --nst) {
      const size_t wb = align_up((size_t)(3 * nst + 5) * pl.rp * 8 + (size_t)nst * 8, 128);
      if (wb * wpc <= limit) {
        pl.wpc = wpc; pl.nst = nst; pl.warp_bytes = (int)wb; pl.smem = wb * wpc;
        pl.grid = (batch + wpc - 1) / wpc;
        return true;
      }
    }
    if (wpc == 1) return false;
  }
}

// fused Burgers path: nx = 32 W Q, padded rows; per sample a ring of nst x 2 input rows + 4 output rows,
// exchange slots, reduction scratch and mbarriers.  pl.wpc = samples per CTA, pl.warp_bytes = bytes per sample.
bool plan_fused(const snap_problem* p, int batch, Plan1d& pl) {
  const int nx = p->dp.nx;
  int W, Q, JT, maxt;
  const bool fisher = p->dp.kind == SNAP_FISHER1D_IE;
  if (!(fisher ? fused_variant_fisher(nx, W, Q, JT, maxt) : fused_variant(nx, W, Q, JT, maxt))) return false;
  pl.wps = W;
  pl.q = Q; pl.full = true; pl.tma = true;
  pl.rp = fused_row_pitch(nx);
  const int sms = p->sm_count > 0 ? p->sm_count : 148;
  int spc = (batch + sms - 1) / sms;      // samples per CTA: one wave over the SMs when possible
  const int spc_max = maxt / (32 * W) < 15 ? maxt / (32 * W) : 15;   // named barriers 1..15
  if (spc < 1) spc = 1;
  if (spc > spc_max) spc = spc_max;
  const size_t limit = (size_t)p->max_smem_optin;
  for (;; --spc) {
    for (int nst = 4; nst >= 2; --nst) {   // deeper rings measured no faster
      // ring + output staging rows (W > 1) + exchange slots + reduction scratch + mass-row level sums (W = 1,
      // JT x 8 levels x 34) + suffix sums of the min-norm correction (W = 1) + mbarriers
      const size_t sb = align_up(((size_t)(2 * nst + (W > 1 ? 4 : 0)) * pl.rp + fused_xch_doubles(W, JT) + W * 24 +
                                  W * JT * 8 * 34 + (W > 1 ? 2 * W * JT * 8 : 0) +
                                  (W == 1 ? (p->dp.nt < 512 ? p->dp.nt : 512) : 0) + nst + 1) * 8, 1024);
      if (sb * spc + 1024 <= limit) {
        pl.wpc = spc; pl.nst = nst; pl.warp_bytes = (int)sb; pl.smem = sb * spc + 1024;
        pl.grid = (batch + spc - 1) / spc;
        return true;
      }
    }
    if (spc == 1) return false;
  }
}

// Tensor map of a [batch][n (+ tail)] fp64 buffer seen as [sample][line of 16 doubles][16]; one TMA box = the
// `box_lines` lines of (a warp's part of) one row, stored in shared memory with the 128-byte swizzle.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      f = nullptr;
    return reinterpret_cast<EncodeTiledFn>(f);
  }();
  return fn;
}
bool make_row_map(CUtensorMap* tm, const void* base, int batch, size_t n, size_t sample_stride_doubles, int box_lines) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  const cuuint64_t dims[3] = {16, (cuuint64_t)(n / 16), (cuuint64_t)batch};
  const cuuint64_t strides[2] = {128, (cuuint64_t)sample_stride_doubles * 8};
  const cuuint32_t box[3] = {16, (cuuint32_t)box_lines, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

size_t aux_bytes(const snap_problem* p, size_t B) { return align_up(B * 2 * (size_t)p->dp.nt * 8, 256); }
// every workspace starts (after alignment to 256 bytes) with the per-sample work counters [B][SNAP_STAT_COUNT]
size_t stats_bytes(size_t B) { return align_up(B * 8 * SNAP_STAT_COUNT, 256); }
unsigned char* ws_base(const void* workspace) {
  return reinterpret_cast<unsigned char*>(align_up(reinterpret_cast<uintptr_t>(workspace), 256));
}

bool aligned16(const void* q) { return (reinterpret_cast<uintptr_t>(q) & 15u) == 0; }

// kind 5: one warp per sample; per sample a ring of nst x 2 swizzled rows, the band system (11 doubles per free
// level) and the mbarriers
int project_fluxk(snap_problem* p, int batch, const double* u_hat, const double* cdata, double* u_star, double* lambda,
                  int* iters, unsigned char* w, long long* stats, cudaStream_t st) {
  const DevParams& d = p->dp;
  if (!(aligned16(u_hat) && aligned16(u_star) && aligned16(w))) return SNAP_EINVAL;   // TMA rows
  const int F = d.nt - 1 - d.fk_K;
  const int rp = fused_row_pitch(d.nx);
  const int sms = p->sm_count > 0 ? p->sm_count : 148;
  int spc = (batch + sms - 1) / sms;
  if (spc < 1) spc = 1;
  if (spc > 8) spc = 8;
  Plan1d pl;
  bool found = false;
  for (; spc >= 1 && !found; --spc) {
    for (int nst = 4; nst >= 2; --nst) {
      const size_t sb = align_up(((size_t)2 * nst * rp + (size_t)12 * (F > 0 ? F : 1) + nst) * 8, 1024);
      if (sb * spc + 1024 <= (size_t)p->max_smem_optin) {
        pl.wpc = spc; pl.nst = nst; pl.warp_bytes = (int)sb; pl.smem = sb * spc + 1024;
        pl.grid = (batch + spc - 1) / spc;
        found = true;
        break;
      }
    }
  }
  if (!found) return SNAP_EINVAL;
  Proj1dArgs a;
  a.P = d;
  a.batch = batch; a.warm = 0;
  a.u_hat = u_hat; a.cdata = cdata; a.u_star = u_star; a.lam = lambda; a.iters = iters;   // fused path: NULL = no multipliers
  const size_t field = align_up((size_t)batch * d.n * 8, 256);
  a.bufA = reinterpret_cast<double*>(w);
  a.bufB = reinterpret_cast<double*>(w + field);
  a.aux = reinterpret_cast<double*>(w + 2 * field);
  a.stats = stats;
  a.fuse = 0;
  a.vel = nullptr; a.u_prior = nullptr; a.u_next = nullptr; a.omt = 0.0; a.taun = 0.0;
  const int box = d.nx / 16;
  const size_t n = (size_t)d.n;
  if (!(make_row_map(&a.tm[TM_UHAT], u_hat, batch, n, n, box) && make_row_map(&a.tm[TM_BUFA], a.bufA, batch, n, n, box) &&
        make_row_map(&a.tm[TM_BUFB], a.bufB, batch, n, n, box) && make_row_map(&a.tm[TM_USTAR], u_star, batch, n, n, box)))
    return SNAP_ECUDA;
  a.tm[TM_LAM] = a.tm[TM_USTAR];   // unused by this kind
  a.nst = pl.nst; a.rp = rp; a.warp_bytes = pl.warp_bytes;
  a.variant = SNAP_VAR_FLUXK_BAND;
  p->launches++;
  return launch_project1d_fluxk(a, pl, st);
}

}  // namespace

extern "C" {

void snap_params_default(snap_params* p) {
  if (!p) return;
  memset(p, 0, sizeof(*p));
  p->dx = p->dy = p->dt = 1.0;
  p->alpha = 1.0;
  p->tol = 1e-10;
  p->max_iter = 50;
  p->polish = 1;
  p->ls_c1 = 1e-4;
  p->ls_shrink = 0.5;
  p->ls_max = 20;
  p->pcg_rtol = 1e-13;
  p->pcg_max = 200;
  p->precond = 2;
  p->lambda_mode = 0;
  p->gn_fuse = 0;
  p->flux_steps = 0;
  p->energy_rows = 0;
  p->flux_kind = 0;
  p->hessian = 0;
}

int snap_problem_create(snap_problem** out, int kind, int nx, int ny, int nt, const snap_params* prm) {
  if (!out || !prm) return SNAP_EINVAL;
  if (kind < SNAP_HEAT1D_IC_MASS || kind > SNAP_NS2D_VORT_ENST) return SNAP_EINVAL;
  if (kind == SNAP_NS2D_VORT_ENST && nt > kNsMaxLevels) return SNAP_EINVAL;
  if (kind == SNAP_BURGERS1D_FLUXK) {
    if (!(nx == 32 || nx == 64 || nx == 128 || nx == 256) || nt > 512) return SNAP_EINVAL;
    if (prm->flux_steps < 0 || prm->flux_steps > nt - 1) return SNAP_EINVAL;
    if (prm->energy_rows < 0 || prm->energy_rows > 1 || prm->flux_kind < 0 || prm->flux_kind > 1) return SNAP_EINVAL;
  }
  if (is_1d(kind)) {
    if (ny != 1 || nx < 2 || nx > 512 || nt < 2 || nt > 65535) return SNAP_EINVAL;
  } else {
    if (nx < 4 || ny < 4 || (long long)nx * ny > 4096 || nt < 2 || nt > 65535) return SNAP_EINVAL;
  }
  if (!(prm->dx > 0.0) || !(prm->dt > 0.0) || !(prm->tol > 0.0)) return SNAP_EINVAL;
  if (!is_1d(kind) && !(prm->dy > 0.0)) return SNAP_EINVAL;
  if (prm->max_iter < 0 || prm->polish < 0 || prm->ls_max < 0 || prm->pcg_max < 1) return SNAP_EINVAL;
  if (!(prm->ls_shrink > 0.0 && prm->ls_shrink < 1.0) || !(prm->ls_c1 > 0.0 && prm->ls_c1 < 1.0)) return SNAP_EINVAL;
  if (prm->gn_fuse < -1 || prm->gn_fuse > 64) return SNAP_EINVAL;
  if (prm->precond < 0 || prm->precond > 2 || prm->lambda_mode < 0 || prm->lambda_mode > 1) return SNAP_EINVAL;
  if (prm->hessian < 0 || prm->hessian > 1) return SNAP_EINVAL;

  snap_problem* p = new (std::nothrow) snap_problem();
  if (!p) return SNAP_ENOMEM;
  memset(p, 0, sizeof(*p));
  p->params = *prm;
  DevParams& d = p->dp;
  d.kind = kind; d.nx = nx; d.ny = ny; d.nt = nt;
  d.lvl = nx * ny;
  d.n = d.lvl * nt;
  d.has_mass = (kind == SNAP_HEAT1D_IC_MASS || kind == SNAP_BURGERS1D_LF_MASS);
  d.m = (kind == SNAP_HEAT1D_IC_MASS) ? nx + nt : d.n + (d.has_mass ? nt : 0);
  if (kind == SNAP_NS2D_VORT_ENST) d.m = d.lvl + 2 * (nt - 1);
  if (kind == SNAP_BURGERS1D_FLUXK) {
    d.fk_K = prm->flux_steps; d.fk_energy = prm->energy_rows; d.fk_flux = prm->flux_kind;
    d.fk_hess = (prm->hessian == 1 && prm->energy_rows == 1) ? 1 : 0;
    const int F = nt - 1 - d.fk_K;
    d.m = (d.fk_K + 1) * nx + F + (d.fk_energy ? F : 0);
    d.fk_s = prm->dt / prm->dx;
    d.fk_c = prm->nu * prm->dt / (prm->dx * prm->dx);
    d.fk_cD = 2.0 * prm->dt * prm->nu / prm->dx;
    d.fk_dtnu = prm->dt * prm->nu;
    d.fk_alpha = prm->alpha;
  }
  d.dx = prm->dx; d.dy = prm->dy; d.dt = prm->dt;
  const double s = prm->dt / prm->dx;
  d.bs_e = 0.5 * s * prm->alpha + prm->nu * prm->dt / (prm->dx * prm->dx);
  d.bs_a0 = 1.0 - 2.0 * d.bs_e;
  d.bs_qs = 0.25 * s;
  d.bs_hs = 0.5 * s;
  d.fi_a = prm->dt * prm->D / (prm->dx * prm->dx);
  d.fi_dtrho = prm->dt * prm->rho;
  d.ac_ax = prm->dt * prm->eps * prm->eps / (prm->dx * prm->dx);
  d.ac_ay = is_1d(kind) ? 0.0 : prm->dt * prm->eps * prm->eps / (prm->dy * prm->dy);
  d.tol = prm->tol; d.ls_c1 = prm->ls_c1; d.ls_shrink = prm->ls_shrink; d.pcg_rtol = prm->pcg_rtol;
  d.max_iter = prm->max_iter; d.polish = prm->polish; d.ls_max = prm->ls_max; d.pcg_max = prm->pcg_max;
  d.precond = prm->precond; d.lambda_mode = prm->lambda_mode;

  int dev = 0;
  if (cudaGetDevice(&dev) == cudaSuccess) {
    cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&p->max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  }
  if (p->sm_count <= 0) p->sm_count = 148;
  if (p->max_smem_optin <= 0) p->max_smem_optin = 227 * 1024;

  if (kind == SNAP_ALLENCAHN2D_IE) {
    std::vector<double> gx, gy;
    circulant_green(d.ac_ax, nx, gx);
    circulant_green(d.ac_ay, ny, gy);
    d.gx_K = (int)gx.size() - 1;
    d.gy_K = (int)gy.size() - 1;
    const size_t bytes = (gx.size() + gy.size()) * sizeof(double);
    if (cudaMalloc(&p->d_green, bytes) != cudaSuccess) { delete p; return SNAP_ENOMEM; }
    std::vector<double> both(gx);
    both.insert(both.end(), gy.begin(), gy.end());
    if (cudaMemcpy(p->d_green, both.data(), bytes, cudaMemcpyHostToDevice) != cudaSuccess) {
      cudaFree(p->d_green); delete p; return SNAP_ECUDA;
    }
    d.gx = p->d_green;
    d.gy = p->d_green + gx.size();
  }
  *out = p;
  return SNAP_OK;
}

int snap_problem_destroy(snap_problem* p) {
  if (!p) return SNAP_EINVAL;
  if (p->d_green) cudaFree(p->d_green);
  if (p->stage) cudaFree(p->stage);
  if (p->s_in) {
    cudaStreamDestroy(p->s_in);
    cudaStreamDestroy(p->s_out);
    for (int i = 0; i < kHostChunksMax; ++i) { cudaEventDestroy(p->ev_in[i]); cudaEventDestroy(p->ev_k[i]); }
    cudaEventDestroy(p->ev_done);
  }
  delete p;
  return SNAP_OK;
}

size_t snap_num_unknowns(const snap_problem* p) { return p ? (size_t)p->dp.n : 0; }
size_t snap_num_rows(const snap_problem* p) { return p ? (size_t)p->dp.m : 0; }
long long snap_launch_count(const snap_problem* p) { return p ? p->launches : 0; }

size_t snap_workspace_bytes(const snap_problem* p, int batch) {
  if (!p || batch <= 0) return 0;
  const size_t n = (size_t)p->dp.n, B = (size_t)batch;
  const size_t head = 256 + stats_bytes(B);   // alignment slack + work counters
  // tail: a multiplier array for multiplier-free calls (lambda == NULL) served by a kernel that needs the storage
  const size_t lam_scratch = align_up(B * (size_t)p->dp.m * 8, 256);
  if (p->dp.kind == SNAP_HEAT1D_IC_MASS || p->dp.kind == SNAP_NS2D_VORT_ENST) return head + lam_scratch;
  if (p->dp.kind == SNAP_ALLENCAHN2D_IE) return head + align_up(B * n * 8 * kPcgVectors, 256) + lam_scratch;
  return head + align_up(B * n * 8, 256) * 2 + aux_bytes(p, B) + lam_scratch;
}

namespace {
// Eq. 1 / Eq. 3 as separate elementwise launches (projection kernels that do not fuse them)
int flow_unfused_shoot(snap_problem* p, int batch, const double* u_hat, const FlowArgs* flow, cudaStream_t st) {
  if (!flow) return SNAP_OK;
  const size_t total = (size_t)batch * p->dp.n;
  flow_shoot_kernel<<<p->sm_count * 4, kMiscThreads, 0, st>>>(total, const_cast<double*>(u_hat), flow->vel, flow->omt);
  return check_launch(p);
}
int flow_unfused_pullback(snap_problem* p, int batch, const double* u_star, const FlowArgs* flow, cudaStream_t st) {
  if (!flow) return SNAP_OK;
  const size_t total = (size_t)batch * p->dp.n;
  flow_pullback_kernel<<<p->sm_count * 4, kMiscThreads, 0, st>>>(total, u_star, flow->u_prior, flow->u_next, flow->taun);
  return check_launch(p);
}
}  // namespace

static int project_impl(const snap_problem* cp, int batch, const double* u_hat, const double* cdata, double* u_star,
                        double* lambda, int* iters, int warm, void* workspace, size_t workspace_bytes, snap_stream stream,
                        const FlowArgs* flow) {
  snap_problem* p = const_cast<snap_problem*>(cp);
  if (!p || batch < 0) return SNAP_EINVAL;
  if (batch == 0) return SNAP_OK;
  if (!u_hat || !cdata || !u_star || !iters || !workspace) return SNAP_EINVAL;
  const size_t need = snap_workspace_bytes(p, batch);
  if (workspace_bytes < need) return SNAP_ENOMEM;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const DevParams& d = p->dp;
  unsigned char* w = ws_base(workspace);
  long long* stats = reinterpret_cast<long long*>(w);
  // multiplier-free call (lambda == NULL): the product-form kernels skip the multiplier work; the other kernels keep
  // their multipliers in the tail of the workspace
  double* const lam_scratch = reinterpret_cast<double*>(w + (need - 256) - align_up((size_t)batch * d.m * 8, 256));
  double* const lam_any = lambda ? lambda : lam_scratch;
  w += stats_bytes((size_t)batch);
  if (d.kind == SNAP_HEAT1D_IC_MASS) {
    int rc = flow_unfused_shoot(p, batch, u_hat, flow, st);
    if (rc != SNAP_OK) return rc;
    heat_project_kernel<<<batch, kMiscThreads, 0, st>>>(d, batch, u_hat, cdata, u_star, lam_any, iters, stats);
    rc = check_launch(p);
    return rc != SNAP_OK ? rc : flow_unfused_pullback(p, batch, u_star, flow, st);
  }
  if (d.kind == SNAP_NS2D_VORT_ENST) {     // closed form per level; lambda == NULL: the multipliers are simply not written
    int rc = flow_unfused_shoot(p, batch, u_hat, flow, st);
    if (rc != SNAP_OK) return rc;
    ns_project_kernel<<<batch, kMiscThreads, 0, st>>>(d, batch, u_hat, cdata, u_star, lambda, iters, stats);
    rc = check_launch(p);
    return rc != SNAP_OK ? rc : flow_unfused_pullback(p, batch, u_star, flow, st);
  }
  if (d.kind == SNAP_ALLENCAHN2D_IE) {
    if (p->params.gn_fuse >= 0) {   // product-form path (in-SMEM level solves) where the shape and parameters allow it
      const int rc = launch_project2d_direct(p, batch, u_hat, cdata, u_star, lambda, iters, w, stats, flow, st);
      if (rc <= 0) return rc;
    }
    int rc = flow_unfused_shoot(p, batch, u_hat, flow, st);
    if (rc != SNAP_OK) return rc;
    rc = launch_project2d(p, batch, u_hat, cdata, u_star, lam_any, iters, lambda ? warm : 0, w, stats, st);
    return rc != SNAP_OK ? rc : flow_unfused_pullback(p, batch, u_star, flow, st);
  }

  if (d.kind == SNAP_BURGERS1D_FLUXK) {
    int rc = flow_unfused_shoot(p, batch, u_hat, flow, st);
    if (rc != SNAP_OK) return rc;
    rc = project_fluxk(p, batch, u_hat, cdata, u_star, lam_any, iters, w, stats, st);
    return rc != SNAP_OK ? rc : flow_unfused_pullback(p, batch, u_star, flow, st);
  }
  Plan1d pl;
  if (!plan_1d(p, batch, pl)) return SNAP_EINVAL;
  Proj1dArgs a;
  a.P = d;
  a.batch = batch; a.warm = warm;
  a.u_hat = u_hat; a.cdata = cdata; a.u_star = u_star; a.lam = lambda; a.iters = iters;   // fused path: NULL = no multipliers
  const size_t field = align_up((size_t)batch * d.n * 8, 256);
  a.bufA = reinterpret_cast<double*>(w);
  a.bufB = reinterpret_cast<double*>(w + field);
  a.aux = reinterpret_cast<double*>(w + 2 * field);
  a.stats = stats;
  a.fuse = p->params.gn_fuse;
  a.vel = nullptr; a.u_prior = nullptr; a.u_next = nullptr; a.omt = 0.0; a.taun = 0.0;
  // bulk (TMA) copies need every row start 16-byte aligned
  const bool bulk_ok = (d.nx % 2 == 0) && (d.m % 2 == 0 || batch == 1) && aligned16(u_hat) && aligned16(u_star) &&
                       aligned16(lam_any) && aligned16(a.bufA);
  if (p->params.gn_fuse >= 0 && bulk_ok) {
    Plan1d pf;
    if (plan_fused(p, batch, pf)) {
      const int box = d.nx / 16 / pf.wps;
      const size_t n = (size_t)d.n;
      const bool ok = make_row_map(&a.tm[TM_UHAT], u_hat, batch, n, n, box) &&
                      make_row_map(&a.tm[TM_BUFA], a.bufA, batch, n, n, box) &&
                      make_row_map(&a.tm[TM_BUFB], a.bufB, batch, n, n, box) &&
                      make_row_map(&a.tm[TM_USTAR], u_star, batch, n, n, box) &&
                      make_row_map(&a.tm[TM_LAM], lam_any, batch, n, (size_t)d.m, box);
      // PCFM step: one warp per sample fuses Eq. 1 into the first pass and Eq. 3 into the multiplier sweep
      const bool fuse_flow = flow && pf.wps == 1 && aligned16(flow->vel) && aligned16(flow->u_prior) && aligned16(flow->u_next);
      bool okf = ok;
      if (okf && fuse_flow) okf = make_row_map(&a.tm[TM_VEL], flow->vel, batch, n, n, box);
      if (okf && (!flow || fuse_flow)) {
        if (flow) { a.vel = flow->vel; a.u_prior = flow->u_prior; a.u_next = flow->u_next; a.omt = flow->omt; a.taun = flow->taun; }
        a.nst = pf.nst; a.rp = pf.rp; a.warp_bytes = pf.warp_bytes;
        a.variant = SNAP_VAR_FUSED_TMA;
        p->launches++;
        return d.kind == SNAP_FISHER1D_IE ? launch_project1d_fisher_fused(a, pf, st)
                                          : launch_project1d_burgers_fused(a, pf, st);
      }
    }
  }
  a.nst = pl.nst; a.rp = pl.rp; a.warp_bytes = pl.warp_bytes;
  a.lam = lam_any;            // the classic sweeps carry the multipliers in every iteration
  pl.tma = bulk_ok;
  if (!pl.tma) pl.full = false;  // the plain-load path is only instantiated with bounds checks
  a.variant = pl.tma ? SNAP_VAR_CLASSIC_BULK : SNAP_VAR_CLASSIC_PLAIN;
  int rc = flow_unfused_shoot(p, batch, u_hat, flow, st);
  if (rc != SNAP_OK) return rc;
  p->launches++;
  rc = (d.kind == SNAP_FISHER1D_IE) ? launch_project1d_fisher(a, pl, st) : launch_project1d_burgers(a, pl, st);
  return rc != SNAP_OK ? rc : flow_unfused_pullback(p, batch, u_star, flow, st);
}

int snap_project(const snap_problem* p, int batch, const double* u_hat, const double* cdata, double* u_star,
                 double* lambda, int* iters, int warm, void* workspace, size_t workspace_bytes, snap_stream stream) {
  return project_impl(p, batch, u_hat, cdata, u_star, lambda, iters, warm, workspace, workspace_bytes, stream, nullptr);
}

int snap_project_f32(const snap_problem* cp, int batch, const float* u_hat, const float* cdata, float* u_star, int* iters,
                     float tol, void* workspace, size_t workspace_bytes, snap_stream stream) {
  snap_problem* p = const_cast<snap_problem*>(cp);
  if (!p || batch < 0) return SNAP_EINVAL;
  if (batch == 0) return SNAP_OK;
  if (!u_hat || !cdata || !u_star || !iters || !workspace || !(tol > 0.0f)) return SNAP_EINVAL;
  const DevParams& d = p->dp;
  if (d.kind != SNAP_BURGERS1D_LF && d.kind != SNAP_BURGERS1D_LF_MASS) return SNAP_EINVAL;
  if (!(d.nx == 32 || d.nx == 64 || d.nx == 128 || d.nx == 256)) return SNAP_EINVAL;
  if (workspace_bytes < snap_workspace_bytes(p, batch)) return SNAP_ENOMEM;
  unsigned char* w = ws_base(workspace) + stats_bytes((size_t)batch);
  if (!(aligned16(u_hat) && aligned16(cdata) && aligned16(u_star) && aligned16(w))) return SNAP_EINVAL;
  return launch_project1d_f32(p, batch, u_hat, cdata, u_star, iters, tol, w, static_cast<cudaStream_t>(stream));
}

int snap_flow_step(const snap_problem* p, int batch, double* u_tau, const double* vel, const double* u_prior, double tau,
                   double tau_next, const double* cdata, double* u1, double* u_next, double* lambda, int* iters,
                   void* workspace, size_t workspace_bytes, snap_stream stream) {
  if (!p || batch < 0) return SNAP_EINVAL;
  if (batch == 0) return SNAP_OK;
  if (!u_tau || !vel || !u_prior || !u1 || !u_next) return SNAP_EINVAL;
  if (!(tau >= 0.0 && tau <= 1.0 && tau_next >= 0.0 && tau_next <= 1.0)) return SNAP_EINVAL;
  // the buffers of a step are distinct: u_tau is overwritten by u_hat_1 while u1 / u_next are being produced
  if (u1 == u_tau || u_next == u_tau || u_next == u1 || u_prior == u_tau || u_prior == u1 || u_prior == u_next ||
      vel == u_tau || vel == u1 || vel == u_next)
    return SNAP_EINVAL;
  FlowArgs f;
  f.vel = vel; f.u_prior = u_prior; f.u_next = u_next; f.omt = 1.0 - tau; f.taun = tau_next;
  return project_impl(p, batch, u_tau, cdata, u1, lambda, iters, 0, workspace, workspace_bytes, stream, &f);
}

int snap_project_host(snap_problem* p, int batch, const double* u_hat_host, const double* cdata_host,
                      double* u_star_host, double* lambda_host, int* iters_host, int warm, snap_stream stream) {
  if (!p || batch < 0) return SNAP_EINVAL;
  if (batch == 0) return SNAP_OK;
  if (!u_hat_host || !cdata_host || !u_star_host || !iters_host) return SNAP_EINVAL;
  if (!lambda_host) warm = 0;   // multiplier-free call: lambda is neither read nor returned
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const DevParams& d = p->dp;
  // The batch is cut into chunks of samples (independent blocks) that flow through three
  // streams: host->device copy of chunk c+1, projection of chunk c and device->host copy of chunk c-1 overlap,
  // so that both directions of the host link are busy at once.
  // (measured on config 5, 2 x 1.07 GB per call: 4 chunks 38.0 k, 8 chunks 40.4 k, 16 chunks 41.4 k projections/s end to end)
  int nchunk = batch >= 1024 ? 16 : (batch >= 512 ? 8 : (batch >= 128 ? 2 : 1));
  const int cb = (batch + nchunk - 1) / nchunk;            // samples per chunk
  nchunk = (batch + cb - 1) / cb;
  const size_t C = (size_t)cb;
  const size_t b_u = align_up(C * d.n * 8, 256), b_c = align_up(C * d.lvl * 8, 256), b_l = align_up(C * d.m * 8, 256),
               b_i = align_up(C * 4, 256), b_w = align_up(snap_workspace_bytes(p, cb), 256);
  const size_t per_chunk = 2 * b_u + b_c + b_l + b_i + b_w;
  const size_t total = per_chunk * nchunk;
  if (p->stage_bytes < total) {
    if (p->stage) cudaFree(p->stage);
    p->stage = nullptr;
    p->stage_bytes = 0;
    if (cudaMalloc(&p->stage, total) != cudaSuccess) return SNAP_ENOMEM;
    p->stage_bytes = total;
  }
  if (!p->s_in) {
    if (cudaStreamCreateWithFlags(&p->s_in, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&p->s_out, cudaStreamNonBlocking) != cudaSuccess)
      return SNAP_ECUDA;
    for (int i = 0; i < kHostChunksMax; ++i)
      if (cudaEventCreateWithFlags(&p->ev_in[i], cudaEventDisableTiming) != cudaSuccess ||
          cudaEventCreateWithFlags(&p->ev_k[i], cudaEventDisableTiming) != cudaSuccess)
        return SNAP_ECUDA;
    if (cudaEventCreateWithFlags(&p->ev_done, cudaEventDisableTiming) != cudaSuccess) return SNAP_ECUDA;
  }
  // order the copy streams after whatever the caller has already enqueued on `stream`
  if (cudaEventRecord(p->ev_done, st) != cudaSuccess || cudaStreamWaitEvent(p->s_in, p->ev_done, 0) != cudaSuccess)
    return SNAP_ECUDA;
  for (int c = 0; c < nchunk; ++c) {
    const int b0 = c * cb, nb = (batch - b0 < cb) ? batch - b0 : cb;
    const size_t B = (size_t)nb;
    unsigned char* s = static_cast<unsigned char*>(p->stage) + (size_t)c * per_chunk;
    double* d_uh = reinterpret_cast<double*>(s);
    double* d_us = reinterpret_cast<double*>(s + b_u);
    double* d_c = reinterpret_cast<double*>(s + 2 * b_u);
    double* d_l = reinterpret_cast<double*>(s + 2 * b_u + b_c);
    int* d_i = reinterpret_cast<int*>(s + 2 * b_u + b_c + b_l);
    void* d_w = s + 2 * b_u + b_c + b_l + b_i;
    bool ok = cudaMemcpyAsync(d_uh, u_hat_host + (size_t)b0 * d.n, B * d.n * 8, cudaMemcpyHostToDevice, p->s_in) == cudaSuccess;
    ok = ok && cudaMemcpyAsync(d_c, cdata_host + (size_t)b0 * d.lvl, B * d.lvl * 8, cudaMemcpyHostToDevice, p->s_in) == cudaSuccess;
    if (warm)
      ok = ok && cudaMemcpyAsync(d_l, lambda_host + (size_t)b0 * d.m, B * d.m * 8, cudaMemcpyHostToDevice, p->s_in) == cudaSuccess;
    ok = ok && cudaEventRecord(p->ev_in[c], p->s_in) == cudaSuccess && cudaStreamWaitEvent(st, p->ev_in[c], 0) == cudaSuccess;
    if (!ok) return SNAP_ECUDA;
    const int rc = snap_project(p, nb, d_uh, d_c, d_us, lambda_host ? d_l : nullptr, d_i, warm, d_w, b_w, stream);
    if (rc != SNAP_OK) return rc;
    ok = cudaEventRecord(p->ev_k[c], st) == cudaSuccess && cudaStreamWaitEvent(p->s_out, p->ev_k[c], 0) == cudaSuccess;
    ok = ok && cudaMemcpyAsync(u_star_host + (size_t)b0 * d.n, d_us, B * d.n * 8, cudaMemcpyDeviceToHost, p->s_out) == cudaSuccess;
    if (lambda_host)
      ok = ok && cudaMemcpyAsync(lambda_host + (size_t)b0 * d.m, d_l, B * d.m * 8, cudaMemcpyDeviceToHost, p->s_out) == cudaSuccess;
    ok = ok && cudaMemcpyAsync(iters_host + b0, d_i, B * 4, cudaMemcpyDeviceToHost, p->s_out) == cudaSuccess;
    if (!ok) return SNAP_ECUDA;
  }
  if (cudaEventRecord(p->ev_done, p->s_out) != cudaSuccess || cudaStreamWaitEvent(st, p->ev_done, 0) != cudaSuccess)
    return SNAP_ECUDA;
  return cudaStreamSynchronize(st) == cudaSuccess ? SNAP_OK : SNAP_ECUDA;
}

int snap_project_stats(const snap_problem* p, int batch, const void* workspace, size_t workspace_bytes,
                       long long* stats, snap_stream stream) {
  if (!p || batch < 0) return SNAP_EINVAL;
  if (batch == 0) return SNAP_OK;
  if (!stats || !workspace) return SNAP_EINVAL;
  if (workspace_bytes < snap_workspace_bytes(p, batch)) return SNAP_ENOMEM;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  return cudaMemcpyAsync(stats, ws_base(workspace), (size_t)batch * 8 * SNAP_STAT_COUNT, cudaMemcpyDeviceToDevice,
                         st) == cudaSuccess ? SNAP_OK : SNAP_ECUDA;
}

int snap_residual(const snap_problem* cp, int batch, const double* u, const double* cdata, double* h, double* norms,
                  snap_stream stream) {
  snap_problem* p = const_cast<snap_problem*>(cp);
  if (!p || batch < 0) return SNAP_EINVAL;
  if (batch == 0) return SNAP_OK;
  if (!u || !cdata || (!h && !norms)) return SNAP_EINVAL;
  if (p->dp.kind == SNAP_BURGERS1D_FLUXK) {
    p->launches++;
    return launch_residual_fluxk(p->dp, batch, u, cdata, h, norms, static_cast<cudaStream_t>(stream));
  }
  if (p->dp.kind == SNAP_NS2D_VORT_ENST) {
    ns_residual_kernel<<<batch, kMiscThreads, 0, static_cast<cudaStream_t>(stream)>>>(p->dp, batch, u, cdata, h, norms);
    return check_launch(p);
  }
  residual_kernel<<<batch, kMiscThreads, 0, static_cast<cudaStream_t>(stream)>>>(p->dp, batch, u, cdata, h, norms);
  return check_launch(p);
}

int snap_schur_apply(const snap_problem* cp, int batch, const double* u, const double* x, double* out, void* workspace,
                     size_t workspace_bytes, snap_stream stream) {
  snap_problem* p = const_cast<snap_problem*>(cp);
  if (!p || batch < 0) return SNAP_EINVAL;
  if (batch == 0) return SNAP_OK;
  if (!u || !x || !out || !workspace) return SNAP_EINVAL;
  if (p->dp.kind >= SNAP_BURGERS1D_FLUXK) return SNAP_EINVAL;   // kinds 0-4 only (include/snap.h)
  if (workspace_bytes < (size_t)batch * p->dp.n * 8) return SNAP_ENOMEM;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  double* g = static_cast<double*>(workspace);
  jt_apply_kernel<<<batch, kMiscThreads, 0, st>>>(p->dp, batch, u, x, g);
  int rc = check_launch(p);
  if (rc != SNAP_OK) return rc;
  j_apply_kernel<<<batch, kMiscThreads, 0, st>>>(p->dp, batch, u, g, out);
  return check_launch(p);
}

// ------------------------------------------------------------------------------------------------------
// No-allocation entry point (include/snap.h "No-allocation variant"): snap_schur_apply with its scratch vector
// g = J^T x in a file-scope device array instead of a caller workspace, for callers that cannot allocate (CUDA graph
// capture, serving loops, harnesses that forbid cudaMalloc).  Every GPU that loads the library holds the array until
// the process exits.  In host code `g_static_scratch` is only the host-side stand-in of the symbol: the device address
// is fetched once per device with cudaGetSymbolAddress, that device current, and handed to the kernels.
// ------------------------------------------------------------------------------------------------------
static __device__ __align__(256) double g_static_scratch[SNAP_STATIC_SCRATCH_BYTES / 8];

namespace {
constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
double* g_static_addr[kStaticMaxDevices] = {};   // device address of g_static_scratch on device i (null: not set up)

// device address of the scratch array on the CURRENT device; first use on a device resolves the symbol there
int static_scratch_addr(double** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return SNAP_ECUDA;
  if (dev < 0 || dev >= kStaticMaxDevices) return SNAP_EINVAL;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_addr[dev]) {
    void* a = nullptr;
    if (cudaGetSymbolAddress(&a, g_static_scratch) != cudaSuccess || !a) return SNAP_ECUDA;
    g_static_addr[dev] = static_cast<double*>(a);
  }
  *out = g_static_addr[dev];
  return SNAP_OK;
}
}  // namespace

size_t snap_static_scratch_bytes(void) { return (size_t)SNAP_STATIC_SCRATCH_BYTES; }

int snap_static_scratch_init(void) {
  double* a = nullptr;
  return static_scratch_addr(&a);
}

int snap_schur_apply_static(const snap_problem* cp, int batch, const double* u, const double* x, double* out,
                            snap_stream stream) {
  snap_problem* p = const_cast<snap_problem*>(cp);
  if (!p || batch < 0) return SNAP_EINVAL;
  if (batch == 0) return SNAP_OK;
  if (!u || !x || !out) return SNAP_EINVAL;
  if (p->dp.kind >= SNAP_BURGERS1D_FLUXK) return SNAP_EINVAL;   // kinds 0-4 only, as snap_schur_apply
  if ((size_t)batch * p->dp.n > (size_t)SNAP_STATIC_SCRATCH_BYTES / 8) return SNAP_ELIMIT;
  double* g = nullptr;
  int rc = static_scratch_addr(&g);
  if (rc != SNAP_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  // nothing in the scratch has to start at zero: the first kernel writes every g[b][0..n) the second one reads
  jt_apply_kernel<<<batch, kMiscThreads, 0, st>>>(p->dp, batch, u, x, g);
  rc = check_launch(p);
  if (rc != SNAP_OK) return rc;
  j_apply_kernel<<<batch, kMiscThreads, 0, st>>>(p->dp, batch, u, g, out);
  return check_launch(p);
}

const char* snap_strerror(int code) {
  switch (code) {
    case SNAP_OK: return "ok";
    case SNAP_EINVAL: return "invalid argument (kind, sizes, NULL pointer or size limit)";
    case SNAP_ECUDA: return "CUDA call or kernel launch failed";
    case SNAP_ENOMEM: return "workspace too small or allocation failed";
    case SNAP_ELIMIT: return "problem larger than the static scratch of a no-allocation entry point (snap_static_scratch_bytes)";
  }
  return "unknown error code";
}

}  // extern "C"
