// Float32 mode of the Burgers kinds (kinds 1, 4), multiplier-free: kernel instantiations and launch.
#include "kernels_1d_f32.cuh"
#include "launch.h"

namespace snap {

template <int Q, int JT>
static int launch_f32_variant(const ProjF32Args& a, int sms, cudaStream_t st) {
  int wpc = (a.batch + sms - 1) / sms;          // warps (samples) per CTA: one wave over the SMs when possible
  if (wpc < 1) wpc = 1;
  if (wpc > 8) wpc = 8;
  const int grid = (a.batch + wpc - 1) / wpc;
  project1d_f32_kernel<Q, JT><<<grid, wpc * 32, 0, st>>>(a);
  return cudaGetLastError() == cudaSuccess ? SNAP_OK : SNAP_ECUDA;
}

int launch_project1d_f32(snap_problem* p, int batch, const float* u_hat, const float* cdata, float* u_star, int* iters,
                         float tol, void* workspace, cudaStream_t st) {
  const DevParams& d = p->dp;
  ProjF32Args a;
  a.P = d;
  a.batch = batch;
  a.u_hat = u_hat; a.cdata = cdata; a.u_star = u_star; a.iters = iters;
  a.bufA = reinterpret_cast<float*>(workspace);
  a.bufB = a.bufA + (size_t)batch * d.n;
  a.tol = tol;
  p->launches++;
  const int sms = p->sm_count > 0 ? p->sm_count : 148;
  switch (d.nx) {
    case 32: return launch_f32_variant<1, 4>(a, sms, st);
    case 64: return launch_f32_variant<2, 4>(a, sms, st);
    case 128: return launch_f32_variant<4, 4>(a, sms, st);
    case 256: return launch_f32_variant<8, 4>(a, sms, st);
  }
  return SNAP_EINVAL;
}

}  // namespace snap
