// Fisher-KPP (kind 2) fused Gauss-Newton kernel instantiations (nx = 32 Q, one warp per sample).
#include "kernels_1d_fused.cuh"

namespace snap {

bool fused_variant_fisher(int nx, int& W, int& Q, int& JT, int& maxt) {
  W = 1; maxt = 256;
  switch (nx) {
    case 32: Q = 1; JT = 4; return true;
    case 64: Q = 2; JT = 4; return true;
    case 128: Q = 4; JT = 3; return true;
    case 256: Q = 8; JT = 2; return true;
  }
  return false;
}

int launch_project1d_fisher_fused(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st) {
  switch (a.P.nx) {
    case 32: return launch_fused_variant<KF_FUSED, 1, 1, 4, 256>(a, pl, st);
    case 64: return launch_fused_variant<KF_FUSED, 1, 2, 4, 256>(a, pl, st);
    case 128: return launch_fused_variant<KF_FUSED, 1, 4, 3, 256>(a, pl, st);
    case 256: return launch_fused_variant<KF_FUSED, 1, 8, 2, 256>(a, pl, st);
  }
  return SNAP_EINVAL;
}

}  // namespace snap
