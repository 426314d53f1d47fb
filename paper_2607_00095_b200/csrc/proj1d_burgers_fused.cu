// Burgers-family (kinds 1, 4) fused Gauss-Newton kernel instantiations (nx = 32 q).
#include "kernels_1d_fused.cuh"

namespace snap {

int fused_row_pitch(int q) { return (32 * q / 16) * 18; }

int launch_project1d_burgers_fused(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st) {
  switch (pl.q) {
    case 1: return launch_fused_variant<1, 4>(a, pl, st);
    case 2: return launch_fused_variant<2, 4>(a, pl, st);
    case 4: return launch_fused_variant<4, 4>(a, pl, st);
    case 8: return launch_fused_variant<8, SNAP_FUSE_Q8>(a, pl, st);
    case 16: return launch_fused_variant<16, 2>(a, pl, st);
  }
  return SNAP_EINVAL;
}

}  // namespace snap
