// Burgers-family (kinds 1, 4) fused Gauss-Newton kernel instantiations (nx = 32 W Q).
#include "kernels_1d_fused.cuh"

namespace snap {

// (W warps per sample, Q cells per lane, JT iterations per pass, max threads per CTA) per supported nx.
// W > 1 needs a warp's part of a row to start on a 1024-byte boundary (Q >= 4).
bool fused_variant(int nx, int& W, int& Q, int& JT, int& maxt) {
  switch (nx) {
    case 32: W = 1; Q = 1; JT = 4; maxt = 256; return true;
    case 64: W = 1; Q = 2; JT = 4; maxt = 256; return true;
    case 128: W = 1; Q = 4; JT = 4; maxt = 256; return true;
    case 256: W = 1; Q = 8; JT = 3; maxt = 256; return true;
    case 512: W = 2; Q = 8; JT = 3; maxt = 256; return true;
  }
  return false;
}

int fused_row_pitch(int nx) { return nx < 128 ? 128 : nx; }

int launch_project1d_burgers_fused(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st) {
  switch (a.P.nx) {
    case 32: return launch_fused_variant<KB_FUSED, 1, 1, 4, 256>(a, pl, st);
    case 64: return launch_fused_variant<KB_FUSED, 1, 2, 4, 256>(a, pl, st);
    case 128: return launch_fused_variant<KB_FUSED, 1, 4, 4, 256>(a, pl, st);
    case 256:
      return launch_fused_variant<KB_FUSED, 1, 8, 3, 256>(a, pl, st);
    case 512: return launch_fused_variant<KB_FUSED, 2, 8, 3, 256>(a, pl, st);
  }
  return SNAP_EINVAL;
}

}  // namespace snap
