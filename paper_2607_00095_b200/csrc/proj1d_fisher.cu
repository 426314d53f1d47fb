// Fisher-KPP (kind 2) instantiations of the persistent 1D projection kernel.
#include "kernels_1d.cuh"

namespace snap {
int launch_project1d_fisher(const Proj1dArgs& a, const Plan1d& pl, cudaStream_t st) {
  return launch_1d_kind<KF>(a, pl, st);
}
}  // namespace snap
