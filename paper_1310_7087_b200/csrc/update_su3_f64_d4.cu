// update_su3_f64_d4.cu -- SU(3) update kernels in double, D = 4 (all mu, storage, kind, field variants).
#include "su3_launch.cuh"

namespace qcd {
cudaError_t launch_update_su3_f64_d4(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  return su3_sel_mu<double, 4, false>(s, g, links, a, st);
}
}  // namespace qcd
