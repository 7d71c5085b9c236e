// update_su3_f32_d4_meas.cu -- the same in the fused-measurement form (last pass of qcd_sweep_measure, parity 1, mu >= 1).
#include "su3_launch.cuh"

namespace qcd {
cudaError_t launch_update_su3_f32_d4_meas(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  return su3_sel_mu<float, 4, true>(s, g, links, a, st);
}
}  // namespace qcd
