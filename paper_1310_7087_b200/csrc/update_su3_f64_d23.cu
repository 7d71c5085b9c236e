// update_su3_f64_d23.cu -- SU(3) update kernels in double, D = 2 and 3 (plain and fused-measurement forms), and the per-D dispatch.
#include "su3_launch.cuh"

namespace qcd {
cudaError_t launch_update_su3_f64(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  switch (s.D) {
    case 2: return s.meas ? su3_sel_mu<double, 2, true>(s, g, links, a, st) : su3_sel_mu<double, 2, false>(s, g, links, a, st);
    case 3: return s.meas ? su3_sel_mu<double, 3, true>(s, g, links, a, st) : su3_sel_mu<double, 3, false>(s, g, links, a, st);
    case 4: return s.meas ? launch_update_su3_f64_d4_meas(s, g, links, a, st) : launch_update_su3_f64_d4(s, g, links, a, st);
  }
  return cudaErrorInvalidValue;
}
}  // namespace qcd
