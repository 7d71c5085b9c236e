// update_su3_f32.cu -- instantiations of the SU(3) update kernel in float (all D, storage, kind, field variants).
#include "launch.h"

namespace qcd {

template <int D, bool COMP, int KIND, bool FIELD>
static cudaError_t go(const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  typedef typename PlaneTraits<float, (COMP ? 12 : 18)>::Vec Vec;
  const unsigned block = 128, grid = (g.Vh + block - 1) / block;
  su3_update_kernel<float, D, COMP, KIND, FIELD><<<grid, block, 0, st>>>(g, (Vec*)links, a);
  return cudaGetLastError();
}
template <int D, bool COMP>
static cudaError_t sel2(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  if (s.kind == 0) return s.field ? go<D, COMP, 0, true>(g, links, a, st) : go<D, COMP, 0, false>(g, links, a, st);
  return s.field ? go<D, COMP, 1, true>(g, links, a, st) : go<D, COMP, 1, false>(g, links, a, st);
}
template <int D>
static cudaError_t sel1(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  return s.comp ? sel2<D, true>(s, g, links, a, st) : sel2<D, false>(s, g, links, a, st);
}
cudaError_t launch_update_su3_f32(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  switch (s.D) {
    case 2: return sel1<2>(s, g, links, a, st);
    case 3: return sel1<3>(s, g, links, a, st);
    case 4: return sel1<4>(s, g, links, a, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace qcd
