// update_su2.cu -- instantiations of the SU(2) (quaternion) update kernel, fp32 and fp64.
#include "launch.h"

namespace qcd {

template <typename R, int D, int KIND, bool FIELD, bool MEAS>
static cudaError_t go(const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  typedef typename PlaneTraits<R, 4>::Vec Vec;
  const unsigned block = 256, grid = (g.Vh_int + block - 1) / block;
  return launch_pdl(su2_update_kernel<R, D, KIND, FIELD, MEAS>, dim3(grid), dim3(block), 0, st, g, (Vec*)links, a);
}
template <typename R, int D, bool MEAS>
static cudaError_t sel3(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  if (s.kind == 0) return s.field ? go<R, D, 0, true, MEAS>(g, links, a, st) : go<R, D, 0, false, MEAS>(g, links, a, st);
  return s.field ? go<R, D, 1, true, MEAS>(g, links, a, st) : go<R, D, 1, false, MEAS>(g, links, a, st);
}
template <typename R, int D>
static cudaError_t sel2(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  return s.meas ? sel3<R, D, true>(s, g, links, a, st) : sel3<R, D, false>(s, g, links, a, st);
}
template <typename R>
static cudaError_t sel1(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  switch (s.D) {
    case 2: return sel2<R, 2>(s, g, links, a, st);
    case 3: return sel2<R, 3>(s, g, links, a, st);
    case 4: return sel2<R, 4>(s, g, links, a, st);
  }
  return cudaErrorInvalidValue;
}
cudaError_t launch_update_su2(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  return s.precision == 0 ? sel1<float>(s, g, links, a, st) : sel1<double>(s, g, links, a, st);
}

}  // namespace qcd
