// launch.h -- host-side launcher declarations; each translation unit instantiates one family of kernels.
#pragma once
#include "common.cuh"
#include "update.cuh"

namespace qcd {

struct UpdateSel {
  int Nc, D, precision;   // precision: 0 fp32, 1 fp64
  bool comp;
  int kind;               // 0 HB, 1 OR
  bool field;
  bool meas;              // fused plaquette measurement (UpdateArgs::meas set; mu >= 1)
};

// returns cudaErrorInvalidValue for an unsupported combination
cudaError_t launch_update_su3_f32(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st);
cudaError_t launch_update_su3_f64(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st);
cudaError_t launch_update_su3_f32_d4(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st);
cudaError_t launch_update_su3_f64_d4(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st);
cudaError_t launch_update_su3_f32_d4_meas(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st);
cudaError_t launch_update_su3_f64_d4_meas(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st);
cudaError_t launch_update_su2(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st);

}  // namespace qcd
