// Launchers of the individual Phi-path kernels (phi_simt.cu, phi_tc.cu); orchestrated by phi.cu.
#pragma once
#include "ltv_internal.h"

namespace ltv {

cudaError_t launch_phi_level0(const PhiArgs& a, int NT, int num_sms, cudaStream_t stream);
// observer variant (a.Lt != nullptr): two launches, Abar_s with the tube partial, then PhiY(s+1,s) = Abar_s Lt_s
cudaError_t launch_phi_obs_level0(const PhiArgs& a, int NT, int num_sms, cudaStream_t stream);
cudaError_t launch_phi_combine_simt(const PhiArgs& a, int level, int num_sms, cudaStream_t stream);
cudaError_t launch_phi_finalize(const PhiArgs& a, int NT, cudaStream_t stream);

// tcgen05 3xTF32 combine.  `nch` = n-tile width / 32 (2..8).  The tensor maps are built once per call.
struct PhiTcMaps;  // opaque (two CUtensorMap)
size_t phi_tc_maps_size();
cudaError_t phi_tc_make_maps(const PhiArgs& a, int nch, void* maps_out);
cudaError_t launch_phi_combine_tc(const PhiArgs& a, int level, int nch, const void* maps, int num_sms,
                                  cudaStream_t stream);

void* get_encode_tiled();  // adjoint.cu

}  // namespace ltv
