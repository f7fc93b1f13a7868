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

// Cross block of a block-triangular closed loop on the geometry of the Phi scan (MODE 2 of the kernel): at `level`, for
// every s < mid < t of a segment, G(t,s) = Pbar(t,mid) G(mid,s) + G(t,mid) Phat(mid,s) with a.phi = G (column-packed,
// nc = n) - one K loop over both operand pairs into one accumulator.  No tube.
cudaError_t phi_tc_make_cross_maps(const PhiArgs& a, const float* pbar, const float* phat, int nch, void* maps_out);
cudaError_t launch_phi_cross_tc(const PhiArgs& a, int level, int nch, const void* maps, int num_sms, cudaStream_t stream);

// Batched fp32 GEMM on the same tcgen05 3xTF32 kernel (its MODE 1): D[b] = L[b] R[b], b < count, all row-major.
//   L  array viewed as [l_rows][K];       problem b reads rows [l_row0 + b l_row_stride, +M)
//   R  array viewed as [r_blocks][K][N];  problem b reads block r_blk0 + b r_blk_stride
//   D  array viewed as [d_blocks][M][N] (transpose_out: [d_blocks][N][M], holding D[b]^T); block d_blk0 + b d_blk_stride
//   diag (may be null): adds diag[b diag_stride + i]^2 to D[b][i][i]
// K, N multiples of 4, every base pointer 16-byte aligned.  The maps depend on the arrays and M, N, K only, so a
// caller stepping l_row0 / r_blk0 / d_blk0 through time builds them once.
struct BatchedGemm {
  const float* L; long long l_rows; int l_row0, l_row_stride;
  const float* R; int r_blocks, r_blk0, r_blk_stride;
  float* D; int d_blocks, d_blk0, d_blk_stride;
  int count, M, N, K;
  int d_rows;   // rows of one D block in memory; 0 = M.  (> M only without transpose_out: rows [M, d_rows) are not written;
                // the maps are built for d_rows, so M may then change from launch to launch)
  int transpose_out;
  const float* diag; long long diag_stride;
  int d_row0 = 0, d_row_stride = 0;   // extra row offset d_row0 + b d_row_stride of problem b inside its D block (plain stores only:
                                      // several problems may then share one big block, e.g. a whole column-packed Phi array)
};
cudaError_t bgemm_tc_make_maps(const BatchedGemm& a, void* maps_out);
cudaError_t launch_bgemm_tc(const BatchedGemm& a, int nch, const void* maps, int num_sms, cudaStream_t stream);
cudaError_t launch_bgemm_simt(const BatchedGemm& a, cudaStream_t stream);   // fp32 FMA, any size (kalman.cu)
int phi_pick_nch(int n);   // phi.cu

void* get_encode_tiled();  // adjoint.cu

}  // namespace ltv
