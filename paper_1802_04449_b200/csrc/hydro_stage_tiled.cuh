// placeholder: replaced by the tiled kernel
#pragma once
#include "hydro_stage_ref.cuh"
namespace clv {
template <typename R, bool VISC, int MODE>
void launch_stage_tiled(const StageArgs<R>& a, cudaStream_t stream) {
  dim3 block(32, 8, 1);
  dim3 grid((a.nx + 31) / 32, (a.ny + 7) / 8, a.nz);
  stage_ref_kernel<R, VISC, MODE><<<grid, block, 0, stream>>>(a);
}
}  // namespace clv
