// Instantiations of the tiled kernel for one (data kind, storage) mode; see das_tiled.cuh.
#include "das_tiled.cuh"
namespace das {
cudaError_t launch_tiled_rf8(int QC, int W, const TiledDev& tp, const Params& P, const void* conv, void* out, int grid, cudaStream_t s) {
  return launch_tiled_mode<kRF8>(QC, W, tp, P, conv, out, grid, s);
}
}  // namespace das
