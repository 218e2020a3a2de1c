// node-kernel instantiations (marut_node.cuh): 2-D compressible Euler, N = 1..7
#include "marut_node.cuh"
#include "marut_launch.h"
namespace marut {
template <int NP>
static cudaError_t go(bool affine, const StageParams &P, cudaStream_t st) {
  return affine ? launch_stage_node_t<2, NP, true>(P, st) : launch_stage_node_t<2, NP, false>(P, st);
}
cudaError_t launch_stage_node2d(int np, bool affine, const StageParams &P, cudaStream_t st) {
  switch (np) {
    case 2: return go<2>(affine, P, st);
    case 3: return go<3>(affine, P, st);
    case 4: return go<4>(affine, P, st);
    case 5: return go<5>(affine, P, st);
    case 6: return go<6>(affine, P, st);
    case 7: return go<7>(affine, P, st);
    case 8: return go<8>(affine, P, st);
  }
  return cudaErrorNotSupported;
}
}  // namespace marut
