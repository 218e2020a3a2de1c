// split-form (entropy-stable) Euler stage kernel instantiations (marut_split.cuh): 2-D N = 1..7, 3-D N = 1..6
// (3-D N = 7 would need 303 KB of shared memory for the pair buffer)
#include "marut_split.cuh"
#include "marut_launch.h"
namespace marut {
template <int DIM, int NP>
static cudaError_t go(bool affine, const StageParams &P, cudaStream_t st) {
  return affine ? launch_stage_split_t<DIM, NP, true>(P, st) : launch_stage_split_t<DIM, NP, false>(P, st);
}
cudaError_t launch_stage_split(int dim, int np, bool affine, const StageParams &P, cudaStream_t st) {
  if (dim == 2) switch (np) {
      case 2: return go<2, 2>(affine, P, st);
      case 3: return go<2, 3>(affine, P, st);
      case 4: return go<2, 4>(affine, P, st);
      case 5: return go<2, 5>(affine, P, st);
      case 6: return go<2, 6>(affine, P, st);
      case 7: return go<2, 7>(affine, P, st);
      case 8: return go<2, 8>(affine, P, st);
    }
  if (dim == 3) switch (np) {
      case 2: return go<3, 2>(affine, P, st);
      case 3: return go<3, 3>(affine, P, st);
      case 4: return go<3, 4>(affine, P, st);
      case 5: return go<3, 5>(affine, P, st);
      case 6: return go<3, 6>(affine, P, st);
      case 7: return go<3, 7>(affine, P, st);
    }
  return cudaErrorNotSupported;
}
}  // namespace marut
