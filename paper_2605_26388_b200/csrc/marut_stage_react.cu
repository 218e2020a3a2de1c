// fused reacting-Euler stage kernel instantiations: 5 species, 2-D and 3-D, N = 1..4
#include "marut_node_phys.cuh"
#include "marut_launch.h"
namespace marut {
template <int DIM, int NP>
static cudaError_t go(bool affine, const StageParams &P, cudaStream_t st) {
  return affine ? launch_stage_phys_t<DIM, NP, 5, PH_REACT, true>(P, st) : launch_stage_phys_t<DIM, NP, 5, PH_REACT, false>(P, st);
}
cudaError_t launch_stage_react(int dim, int np, int nsp, bool affine, const StageParams &P, cudaStream_t st) {
  if (nsp != 5) return cudaErrorNotSupported;
  if (dim == 2) switch (np) {
      case 2: return go<2, 2>(affine, P, st);
      case 3: return go<2, 3>(affine, P, st);
      case 4: return go<2, 4>(affine, P, st);
      case 5: return go<2, 5>(affine, P, st);
    }
  if (dim == 3) switch (np) {
      case 2: return go<3, 2>(affine, P, st);
      case 3: return go<3, 3>(affine, P, st);
      case 4: return go<3, 4>(affine, P, st);
      case 5: return go<3, 5>(affine, P, st);
    }
  return cudaErrorNotSupported;
}
}  // namespace marut
