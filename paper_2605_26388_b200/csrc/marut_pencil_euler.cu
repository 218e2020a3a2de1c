// pencil-kernel instantiations (marut_pencil.cuh): compressible Euler on affine meshes, 2-D N = 1..7, 3-D N = 1..5
#include "marut_pencil.cuh"
#include "marut_launch.h"
namespace marut {
cudaError_t launch_stage_pencil(int dim, int np, bool mortar, bool force, const StageParams &P, cudaStream_t st) {
  if (dim == 2) switch (np) {
      case 2: return mortar ? launch_stage_pencil_t<2, 2, true>(P, force, st) : launch_stage_pencil_t<2, 2, false>(P, force, st);
      case 3: return mortar ? launch_stage_pencil_t<2, 3, true>(P, force, st) : launch_stage_pencil_t<2, 3, false>(P, force, st);
      case 4: return mortar ? launch_stage_pencil_t<2, 4, true>(P, force, st) : launch_stage_pencil_t<2, 4, false>(P, force, st);
      case 5: return mortar ? launch_stage_pencil_t<2, 5, true>(P, force, st) : launch_stage_pencil_t<2, 5, false>(P, force, st);
      case 6: return mortar ? launch_stage_pencil_t<2, 6, true>(P, force, st) : launch_stage_pencil_t<2, 6, false>(P, force, st);
      case 7: return mortar ? launch_stage_pencil_t<2, 7, true>(P, force, st) : launch_stage_pencil_t<2, 7, false>(P, force, st);
      case 8: return mortar ? launch_stage_pencil_t<2, 8, true>(P, force, st) : launch_stage_pencil_t<2, 8, false>(P, force, st);
    }
  if (dim == 3 && !mortar) switch (np) {
      case 2: return launch_stage_pencil_t<3, 2, false>(P, force, st);
      case 3: return launch_stage_pencil_t<3, 3, false>(P, force, st);
      case 4: return launch_stage_pencil_t<3, 4, false>(P, force, st);
      case 5: return launch_stage_pencil_t<3, 5, false>(P, force, st);
      case 6: return launch_stage_pencil_t<3, 6, false>(P, force, st);
    }
  return cudaErrorNotSupported;
}
}  // namespace marut
