// register-tiled line kernel instantiations (marut_line2.cuh): 3-D compressible Euler, affine meshes, N = 2..5
#include "marut_line2.cuh"
#include "marut_launch.h"
namespace marut {
cudaError_t launch_stage_line2_3d(int np, const StageParams &P, cudaStream_t st) {
  switch (np) {
    case 3: return launch_stage_line2_t<3>(P, st);
    case 4: return launch_stage_line2_t<4>(P, st);
    case 5: return launch_stage_line2_t<5>(P, st);
    case 6: return launch_stage_line2_t<6>(P, st);
  }
  return cudaErrorNotSupported;
}
}  // namespace marut
