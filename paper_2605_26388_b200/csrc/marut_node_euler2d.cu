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
// F* at the fine face nodes of every 2-D mortar, stored ahead of the line kernel (marut_node.cuh)
cudaError_t launch_mortar_flux2d(int np, const double *u, const double *metric, int affine, const int *info, const int *fine,
                                 const double *mat, double gamma, double *mflux, long n_mortar, cudaStream_t st) {
  switch (np) {
    case 2: return launch_mortar_flux2d_t<2>(u, metric, affine, info, fine, mat, gamma, mflux, n_mortar, st);
    case 3: return launch_mortar_flux2d_t<3>(u, metric, affine, info, fine, mat, gamma, mflux, n_mortar, st);
    case 4: return launch_mortar_flux2d_t<4>(u, metric, affine, info, fine, mat, gamma, mflux, n_mortar, st);
    case 5: return launch_mortar_flux2d_t<5>(u, metric, affine, info, fine, mat, gamma, mflux, n_mortar, st);
    case 6: return launch_mortar_flux2d_t<6>(u, metric, affine, info, fine, mat, gamma, mflux, n_mortar, st);
    case 7: return launch_mortar_flux2d_t<7>(u, metric, affine, info, fine, mat, gamma, mflux, n_mortar, st);
    case 8: return launch_mortar_flux2d_t<8>(u, metric, affine, info, fine, mat, gamma, mflux, n_mortar, st);
  }
  return cudaErrorNotSupported;
}
}  // namespace marut
