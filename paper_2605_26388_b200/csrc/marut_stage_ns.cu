// BR1 gradient + fused Navier-Stokes stage kernel instantiations: 2-D and 3-D, N = 1..5
#include "marut_node_phys.cuh"
#include "marut_launch.h"
namespace marut {
template <int DIM, int NP>
static cudaError_t go(bool affine, const StageParams &P, cudaStream_t st) {
  return affine ? launch_stage_phys_t<DIM, NP, 1, PH_NS, true>(P, st) : launch_stage_phys_t<DIM, NP, 1, PH_NS, false>(P, st);
}
template <int DIM, int NP>
static cudaError_t gr(bool affine, const GradParams &P, cudaStream_t st) {
  return affine ? launch_gradient_t<DIM, NP, true>(P, st) : launch_gradient_t<DIM, NP, false>(P, st);
}
#define MARUT_NS_CASES(FN, ...)                                   \
  if (dim == 2) switch (np) {                                     \
      case 2: return FN<2, 2>(__VA_ARGS__);                       \
      case 3: return FN<2, 3>(__VA_ARGS__);                       \
      case 4: return FN<2, 4>(__VA_ARGS__);                       \
      case 5: return FN<2, 5>(__VA_ARGS__);                       \
      case 6: return FN<2, 6>(__VA_ARGS__);                       \
    }                                                             \
  if (dim == 3) switch (np) {                                     \
      case 2: return FN<3, 2>(__VA_ARGS__);                       \
      case 3: return FN<3, 3>(__VA_ARGS__);                       \
      case 4: return FN<3, 4>(__VA_ARGS__);                       \
      case 5: return FN<3, 5>(__VA_ARGS__);                       \
      case 6: return FN<3, 6>(__VA_ARGS__);                       \
    }                                                             \
  return cudaErrorNotSupported;
cudaError_t launch_stage_ns(int dim, int np, bool affine, const StageParams &P, cudaStream_t st) {
  MARUT_NS_CASES(go, affine, P, st)
}
cudaError_t launch_gradient(int dim, int np, bool affine, const GradParams &P, cudaStream_t st) {
  MARUT_NS_CASES(gr, affine, P, st)
}
// pre-kernels of the 3-D mortars of a Navier-Stokes mesh (readings R21 + R23)
cudaError_t launch_mortar_trace3d(int np, const double *u, const int *info, const int *fine, const double *mat, double gamma,
                                  double *mW, long n_mortar, cudaStream_t st) {
  switch (np) {
    case 2: return launch_mortar_trace3d_t<2>(u, info, fine, mat, gamma, mW, n_mortar, st);
    case 3: return launch_mortar_trace3d_t<3>(u, info, fine, mat, gamma, mW, n_mortar, st);
    case 4: return launch_mortar_trace3d_t<4>(u, info, fine, mat, gamma, mW, n_mortar, st);
    case 5: return launch_mortar_trace3d_t<5>(u, info, fine, mat, gamma, mW, n_mortar, st);
    case 6: return launch_mortar_trace3d_t<6>(u, info, fine, mat, gamma, mW, n_mortar, st);
  }
  return cudaErrorNotSupported;
}
cudaError_t launch_mortar_flux3d_ns(int np, bool hyp, const double *u, const double *S, const double *metric, const int *info,
                                    const int *fine, const double *mat, double gamma, double *mflux, long n_mortar,
                                    cudaStream_t st) {
  switch (np) {
    case 2: return launch_mortar_flux3d_ns_t<2>(hyp, u, S, metric, info, fine, mat, gamma, mflux, n_mortar, st);
    case 3: return launch_mortar_flux3d_ns_t<3>(hyp, u, S, metric, info, fine, mat, gamma, mflux, n_mortar, st);
    case 4: return launch_mortar_flux3d_ns_t<4>(hyp, u, S, metric, info, fine, mat, gamma, mflux, n_mortar, st);
    case 5: return launch_mortar_flux3d_ns_t<5>(hyp, u, S, metric, info, fine, mat, gamma, mflux, n_mortar, st);
    case 6: return launch_mortar_flux3d_ns_t<6>(hyp, u, S, metric, info, fine, mat, gamma, mflux, n_mortar, st);
  }
  return cudaErrorNotSupported;
}
}  // namespace marut
