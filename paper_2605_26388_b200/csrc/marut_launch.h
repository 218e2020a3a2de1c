// marut_launch.h -- launchers defined in the per-physics translation units (compiled in parallel).
// Each returns cudaErrorNotSupported when (dim, n, n_species) was not instantiated.
#pragma once
#include "marut_common.cuh"

namespace marut {
struct GradParams;
// marut_pencil.cuh: Euler, strong form, affine meshes (mortar: the 2-D instantiation that knows 2:1 mortar faces)
cudaError_t launch_stage_pencil(int dim, int np, bool mortar, bool force, const StageParams &P, cudaStream_t st);
cudaError_t launch_stage_node2d(int np, bool affine, const StageParams &P, cudaStream_t st);
cudaError_t launch_stage_node3d(int np, bool affine, const StageParams &P, cudaStream_t st);
cudaError_t launch_mortar_flux3d(int np, const double *u, const double *metric, const int *info, const int *fine, const double *mat,
                                 double gamma, double *mflux, long n_mortar, cudaStream_t st);
cudaError_t launch_mortar_flux2d(int np, const double *u, const double *metric, int affine, const int *info, const int *fine,
                                 const double *mat, double gamma, double *mflux, long n_mortar, cudaStream_t st);
cudaError_t launch_stage_split(int dim, int np, bool affine, const StageParams &P, cudaStream_t st);
cudaError_t launch_stage_ns(int dim, int np, bool affine, const StageParams &P, cudaStream_t st);
cudaError_t launch_gradient(int dim, int np, bool affine, const GradParams &P, cudaStream_t st);
cudaError_t launch_mortar_trace3d(int np, const double *u, const int *info, const int *fine, const double *mat, double gamma,
                                  double *mW, long n_mortar, cudaStream_t st);
cudaError_t launch_mortar_flux3d_ns(int np, bool hyp, const double *u, const double *S, const double *metric, const int *info,
                                    const int *fine, const double *mat, double gamma, double *mflux, long n_mortar,
                                    cudaStream_t st);
cudaError_t launch_stage_react(int dim, int np, int nsp, bool affine, const StageParams &P, cudaStream_t st);
}  // namespace marut
