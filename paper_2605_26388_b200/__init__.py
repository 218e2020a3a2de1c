"""B200-native DG right-hand side + SSP-RK33 hot path of MARUT (arxiv 2605.26388).

Thin Python binding over the C ABI of include/marut.h (argument marshalling only: every step of
the path runs in the CUDA kernels of csrc/).  PyTorch provides device memory and streams.
There is no CPU fallback: importing works anywhere, but every call needs libmarut.so and a GPU.
"""
from .binding import (MarutError, MarutMesh, lib, lib_path, EULER, NAVIER_STOKES, REACTING_EULER,  # noqa: F401
                      marut_mesh_create, marut_mesh_destroy, marut_rhs, marut_ssprk_stage, marut_max_dt,
                      marut_chem_source, ssprk3_step)
