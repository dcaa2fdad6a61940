// kg_tb2_launch.h — host entry point of the two-step kernels (kg_tb2.cu).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

struct Tb2Args;
// row widths the two-step kernel is compiled for
inline bool kg_tb2_k_supported(int K) { return K == 2 || K == 3 || K == 4 || K == 6; }
// mode: MODE_MOM2 (C = 1, 2) or MODE_MOMX (C = 2); nstep 1 or 2.  cudaErrorInvalidValue if not compiled.
cudaError_t kg_tb2_launch(int K, int mode, int C, bool has_onsite, int nstep, const Tb2Args &a, int grid, size_t smem,
                          int device, cudaStream_t st);
