// kg_small_launch.h — host entry point of the single-launch moment loop (kg_small.cu).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

struct SmallArgs;
// mode: MODE_MOM / MODE_MOM2 / MODE_MOMX; R columns (1, 2, 4, 8; MOMX: >= 2); ncta CTAs in one cluster (<= 8).
cudaError_t kg_small_launch(int mode, int R, const SmallArgs &a, int ncta, size_t smem, int device, cudaStream_t st);
