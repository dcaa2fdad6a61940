// kg_staged_launch.h — host entry points of the TMA-staged kernels, one per compiled row width K
// (kg_staged_k2.cu, kg_staged_k3.cu, kg_staged_k4.cu, kg_staged_k6.cu, kg_staged_k9.cu; body in kg_staged_impl.cuh).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

struct StagedArgs;
struct StagedLaunch {
    int grid;
    size_t smem;          // dynamic shared memory per CTA
    int device;
    bool has_onsite;      // ONS template flag
    bool dict;            // DICT template flag
    bool pdl;             // launch with programmatic stream serialization
};

// mode: MODE_MOM / MODE_EVO / MODE_PAIR / MODE_MOM2 / MODE_MOMX; R: columns of the batch.
// cudaErrorInvalidValue if the (mode, R) pair is not compiled.
cudaError_t kg_staged_launch_k2(int mode, int R, const StagedArgs &a, const StagedLaunch &l, cudaStream_t st);
cudaError_t kg_staged_launch_k3(int mode, int R, const StagedArgs &a, const StagedLaunch &l, cudaStream_t st);
cudaError_t kg_staged_launch_k4(int mode, int R, const StagedArgs &a, const StagedLaunch &l, cudaStream_t st);
cudaError_t kg_staged_launch_k6(int mode, int R, const StagedArgs &a, const StagedLaunch &l, cudaStream_t st);
cudaError_t kg_staged_launch_k9(int mode, int R, const StagedArgs &a, const StagedLaunch &l, cudaStream_t st);
