// kg_smem_config.h — once-per-device opt-in to large dynamic shared memory (and non-portable cluster
// sizes) for one kernel instantiation, safe when several host threads drive different handles:
// the attribute only ever grows, under a lock.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

#include <mutex>

struct KgSmemConfig {
    std::mutex m;
    size_t configured[64] = {0};
    bool big_cluster[64] = {false};

    template <class Kernel>
    cudaError_t ensure(Kernel kernel, int device, size_t smem, bool non_portable_cluster = false)
    {
        const int dev = device & 63;
        std::lock_guard<std::mutex> lock(m);
        if (configured[dev] < smem) {
            cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
            configured[dev] = smem;
        }
        if (non_portable_cluster && !big_cluster[dev]) {
            cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
            if (e != cudaSuccess) return e;
            big_cluster[dev] = true;
        }
        return cudaSuccess;
    }
};
