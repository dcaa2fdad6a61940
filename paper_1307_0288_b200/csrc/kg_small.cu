// Single-launch moment loop for launch-bound sizes (kg_small.cuh): template dispatch and cluster launch.
#include "kg_small.cuh"
#include "kg_small_launch.h"
#include "kg_smem_config.h"

namespace {

template <int R, int MODE, int KU>
cudaError_t launch_ku(const SmallArgs &a, int ncta, size_t smem, int device, cudaStream_t st);

template <int R, int MODE>
cudaError_t launch_t(const SmallArgs &a, int ncta, size_t smem, int device, cudaStream_t st)
{
    if (a.K <= 4) return launch_ku<R, MODE, 4>(a, ncta, smem, device, st);
    if (a.K <= 12) return launch_ku<R, MODE, 12>(a, ncta, smem, device, st);
    return cudaErrorInvalidValue;
}

template <int R, int MODE, int KU, int VT>
cudaError_t launch_reg(const SmallArgs &a, int ncta, size_t smem, int device, cudaStream_t st)
{
    static KgSmemConfig cfg_once;
    if (cudaError_t e = cfg_once.ensure(kg_small_reg_kernel<R, MODE, KU, VT>, device, smem, ncta > SM_MAX_CLUSTER)) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)ncta);
    cfg.blockDim = dim3(SM_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)ncta;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kg_small_reg_kernel<R, MODE, KU, VT>, a);
}

template <int R, int MODE, int KU>
cudaError_t launch_ku(const SmallArgs &a, int ncta, size_t smem, int device, cudaStream_t st)
{
    // the register-resident form for the paper's row widths and <= 2 tiles per CTA
    if constexpr (KU == 4) {
        if (a.vt == 1) return launch_reg<R, MODE, KU, 1>(a, ncta, smem, device, st);
        if (a.vt == 2) return launch_reg<R, MODE, KU, 2>(a, ncta, smem, device, st);
    }
    static KgSmemConfig cfg_once;
    if (cudaError_t e = cfg_once.ensure(kg_small_kernel<R, MODE, KU>, device, smem, ncta > SM_MAX_CLUSTER)) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)ncta);
    cfg.blockDim = dim3(SM_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)ncta;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kg_small_kernel<R, MODE, KU>, a);
}

template <int R>
cudaError_t launch_r(int mode, const SmallArgs &a, int ncta, size_t smem, int device, cudaStream_t st)
{
    switch (mode) {
    case MODE_MOM: return launch_t<R, MODE_MOM>(a, ncta, smem, device, st);
    case MODE_MOM2: return launch_t<R, MODE_MOM2>(a, ncta, smem, device, st);
    case MODE_MOMX:
        if constexpr (R >= 2) return launch_t<R, MODE_MOMX>(a, ncta, smem, device, st);
        break;
    }
    return cudaErrorInvalidValue;
}

}  // namespace

cudaError_t kg_small_launch(int mode, int R, const SmallArgs &a, int ncta, size_t smem, int device, cudaStream_t st)
{
    if (ncta < 1 || ncta > SM_BIG_CLUSTER) return cudaErrorInvalidValue;
    switch (R) {
    case 1: return launch_r<1>(mode, a, ncta, smem, device, st);
    case 2: return launch_r<2>(mode, a, ncta, smem, device, st);
    case 4: return launch_r<4>(mode, a, ncta, smem, device, st);
    case 8: return launch_r<8>(mode, a, ncta, smem, device, st);
    case 16: return launch_r<16>(mode, a, ncta, smem, device, st);
    }
    return cudaErrorInvalidValue;
}
