// Two-step Chebyshev kernels (kg_tb2.cuh): template dispatch (K, columns, mode, ONS, steps per pass).
#include "kg_tb2.cuh"
#include "kg_tb2_launch.h"
#include "kg_smem_config.h"

namespace {

template <int C, int K, int MODE, bool ONS, int NSTEP>
cudaError_t launch_t(const Tb2Args &a, int grid, size_t smem, int device, cudaStream_t st)
{
    static KgSmemConfig cfg_once;
    if (cudaError_t e = cfg_once.ensure(kg_tb2_kernel<C, K, MODE, ONS, NSTEP>, device, smem)) return e;
    kg_tb2_kernel<C, K, MODE, ONS, NSTEP><<<grid, TB_THREADS, smem, st>>>(a);
    return cudaGetLastError();
}

template <int C, int K, int MODE>
cudaError_t launch_cm(bool ons, int nstep, const Tb2Args &a, int grid, size_t smem, int device, cudaStream_t st)
{
    if (ons) return nstep == 2 ? launch_t<C, K, MODE, true, 2>(a, grid, smem, device, st) : launch_t<C, K, MODE, true, 1>(a, grid, smem, device, st);
    return nstep == 2 ? launch_t<C, K, MODE, false, 2>(a, grid, smem, device, st) : launch_t<C, K, MODE, false, 1>(a, grid, smem, device, st);
}

template <int K>
cudaError_t launch_k(int mode, int C, bool ons, int nstep, const Tb2Args &a, int grid, size_t smem, int device, cudaStream_t st)
{
    if (mode == MODE_MOM2 && C == 1) return launch_cm<1, K, MODE_MOM2>(ons, nstep, a, grid, smem, device, st);
    if (mode == MODE_MOM2 && C == 2) return launch_cm<2, K, MODE_MOM2>(ons, nstep, a, grid, smem, device, st);
    if (mode == MODE_MOMX && C == 2) return launch_cm<2, K, MODE_MOMX>(ons, nstep, a, grid, smem, device, st);
    return cudaErrorInvalidValue;
}

}  // namespace

cudaError_t kg_tb2_launch(int K, int mode, int C, bool has_onsite, int nstep, const Tb2Args &a, int grid, size_t smem,
                          int device, cudaStream_t st)
{
    if (nstep != 1 && nstep != 2) return cudaErrorInvalidValue;
    switch (K) {
    case 2: return launch_k<2>(mode, C, has_onsite, nstep, a, grid, smem, device, st);
    case 3: return launch_k<3>(mode, C, has_onsite, nstep, a, grid, smem, device, st);
    case 4: return launch_k<4>(mode, C, has_onsite, nstep, a, grid, smem, device, st);
    case 6: return launch_k<6>(mode, C, has_onsite, nstep, a, grid, smem, device, st);
    }
    return cudaErrorInvalidValue;
}
