// kg_staged_impl.cuh — template dispatch (R, mode, ONS, DICT) of kg_staged_kernel for ONE row
// width KG_STAGED_K, included by kg_staged_k<K>.cu.  Each such file is its own translation unit.
#include "kg_staged.cuh"
#include "kg_staged_launch.h"
#include "kg_smem_config.h"

#ifndef KG_STAGED_K
#error "define KG_STAGED_K before including kg_staged_impl.cuh"
#endif

namespace {

template <int R, int K, int MODE, bool ONS, bool DICT>
cudaError_t launch_t(const StagedArgs &a, const StagedLaunch &l, cudaStream_t st)
{
    static KgSmemConfig cfg_once;
    if (cudaError_t e = cfg_once.ensure(kg_staged_kernel<R, K, MODE, ONS, DICT>, l.device, l.smem)) return e;
    if (!l.pdl) {
        kg_staged_kernel<R, K, MODE, ONS, DICT><<<l.grid, SG_THREADS, l.smem, st>>>(a);
        return cudaGetLastError();
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)l.grid);
    cfg.blockDim = dim3(SG_THREADS);
    cfg.dynamicSmemBytes = l.smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kg_staged_kernel<R, K, MODE, ONS, DICT>, a);
}

template <int R, int K, int MODE>
cudaError_t launch_rm(const StagedArgs &a, const StagedLaunch &l, cudaStream_t st)
{
    if (l.has_onsite) return l.dict ? launch_t<R, K, MODE, true, true>(a, l, st) : launch_t<R, K, MODE, true, false>(a, l, st);
    return l.dict ? launch_t<R, K, MODE, false, true>(a, l, st) : launch_t<R, K, MODE, false, false>(a, l, st);
}

template <int K, int MODE>
cudaError_t launch_m(int R, const StagedArgs &a, const StagedLaunch &l, cudaStream_t st)
{
    switch (R) {
    case 1: return launch_rm<1, K, MODE>(a, l, st);
    case 2: return launch_rm<2, K, MODE>(a, l, st);
    case 4: return launch_rm<4, K, MODE>(a, l, st);
    case 8: return launch_rm<8, K, MODE>(a, l, st);
    case 16:
        if constexpr (MODE == MODE_EVO || MODE == MODE_MOMX || MODE == MODE_CLEN) return launch_rm<16, K, MODE>(a, l, st);
        break;
    }
    return cudaErrorInvalidValue;
}

template <int K>
cudaError_t launch_k(int mode, int R, const StagedArgs &a, const StagedLaunch &l, cudaStream_t st)
{
    switch (mode) {
    case MODE_MOM: return launch_m<K, MODE_MOM>(R, a, l, st);
    case MODE_EVO: return launch_m<K, MODE_EVO>(R, a, l, st);
    case MODE_PAIR: return launch_m<K, MODE_PAIR>(R, a, l, st);
    case MODE_MOM2: return launch_m<K, MODE_MOM2>(R, a, l, st);
    case MODE_MOMX: return launch_m<K, MODE_MOMX>(R, a, l, st);
    case MODE_CLEN: return launch_m<K, MODE_CLEN>(R, a, l, st);
    case MODE_PCLEN: return launch_m<K, MODE_PCLEN>(R, a, l, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace

#define KG_CAT2(a, b) a##b
#define KG_CAT(a, b) KG_CAT2(a, b)
cudaError_t KG_CAT(kg_staged_launch_k, KG_STAGED_K)(int mode, int R, const StagedArgs &a, const StagedLaunch &l, cudaStream_t st)
{
    return launch_k<KG_STAGED_K>(mode, R, a, l, st);
}
