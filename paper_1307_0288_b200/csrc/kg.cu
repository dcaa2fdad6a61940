// kg.cu — host side of libkg: the C ABI of include/kg.h, workspace, driver loops (a7).
// All arithmetic on vectors runs in the kernels of kg_kernels.cuh; this file only computes the
// O(N_p) series coefficients (Bessel functions, eq 36) on the host and enqueues kernels.
#include "kg.h"
#include "kg_kernels.cuh"
#include "kg_staged.cuh"
#include "kg_staged_launch.h"
#include "kg_partition.h"
#include "kg_tb2.cuh"
#include "kg_tb2_launch.h"
#include "kg_small.cuh"
#include "kg_small_launch.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#define KG_HBAR 0.6582119569 /* eV fs */

static thread_local char g_err[512] = "";

static int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

// Nothing may throw across the C ABI: the bodies of the extern "C" calls run inside this guard
// (std::vector growth in the host-side tables can throw std::bad_alloc).
template <class F>
static int guarded(F &&body)
{
    try {
        return body();
    } catch (const std::bad_alloc &) {
        return fail(KG_ENOMEM, "host allocation failed");
    } catch (const std::exception &e) {
        return fail(KG_ECUDA, "internal error: %s", e.what());
    } catch (...) {
        return fail(KG_ECUDA, "internal error");
    }
}

#define CUDA_TRY(expr)                                                                        \
    do {                                                                                      \
        cudaError_t e_ = (expr);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return fail(e_ == cudaErrorMemoryAllocation ? KG_ENOMEM : KG_ECUDA, "%s: %s",     \
                        #expr, cudaGetErrorString(e_));                                       \
    } while (0)

extern "C" const char *kg_last_error(void) { return g_err; }

// options read by kg_create_hamiltonian[_csr] (set before create; process-wide)
static int g_reorder = -1;                    // KG_OPT_REORDER: -1 auto, 0 off, 1 always
#define KG_REORDER_MIN_SITES ((int64_t)1 << 16)
#ifndef KG_REORDER_GROUP
#define KG_REORDER_GROUP 8           // consecutive caller sites that stay together (kg_partition.h)
#endif
#ifndef KG_REORDER_LEAF
#define KG_REORDER_LEAF 64
#endif

extern "C" int kg_set_default_option(int option, int64_t value)
{
    return guarded([&]() -> int {
    switch (option) {
    case KG_OPT_REORDER: g_reorder = value < 0 ? -1 : (value != 0); return KG_OK;
    }
    return fail(KG_EINVAL, "kg_set_default_option: option %d has no process-wide default", option);
    });
}

// --------------------------------------------------------------------------------------
// handle
// --------------------------------------------------------------------------------------
enum {
    WS_TA = 0, WS_TB, WS_DA, WS_DB,        // Chebyshev vectors of the a- and d-chains
    WS_S0, WS_S1, WS_X0, WS_X1,            // persistent time-stepping states (D6)
    WS_PHIL,                               // V psi_k (VAC left vector)
    WS_PART,                               // per-block moment partials [M][B][R]
    WS_IN0, WS_IN1, WS_OUT0, WS_OUT1,      // internal-order copies of caller vectors (host pointers and / or re-ordered sites)
    WS_RAW0, WS_RAW1,                      // caller-order staging between a host pointer and the permutation kernel
    WS_TC, WS_TD,                          // third / fourth Chebyshev vector of the two-step kernel
    WS_MU,                                 // device moments when the caller's mu is host memory
    WS_PLANE,                              // one column pair [n][2] of a wider batch (two-step kernel on R > 2)
    WS_COUNT
};

struct GraphEntry {
    const void *phiL, *phiR;
    int ldL, ldR, R, M, grid, threads, dbl;
    cudaGraphExec_t exec;
};

// per-tile plan of the two-step kernel (kg_tb2.cuh), one per column count C = 1, 2
struct Tb2Plan {
    bool built, ok;
    int cap1, cap2, ntiles;
    int2 *tinfo;
    uint16_t *rows;
    int32_t *hid;
    double *hons;
    size_t bytes;
};

struct kg_hamiltonian {
    int64_t n, ns;
    int kmax;
    double s, e0, period;
    bool has_onsite;
    int32_t *nl;
    int32_t *nlp;             // (dictionary id << 28) | NL_ik, for the staged kernel (DICT)
    int32_t *perm, *iperm;    // site re-ordering (kg_partition.h): internal i = caller perm[i]; NULL: caller order
    double *hop, *xhop, *onsite;
    double dict[16];          // hopping dictionary, dict[0] = 0
    int ndict;                // entries in use (0: hoppings do not fit a dictionary)
    int staged, stages, staged_ctas, alternate, doubling, clenshaw, pdl;   // options of the staged kernel
    int tb2;                  // KG_OPT_TWO_STEP: -1 auto, 0 off, 1 whenever a plan exists
    int big_cluster;          // 1 until a 16-CTA cluster launch has been refused by the device
    int one_launch;           // KG_OPT_ONE_LAUNCH: -1 auto, 0 off: the moment loop of launch-bound sizes as one cluster kernel
    int check_input;          // KG_OPT_CHECK_INPUT: input vectors are scanned for NaN / Inf (one pass + a synchronisation)
    unsigned int *d_flag;     // device flag of that scan
    Tb2Plan tbp[2];
    void *ws[WS_COUNT];
    size_t ws_bytes[WS_COUNT];
    size_t matrix_bytes;
    int device, num_sms, l2_bytes;
    int threads, blocks_per_sm, use_graphs;
    int64_t launches;
    std::vector<GraphEntry> graphs;
};

static int ws_get(kg_hamiltonian *h, int slot, size_t bytes, void **out)
{
    if (h->ws_bytes[slot] < bytes) {
        if (h->ws[slot]) {
            // a cached graph may reference the old buffer
            for (auto &g : h->graphs) cudaGraphExecDestroy(g.exec);
            h->graphs.clear();
            CUDA_TRY(cudaDeviceSynchronize());
            CUDA_TRY(cudaFree(h->ws[slot]));
            h->ws[slot] = nullptr;
            h->ws_bytes[slot] = 0;
        }
        CUDA_TRY(cudaMalloc(&h->ws[slot], bytes));
        h->ws_bytes[slot] = bytes;
    }
    *out = h->ws[slot];
    return KG_OK;
}

static bool is_device_ptr(const void *p)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

static int grid_for(const kg_hamiltonian *h, int64_t elems);

// Internal-order device view of a caller vector [n][R] (host or device pointer, caller's site order):
// the pointer itself when it is a device pointer and the sites are not re-ordered; else a copy in
// workspace slot `slot` (host -> device copy and / or the permutation kernel).
static int vec_in_raw(kg_hamiltonian *h, int slot, const void *p, int R, cudaStream_t st, const void **dev);
static int vec_in(kg_hamiltonian *h, int slot, const void *p, int R, cudaStream_t st, const void **dev)
{
    int rc = vec_in_raw(h, slot, p, R, st, dev);
    if (rc || !h->check_input) return rc;
    // KG_OPT_CHECK_INPUT: "non-finite input -> KG_EINVAL" for state vectors costs one pass and a synchronisation
    if (!h->d_flag) CUDA_TRY(cudaMalloc(&h->d_flag, 4));
    CUDA_TRY(cudaMemsetAsync(h->d_flag, 0, 4, st));
    kg_check_finite<<<grid_for(h, h->n * R), 256, 0, st>>>((const double *)*dev, h->n * R * 2, h->d_flag);
    h->launches++;
    unsigned int bad = 0;
    CUDA_TRY(cudaMemcpyAsync(&bad, h->d_flag, 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (bad) return fail(KG_EINVAL, "input vector holds a non-finite value");
    return KG_OK;
}
static int vec_in_raw(kg_hamiltonian *h, int slot, const void *p, int R, cudaStream_t st, const void **dev)
{
    const size_t bytes = (size_t)h->n * R * 16;
    const bool on_dev = is_device_ptr(p);
    if (on_dev && !h->perm) { *dev = p; return KG_OK; }
    void *d;
    int rc = ws_get(h, slot, bytes, &d);
    if (rc) return rc;
    const void *src = p;
    if (!on_dev) {
        void *raw = d;
        if (h->perm && (rc = ws_get(h, WS_RAW0 + (slot == WS_IN1 ? 1 : 0), bytes, &raw))) return rc;
        CUDA_TRY(cudaMemcpyAsync(raw, p, bytes, cudaMemcpyHostToDevice, st));
        src = raw;
    }
    if (h->perm) {
        kg_permute_rows<<<grid_for(h, h->n * R), 256, 0, st>>>((const c128 *)src, (c128 *)d, h->perm, h->n, R);
        h->launches++;
        CUDA_TRY(cudaGetLastError());
    }
    *dev = d;
    return KG_OK;
}

// Output vector [n][R]: `dev` is the internal-order device buffer the kernels write; vec_out_finish
// brings it to the caller's array (inverse permutation and / or device -> host copy).
struct VecOut { void *user; void *dev; int R; int slot; bool host; };
static int vec_out(kg_hamiltonian *h, int slot, void *p, int R, VecOut *o)
{
    o->user = p; o->R = R; o->slot = slot; o->host = !is_device_ptr(p);
    if (!o->host && !h->perm) { o->dev = p; return KG_OK; }
    return ws_get(h, slot, (size_t)h->n * R * 16, &o->dev);
}
static int vec_out_finish(kg_hamiltonian *h, const VecOut &o, cudaStream_t st)
{
    const size_t bytes = (size_t)h->n * o.R * 16;
    if (!o.host && !h->perm) return KG_OK;
    const void *src = o.dev;
    if (h->perm) {
        void *dst = o.user;
        int rc;
        if (o.host && (rc = ws_get(h, WS_RAW0 + (o.slot == WS_OUT1 ? 1 : 0), bytes, &dst))) return rc;
        kg_permute_rows<<<grid_for(h, h->n * o.R), 256, 0, st>>>((const c128 *)o.dev, (c128 *)dst, h->iperm, h->n, o.R);
        h->launches++;
        CUDA_TRY(cudaGetLastError());
        src = dst;
    }
    if (o.host) CUDA_TRY(cudaMemcpyAsync(o.user, src, bytes, cudaMemcpyDeviceToHost, st));
    return KG_OK;
}

static int grid_for(const kg_hamiltonian *h, int64_t elems)
{
    int64_t want = (elems + h->threads - 1) / h->threads;
    int64_t cap = (int64_t)h->num_sms * h->blocks_per_sm;
    if (want < 1) want = 1;
    return (int)(want < cap ? want : cap);
}

// --------------------------------------------------------------------------------------
// kernel dispatch
// --------------------------------------------------------------------------------------
template <int R, int MODE, bool FIRST>
static cudaError_t launch_rmf(const kg_hamiltonian *h, const StepArgs &a, int grid, cudaStream_t st)
{
    const int th = h->threads;
    if (h->kmax == 3) {
        if (h->has_onsite) kg_step_kernel<R, MODE, FIRST, true, 3><<<grid, th, 0, st>>>(a);
        else kg_step_kernel<R, MODE, FIRST, false, 3><<<grid, th, 0, st>>>(a);
    } else {
        if (h->has_onsite) kg_step_kernel<R, MODE, FIRST, true, 0><<<grid, th, 0, st>>>(a);
        else kg_step_kernel<R, MODE, FIRST, false, 0><<<grid, th, 0, st>>>(a);
    }
    return cudaGetLastError();
}

template <int MODE, bool FIRST>
static cudaError_t launch_mf(const kg_hamiltonian *h, int R, const StepArgs &a, int grid, cudaStream_t st)
{
    switch (R) {
    case 1: return launch_rmf<1, MODE, FIRST>(h, a, grid, st);
    case 2: return launch_rmf<2, MODE, FIRST>(h, a, grid, st);
    case 4: return launch_rmf<4, MODE, FIRST>(h, a, grid, st);
    case 8: return launch_rmf<8, MODE, FIRST>(h, a, grid, st);
    case 16: return launch_rmf<16, MODE, FIRST>(h, a, grid, st);
    }
    return cudaErrorInvalidValue;
}

static cudaError_t launch_step(kg_hamiltonian *h, int mode, bool first, int R, const StepArgs &a,
                               int grid, cudaStream_t st)
{
    h->launches++;
    switch (mode) {
    case MODE_MOM: return first ? launch_mf<MODE_MOM, true>(h, R, a, grid, st) : launch_mf<MODE_MOM, false>(h, R, a, grid, st);
    case MODE_EVO: return first ? launch_mf<MODE_EVO, true>(h, R, a, grid, st) : launch_mf<MODE_EVO, false>(h, R, a, grid, st);
    case MODE_PAIR: return first ? launch_mf<MODE_PAIR, true>(h, R, a, grid, st) : launch_mf<MODE_PAIR, false>(h, R, a, grid, st);
    case MODE_VEL: return launch_mf<MODE_VEL, true>(h, R, a, grid, st);
    case MODE_MOM2: return first ? launch_mf<MODE_MOM2, true>(h, R, a, grid, st) : launch_mf<MODE_MOM2, false>(h, R, a, grid, st);
    case MODE_MOMX: return first ? launch_mf<MODE_MOMX, true>(h, R, a, grid, st) : launch_mf<MODE_MOMX, false>(h, R, a, grid, st);
    }
    return cudaErrorInvalidValue;
}

static StepArgs base_args(const kg_hamiltonian *h)
{
    StepArgs a;
    memset(&a, 0, sizeof(a));
    a.nl = h->nl; a.hop = h->hop; a.xhop = h->xhop; a.onsite = h->onsite;
    a.n = h->n; a.ns = h->ns; a.kmax = h->kmax;
    a.alpha = 2.0;
    return a;
}

// ---- staged kernels (kg_staged.cuh): plan + dispatch ----
struct StagedPlan { bool ok; int grid, nst, ntiles; size_t smem; };

// The staged kernels are compiled one row width K per translation unit (kg_staged_k<K>.cu) so
// that the build can run them in parallel; kg_staged_launch.h declares their entry points.
static cudaError_t staged_launch(kg_hamiltonian *h, int mode, int R, const StagedArgs &a, const StagedPlan &p, cudaStream_t st)
{
    h->launches++;
    StagedLaunch l;
    l.grid = p.grid; l.smem = p.smem; l.device = h->device; l.has_onsite = h->has_onsite; l.dict = h->ndict > 0;
    // programmatic dependent launch pays where launch latency dominates (config 1: 4.1 -> 2.8 us per
    // sweep); on multi-megabyte sweeps it was measured slower (config 4 MOM2 43 -> 52 us)
    l.pdl = h->pdl > 0 || (h->pdl < 0 && h->n * (int64_t)R <= ((int64_t)1 << 18));
    switch (h->kmax) {
    case 2: return kg_staged_launch_k2(mode, R, a, l, st);
    case 3: return kg_staged_launch_k3(mode, R, a, l, st);
    case 4: return kg_staged_launch_k4(mode, R, a, l, st);
    case 6: return kg_staged_launch_k6(mode, R, a, l, st);
    case 9: return kg_staged_launch_k9(mode, R, a, l, st);
    }
    return cudaErrorInvalidValue;
}

static StagedPlan staged_plan(const kg_hamiltonian *h, int mode, int R)
{
    StagedPlan p;
    memset(&p, 0, sizeof(p));
    if (!h->staged || !sg_k_supported(h->kmax) || R > ((mode == MODE_EVO || mode == MODE_MOMX || mode == MODE_CLEN) ? 16 : 8)) return p;
    const int te = sg_tile_e(mode);
    const size_t stage = (size_t)sg_stage_bytes(R, h->kmax, mode, h->has_onsite, h->ndict > 0);
    const size_t header = (size_t)sg_header_bytes(R);
    // auto: 3 CTAs per SM with a 2-deep ring measured best on configs 4 and 5 (profiles/): deeper
    // rings only take shared memory away from the L1 that serves the out-of-tile gathers.  Fewer
    // CTAs when a stage is too large for that (fp64 hoppings staged).
    int ctas = h->staged_ctas > 0 ? h->staged_ctas : 3, nst = 0;
    for (;; --ctas) {
        const size_t budget = (size_t)228 * 1024 / ctas - 1024;
        nst = h->stages > 0 ? h->stages : (int)((budget - header) / stage);
        if (h->stages == 0 && nst > 2) nst = 2;
        if (nst >= 2 || h->staged_ctas > 0 || ctas == 1) break;
    }
    if (nst > SG_MAX_STAGES) nst = SG_MAX_STAGES;
    if (nst < 2 || header + (size_t)nst * stage > (size_t)227 * 1024) return p;
    p.nst = nst;
    p.smem = header + (size_t)nst * stage;
    const int64_t nt = (h->n * R + te - 1) / te;
    p.ntiles = (int)nt;
    const int64_t cap = (int64_t)h->num_sms * ctas;
    p.grid = (int)(nt < cap ? nt : cap);
    p.ok = true;
    return p;
}

static StagedArgs staged_base_args(const kg_hamiltonian *h, const StagedPlan &sp)
{
    StagedArgs sa;
    memset(&sa, 0, sizeof(sa));
    sa.idx = h->ndict > 0 ? h->nlp : h->nl; sa.hop = h->hop; sa.xhop = h->xhop; sa.onsite = h->onsite;
    memcpy(sa.dict, h->dict, sizeof(sa.dict));
    sa.n = h->n; sa.ns = h->ns; sa.ntiles = sp.ntiles; sa.nstages = sp.nst;
    return sa;
}


// ---- two-step kernel (kg_tb2.cuh): host-side plan + dispatch ----
__global__ void kg_tb2_gather_onsite(const double *__restrict__ onsite, const int32_t *__restrict__ hid,
                                     const int2 *__restrict__ tinfo, int ntiles, int cap1, int cap2,
                                     double *__restrict__ hons)
{
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < (int64_t)ntiles * cap1;
         e += (int64_t)gridDim.x * blockDim.x) {
        const int t = (int)(e / cap1), j = (int)(e - (int64_t)t * cap1);
        hons[e] = j < tinfo[t].x ? onsite[hid[(int64_t)t * (cap1 + cap2) + j]] : 0.0;
    }
}

// Build the per-tile plan for C columns per site from the packed list (dictionary id << 28 | index,
// internal order).  Runs once per handle and C — at create for the handles the automatic choice serves, else at
// the first eligible moments call; synchronises.
static int tb2_build_plan(kg_hamiltonian *h, int C, cudaStream_t st)
{
    Tb2Plan &tp = h->tbp[C - 1];
    tp.built = true;
    tp.ok = false;
    if (!h->nlp || h->ndict <= 0 || !kg_tb2_k_supported(h->kmax)) return KG_OK;
    const int K = h->kmax, KP = tb_kp(K), CS = tb_cs(C);
    const int64_t n = h->n, ns = h->ns;
    const int ntiles = (int)((n + CS - 1) / CS);
    std::vector<int32_t> idx((size_t)ns * K);
    CUDA_TRY(cudaMemcpyAsync(idx.data(), h->nlp, (size_t)ns * K * 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    // pass 1 and 2 share the marker arrays: mark[m] = tile that last touched m, slot[m] = its local slot
    std::vector<int32_t> mark((size_t)n, -1), slot((size_t)n, 0);
    std::vector<int2> tinfo((size_t)ntiles);
    std::vector<std::vector<int32_t>> halo((size_t)ntiles);    // H1 then H2 ids per tile
    int max1 = 0, max2 = 0;
    for (int t = 0; t < ntiles; ++t) {
        const int64_t s0 = (int64_t)t * CS, s1 = std::min<int64_t>(n, s0 + CS);
        std::vector<int32_t> &hl = halo[(size_t)t];
        for (int64_t i = s0; i < s1; ++i)
            for (int k = 0; k < K; ++k) {
                const int32_t m = idx[(size_t)k * ns + i] & SG_IDX_MASK;
                if (m >= s0 && m < s1) continue;
                if (mark[(size_t)m] != t) { mark[(size_t)m] = t; slot[(size_t)m] = CS + (int)hl.size(); hl.push_back(m); }
            }
        const int n1 = (int)hl.size();
        for (int j = 0; j < n1; ++j) {
            const int32_t g = hl[(size_t)j];
            for (int k = 0; k < K; ++k) {
                const int32_t m = idx[(size_t)k * ns + g] & SG_IDX_MASK;
                if (m >= s0 && m < s1) continue;
                if (mark[(size_t)m] != t) { mark[(size_t)m] = t; slot[(size_t)m] = CS + (int)hl.size(); hl.push_back(m); }
            }
        }
        const int n2 = (int)hl.size() - n1;
        tinfo[(size_t)t] = make_int2(n1, n2);
        max1 = std::max(max1, n1); max2 = std::max(max2, n2);
    }
    const int cap1 = std::max(8, (max1 + 7) / 8 * 8), cap2 = std::max(8, (max2 + 7) / 8 * 8);
    if (CS + cap1 + cap2 > TB_SLOT_MASK + 1 || TB_HEADER + 2 * tb_stage_bytes(C, K, cap1, cap2) > (size_t)227 * 1024) return KG_OK;
    // pass 2: tile-local rows (own rows, then H1 rows)
    const size_t rstride = (size_t)(CS + cap1) * KP;
    std::vector<uint16_t> rows((size_t)ntiles * rstride, 0);
    std::vector<int32_t> hid((size_t)ntiles * (cap1 + cap2), 0);
    for (int t = 0; t < ntiles; ++t) {
        const int64_t s0 = (int64_t)t * CS, s1 = std::min<int64_t>(n, s0 + CS);
        const std::vector<int32_t> &hl = halo[(size_t)t];
        const int n1 = tinfo[(size_t)t].x;
        for (size_t j = 0; j < hl.size(); ++j) {
            mark[(size_t)hl[j]] = t; slot[(size_t)hl[j]] = CS + (int)j;
            hid[(size_t)t * (cap1 + cap2) + j] = hl[j];
        }
        uint16_t *rt = rows.data() + (size_t)t * rstride;
        auto fill = [&](int row, int64_t site) {
            for (int k = 0; k < K; ++k) {
                const uint32_t w = (uint32_t)idx[(size_t)k * ns + site];
                const int32_t m = (int32_t)(w & SG_IDX_MASK);
                const int sl = (m >= s0 && m < s1) ? (int)(m - s0) : slot[(size_t)m];
                rt[(size_t)row * KP + k] = (uint16_t)(((w >> 28) << 12) | (uint32_t)sl);
            }
            for (int k = K; k < KP; ++k) rt[(size_t)row * KP + k] = (uint16_t)row;      // unused: id 0 (value 0)
        };
        for (int64_t i = s0; i < s1; ++i) fill((int)(i - s0), i);
        for (int j = 0; j < n1; ++j) fill(CS + j, hl[(size_t)j]);
    }
    if (cudaMalloc(&tp.tinfo, (size_t)ntiles * sizeof(int2)) != cudaSuccess ||
        cudaMalloc(&tp.rows, rows.size() * 2) != cudaSuccess || cudaMalloc(&tp.hid, hid.size() * 4) != cudaSuccess ||
        cudaMalloc(&tp.hons, (size_t)ntiles * cap1 * 8) != cudaSuccess) {
        // no room for the plan: not an error of the call — release the part that was allocated and leave
        // tp.ok = false, the one-step kernels serve the handle
        cudaGetLastError();
        cudaFree(tp.tinfo); cudaFree(tp.rows); cudaFree(tp.hid); cudaFree(tp.hons);
        tp.tinfo = nullptr; tp.rows = nullptr; tp.hid = nullptr; tp.hons = nullptr;
        return KG_OK;
    }
    tp.bytes = (size_t)ntiles * sizeof(int2) + rows.size() * 2 + hid.size() * 4 + (size_t)ntiles * cap1 * 8;
    CUDA_TRY(cudaMemcpyAsync(tp.tinfo, tinfo.data(), (size_t)ntiles * sizeof(int2), cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(tp.rows, rows.data(), rows.size() * 2, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(tp.hid, hid.data(), hid.size() * 4, cudaMemcpyHostToDevice, st));
    kg_tb2_gather_onsite<<<std::min<int64_t>(((int64_t)ntiles * cap1 + 255) / 256, (int64_t)h->num_sms * 8), 256, 0, st>>>(
        h->onsite, tp.hid, tp.tinfo, ntiles, cap1, cap2, tp.hons);
    h->launches++;
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaStreamSynchronize(st));             // the host vectors go out of scope
    tp.cap1 = cap1; tp.cap2 = cap2; tp.ntiles = ntiles;
    tp.ok = true;
    return KG_OK;
}

struct Tb2Launch { bool ok; int grid, nst; size_t smem; };

// Is the two-step kernel to be used for a doubling moment loop on C contiguous columns?
static int tb2_plan(kg_hamiltonian *h, int mode, int C, int nplanes, cudaStream_t st, Tb2Launch *out)
{
    out->ok = false;
    if (h->tb2 == 0 || !h->staged || !h->doubling || C > 2 || (mode == MODE_MOMX && C != 2) ||
        (mode != MODE_MOM2 && mode != MODE_MOMX))
        return KG_OK;
    const int64_t nt = (h->n + tb_cs(C) - 1) / tb_cs(C);
    if (h->tb2 < 0 && (!h->perm || nt * nplanes < 4 * (int64_t)h->num_sms)) return KG_OK;    // auto: re-ordered sites, >= 4 tiles per SM
    // auto, wider batches as column-pair planes: only when three vectors of the batch do not fit L2 — an
    // L2-resident wide batch is served faster by the one-step kernel, which shares a matrix row among all
    // R columns (config 2: 13.8 us per one-step sweep of 8 columns against 35 us per two-step pass)
    if (h->tb2 < 0 && nplanes > 1 && (int64_t)h->n * C * nplanes * 48 <= (int64_t)h->l2_bytes) return KG_OK;
    if (nplanes > h->num_sms) return KG_OK;
    Tb2Plan &tp = h->tbp[C - 1];
    if (!tp.built) { int rc = tb2_build_plan(h, C, st); if (rc) return rc; }
    if (!tp.ok) return KG_OK;
    // one persistent CTA per SM; as many shared-memory stages as fit (2..4)
    const size_t stage = tb_stage_bytes(C, h->kmax, tp.cap1, tp.cap2);
    out->nst = (int)std::min<size_t>(h->stages > 0 ? (size_t)h->stages : (size_t)3, ((size_t)227 * 1024 - TB_HEADER) / stage);
    if (out->nst > TB_MAX_STAGES) out->nst = TB_MAX_STAGES;
    if (out->nst < 2) return KG_OK;
    out->smem = TB_HEADER + (size_t)out->nst * stage;
    out->grid = (int)std::min<int64_t>(tp.ntiles, (int64_t)h->num_sms / nplanes);     // CTAs per plane
    out->ok = true;
    return KG_OK;
}

static Tb2Args tb2_base_args(const kg_hamiltonian *h, int C)
{
    const Tb2Plan &tp = h->tbp[C - 1];
    Tb2Args a;
    memset(&a, 0, sizeof(a));
    a.tinfo = tp.tinfo; a.rows = tp.rows; a.hid = tp.hid; a.hons = tp.hons; a.onsite = h->onsite;
    memcpy(a.dict, h->dict, sizeof(a.dict));
    a.n = h->n; a.cap1 = tp.cap1; a.cap2 = tp.cap2; a.ntiles = tp.ntiles;
    a.nplanes = 1; a.plane_stride = 0;
    return a;
}

static bool r_ok(int R, bool allow16) { return R == 1 || R == 2 || R == 4 || R == 8 || (allow16 && R == 16); }

// --------------------------------------------------------------------------------------
// Bessel coefficients (R4): Miller backward recurrence in long double, normalised by
// J_0 + 2 sum_k J_2k = 1.  N_p = 1 + max{m : |J_m(x)| >= eps}, scanned from above.
// --------------------------------------------------------------------------------------
static void bessel_table(double x, double eps, std::vector<double> &j)
{
    const double ax = std::fabs(x);
    if (eps <= 0.0) eps = 1e-15;
    if (ax == 0.0) { j.assign(1, 1.0); return; }
    // start high enough that J_start/J_max is far below double rounding
    int mtop = (int)std::ceil(ax) + 64 + (int)std::ceil(40.0 * std::cbrt(ax));
    mtop += mtop & 1;
    std::vector<long double> v((size_t)mtop + 2, 0.0L);
    long double jp1 = 0.0L, jm = 1e-300L;
    v[mtop] = jm;
    for (int m = mtop; m >= 1; --m) {
        const long double jm1 = (2.0L * m / (long double)ax) * jm - jp1;
        jp1 = jm; jm = jm1;
        v[m - 1] = jm;
        if (fabsl(jm) > 1e300L) {                     // rescale to stay in range
            for (int q = m - 1; q <= mtop; ++q) v[q] *= 1e-300L;
            jm *= 1e-300L; jp1 *= 1e-300L;
        }
    }
    long double norm = v[0];
    for (int m = 2; m <= mtop; m += 2) norm += 2.0L * v[m];
    int np = 1;
    for (int m = mtop; m >= 0; --m)
        if (fabsl(v[m] / norm) >= (long double)eps) { np = m + 1; break; }
    j.resize(np);
    for (int m = 0; m < np; ++m) {
        double val = (double)(v[m] / norm);
        if (x < 0.0 && (m & 1)) val = -val;           // J_m(-x) = (-1)^m J_m(x)
        j[m] = val;
    }
}

extern "C" int kg_bessel_terms(double x, double bessel_eps, int *np_out, double *j, int cap)
{
    return guarded([&]() -> int {
    if (!np_out || !std::isfinite(x)) return fail(KG_EINVAL, "kg_bessel_terms: bad argument");
    std::vector<double> t;
    bessel_table(x, bessel_eps, t);
    *np_out = (int)t.size();
    if (j) for (int m = 0; m < (int)t.size() && m < cap; ++m) j[m] = t[m];
    return KG_OK;
    });
}

// c_m = (2 - delta_m0) (-+ i)^m J_m(x) * exp(-i E0 dt/hbar), upper sign for dt > 0 (eq 36)
static void series_coefficients(const kg_hamiltonian *h, double dt_fs, double eps, std::vector<c128> &c)
{
    const double xarg = h->s * std::fabs(dt_fs) / KG_HBAR;
    std::vector<double> j;
    bessel_table(xarg, eps, j);
    const double ph = -h->e0 * dt_fs / KG_HBAR;
    const double pr = std::cos(ph), pi = std::sin(ph);
    c.resize(j.size());
    for (size_t m = 0; m < j.size(); ++m) {
        const double mag = (m == 0 ? 1.0 : 2.0) * j[m];
        double re = 0.0, im = 0.0;                    // (-+ i)^m
        switch (m & 3) {
        case 0: re = 1.0; break;
        case 1: im = dt_fs > 0 ? -1.0 : 1.0; break;
        case 2: re = -1.0; break;
        case 3: im = dt_fs > 0 ? 1.0 : -1.0; break;
        }
        re *= mag; im *= mag;
        if (h->e0 != 0.0) c[m] = make_double2(re * pr - im * pi, re * pi + im * pr);
        else c[m] = make_double2(re, im);
    }
}

// --------------------------------------------------------------------------------------
// create / destroy
// --------------------------------------------------------------------------------------
static int create_from_device_list(kg_hamiltonian **out, int64_t n, int kmax, const int32_t *d_nn,
                                   const int32_t *d_nl, const double *d_hop, const double *d_ons,
                                   const double *d_x, double period, double e0, double s,
                                   cudaStream_t st)
{
    kg_hamiltonian *h = new (std::nothrow) kg_hamiltonian();
    if (!h) return fail(KG_ENOMEM, "host allocation failed");
    h->n = n; h->ns = (n + SG_TILE_E - 1) / SG_TILE_E * SG_TILE_E; h->kmax = kmax;
    h->s = s; h->e0 = e0; h->period = period;
    h->nl = h->nlp = nullptr; h->hop = h->xhop = h->onsite = nullptr;
    h->perm = h->iperm = nullptr;
    h->tb2 = -1; memset(h->tbp, 0, sizeof(h->tbp)); h->big_cluster = 1;
    h->check_input = 0; h->d_flag = nullptr; h->one_launch = -1;
    h->ndict = 0; h->staged = 1; h->stages = 0; h->staged_ctas = 0; h->alternate = 1; h->doubling = 1; h->clenshaw = 1; h->pdl = -1;
    memset(h->dict, 0, sizeof(h->dict));
    memset(h->ws, 0, sizeof(h->ws));
    memset(h->ws_bytes, 0, sizeof(h->ws_bytes));
    h->launches = 0;
    h->threads = 256; h->blocks_per_sm = 6; h->use_graphs = -1;
    unsigned int *d_flags = nullptr;
    int rc = KG_OK;
    auto cleanup = [&](int code) { if (d_flags) cudaFree(d_flags); kg_destroy_hamiltonian(h); return code; };
    cudaError_t e;
    if ((e = cudaGetDevice(&h->device)) != cudaSuccess ||
        (e = cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, h->device)) != cudaSuccess ||
        (e = cudaDeviceGetAttribute(&h->l2_bytes, cudaDevAttrL2CacheSize, h->device)) != cudaSuccess)
        return cleanup(fail(KG_ECUDA, "device query: %s", cudaGetErrorString(e)));
    const size_t slab = (size_t)h->ns * kmax;
    h->matrix_bytes = slab * (4 + 8 + 8) + (size_t)h->ns * 8;
    if ((e = cudaMalloc(&h->nl, slab * 4)) != cudaSuccess || (e = cudaMalloc(&h->hop, slab * 8)) != cudaSuccess ||
        (e = cudaMalloc(&h->xhop, slab * 8)) != cudaSuccess || (e = cudaMalloc(&h->onsite, (size_t)h->ns * 8)) != cudaSuccess ||
        (e = cudaMalloc(&d_flags, 16)) != cudaSuccess)
        return cleanup(fail(KG_ENOMEM, "matrix allocation: %s", cudaGetErrorString(e)));
    if ((e = cudaMemsetAsync(d_flags, 0, 16, st)) != cudaSuccess)
        return cleanup(fail(KG_ECUDA, "memset: %s", cudaGetErrorString(e)));
    // site re-ordering: recursive breadth-first bisection of the neighbour list on the host
    // (kg_partition.h), so that every aligned block of consecutive internal sites is a compact patch
    if (g_reorder > 0 || (g_reorder < 0 && n >= KG_REORDER_MIN_SITES)) try {
        std::vector<int32_t> h_nn((size_t)n), h_nl((size_t)n * kmax), perm, iperm((size_t)n);
        if ((e = cudaMemcpyAsync(h_nn.data(), d_nn, (size_t)n * 4, cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
            (e = cudaMemcpyAsync(h_nl.data(), d_nl, (size_t)n * kmax * 4, cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
            (e = cudaStreamSynchronize(st)) != cudaSuccess)
            return cleanup(fail(KG_ECUDA, "neighbour list to host: %s", cudaGetErrorString(e)));
        kg_partition_grouped(n, kmax, h_nn.data(), h_nl.data(), KG_REORDER_LEAF, KG_REORDER_GROUP, perm);
        for (int64_t i = 0; i < n; ++i) iperm[(size_t)perm[(size_t)i]] = (int32_t)i;
        if ((e = cudaMalloc(&h->perm, (size_t)n * 4)) != cudaSuccess || (e = cudaMalloc(&h->iperm, (size_t)n * 4)) != cudaSuccess)
            return cleanup(fail(KG_ENOMEM, "permutation allocation: %s", cudaGetErrorString(e)));
        h->matrix_bytes += (size_t)n * 8;
        if ((e = cudaMemcpyAsync(h->perm, perm.data(), (size_t)n * 4, cudaMemcpyHostToDevice, st)) != cudaSuccess ||
            (e = cudaMemcpyAsync(h->iperm, iperm.data(), (size_t)n * 4, cudaMemcpyHostToDevice, st)) != cudaSuccess ||
            (e = cudaStreamSynchronize(st)) != cudaSuccess)          // the host vectors go out of scope
            return cleanup(fail(KG_ECUDA, "permutation upload: %s", cudaGetErrorString(e)));
    } catch (const std::bad_alloc &) {       // the host tables of the bisection: release the half-built handle
        return cleanup(fail(KG_ENOMEM, "host allocation failed in the site re-ordering"));
    }
    const int grid = (int)std::min<int64_t>((h->ns + 255) / 256, (int64_t)h->num_sms * 8);
    kg_build_matrix<<<grid, 256, 0, st>>>(n, h->ns, kmax, d_nn, d_nl, d_hop, d_ons, d_x, period, e0, s,
                                          h->perm, h->iperm, h->nl, h->hop, h->xhop, h->onsite, d_flags,
                                          (unsigned long long *)(d_flags + 2));
    h->launches++;
    unsigned int host_flags[4];
    if ((e = cudaGetLastError()) != cudaSuccess ||
        (e = cudaMemcpyAsync(host_flags, d_flags, 16, cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
        (e = cudaStreamSynchronize(st)) != cudaSuccess)
        return cleanup(fail(KG_ECUDA, "kg_build_matrix: %s", cudaGetErrorString(e)));
    double gersh;
    memcpy(&gersh, host_flags + 2, 8);
    if (host_flags[0] & 2u) rc = fail(KG_EINVAL, "nn[i] outside [0, kmax]");
    else if (host_flags[0] & 1u) rc = fail(KG_EINVAL, "neighbour index outside [0, n)");
    else if (host_flags[0] & 4u) rc = fail(KG_EINVAL, "non-finite hopping, on-site energy or coordinate");
    else if (host_flags[0] & 8u) rc = fail(KG_EINVAL, "H is not symmetric (H_mi != H_im, missing reverse bond, or a diagonal entry in the list)");
    else if (gersh > s * (1.0 + 1e-12))
        rc = fail(KG_ESPECTRUM, "Gershgorin bound %.6g eV of (H - E0) exceeds scale %.6g eV", gersh, s);
    if (rc) return cleanup(rc);
    h->has_onsite = d_ons != nullptr || e0 != 0.0;
    // hopping dictionary for the staged kernel: <= 15 distinct non-zero values of H_ik/s
    if (sg_k_supported(kmax) && n <= (int64_t)SG_IDX_MASK + 1) {
        unsigned long long tab[16];
        for (int q = 0; q < 16; ++q) tab[q] = SG_DICT_EMPTY;
        tab[15] = 0;   // overflow flag lives in slot 15
        unsigned long long *d_tab = nullptr;
        double *d_dict = nullptr;
        if ((e = cudaMalloc(&d_tab, 16 * 8)) != cudaSuccess || (e = cudaMalloc(&d_dict, 16 * 8)) != cudaSuccess ||
            (e = cudaMalloc(&h->nlp, slab * 4)) != cudaSuccess) {
            cudaFree(d_tab); cudaFree(d_dict);
            return cleanup(fail(KG_ENOMEM, "dictionary allocation: %s", cudaGetErrorString(e)));
        }
        h->matrix_bytes += slab * 4;
        auto cleanup2 = [&](int code) { cudaFree(d_tab); cudaFree(d_dict); return cleanup(code); };
        if ((e = cudaMemcpyAsync(d_tab, tab, sizeof(tab), cudaMemcpyHostToDevice, st)) != cudaSuccess)
            return cleanup2(fail(KG_ECUDA, "dictionary: %s", cudaGetErrorString(e)));
        kg_dict_collect<<<grid, 256, 0, st>>>(h->hop, (int64_t)slab, d_tab, (unsigned int *)(d_tab + 15));
        h->launches++;
        if ((e = cudaGetLastError()) != cudaSuccess ||
            (e = cudaMemcpyAsync(tab, d_tab, sizeof(tab), cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
            (e = cudaStreamSynchronize(st)) != cudaSuccess)
            return cleanup2(fail(KG_ECUDA, "kg_dict_collect: %s", cudaGetErrorString(e)));
        if ((unsigned int)tab[15] == 0) {
            double vals[15];
            int nvals = 0;
            for (int q = 0; q < 15; ++q)
                if (tab[q] != SG_DICT_EMPTY) memcpy(&vals[nvals++], &tab[q], 8);
            std::sort(vals, vals + nvals);
            h->ndict = 1 + nvals;
            for (int q = 0; q < nvals; ++q) h->dict[1 + q] = vals[q];
            if ((e = cudaMemcpyAsync(d_dict, h->dict, 16 * 8, cudaMemcpyHostToDevice, st)) != cudaSuccess)
                return cleanup2(fail(KG_ECUDA, "dictionary: %s", cudaGetErrorString(e)));
            kg_dict_pack<<<grid, 256, 0, st>>>(h->nl, h->hop, (int64_t)slab, d_dict, h->ndict, h->nlp);
            h->launches++;
            if ((e = cudaGetLastError()) != cudaSuccess || (e = cudaStreamSynchronize(st)) != cudaSuccess)
                return cleanup2(fail(KG_ECUDA, "kg_dict_pack: %s", cudaGetErrorString(e)));
        } else {
            cudaFree(h->nlp); h->nlp = nullptr; h->matrix_bytes -= slab * 4;
        }
        cudaFree(d_tab); cudaFree(d_dict);
    }
    cudaFree(d_flags);
    d_flags = nullptr;
    // Tile plans of the two-step kernel for the handles on which the automatic choice (tb2_plan) will use it —
    // re-ordered sites, at least four tiles per SM — are built here, so that no moments call has to stop and
    // synchronise for them.  (A handle on which KG_OPT_TWO_STEP is forced later builds its plan at the first
    // moments call, as before.)
    if (h->perm) try {
        for (int C = 1; C <= 2; ++C) {
            const int64_t nt = (n + tb_cs(C) - 1) / tb_cs(C);
            if (nt < 4 * (int64_t)h->num_sms) continue;
            if ((rc = tb2_build_plan(h, C, st))) return cleanup(rc);
        }
    } catch (const std::bad_alloc &) {
        return cleanup(fail(KG_ENOMEM, "host allocation failed in the two-step tile plan"));
    }
    *out = h;
    return KG_OK;
}

static int check_create_args(kg_hamiltonian **out, int64_t n, int64_t kmax, const void *a, const void *b,
                             const void *c, const void *x, double period, double e0, double s)
{
    if (!out) return fail(KG_EINVAL, "out is NULL");
    *out = nullptr;
    if (!a || !b || !c || !x) return fail(KG_EINVAL, "NULL array argument");
    if (n <= 0 || n >= ((int64_t)1 << 31) - 1024) return fail(KG_EINVAL, "n must be in [1, 2^31 - 1024)");
    if (kmax <= 0) return fail(KG_EINVAL, "kmax must be positive");
    if (kmax > 32) return fail(KG_EUNSUPPORTED, "kmax > 32 not supported");
    if (!(s > 0.0) || !std::isfinite(s) || !std::isfinite(e0) || !std::isfinite(period))
        return fail(KG_EINVAL, "scale must be positive and finite; e0 and period finite");
    return KG_OK;
}

// temporary device copies of host inputs for create
struct TmpDev {
    std::vector<void *> ptrs;
    ~TmpDev() { for (void *p : ptrs) cudaFree(p); }
    int get(const void *src, size_t bytes, cudaStream_t st, const void **dev)
    {
        if (!src) { *dev = nullptr; return KG_OK; }
        if (is_device_ptr(src)) { *dev = src; return KG_OK; }
        void *d = nullptr;
        CUDA_TRY(cudaMalloc(&d, bytes));
        ptrs.push_back(d);
        CUDA_TRY(cudaMemcpyAsync(d, src, bytes, cudaMemcpyHostToDevice, st));
        *dev = d;
        return KG_OK;
    }
};

// Stream-ordered temporaries of the handle-free post-processing calls: cudaMallocFromPoolAsync from a
// memory pool the library owns (one per device, created at the first such call there, kept warm:
// release threshold = never, alive until the process exits), cudaFreeAsync when the call returns — no
// cudaMalloc, no cudaFree and no synchronisation once the pool has grown.  The application's default
// pool is left as it is; it only serves as the fallback when the library's pool cannot be created.
struct AsyncTmp {
    cudaStream_t st;
    cudaMemPool_t pool;
    std::vector<void *> ptrs;
    static cudaMemPool_t pool_of_current_device()
    {
        constexpr int MAXDEV = 64;
        static std::once_flag once[MAXDEV];
        static cudaMemPool_t pools[MAXDEV];
        int dev = -1;
        if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAXDEV) { cudaGetLastError(); return nullptr; }
        std::call_once(once[dev], [dev] {
            cudaMemPoolProps props;
            memset(&props, 0, sizeof(props));
            props.allocType = cudaMemAllocationTypePinned;
            props.handleTypes = cudaMemHandleTypeNone;
            props.location.type = cudaMemLocationTypeDevice;
            props.location.id = dev;
            cudaMemPool_t p = nullptr;
            if (cudaMemPoolCreate(&p, &props) != cudaSuccess) { cudaGetLastError(); pools[dev] = nullptr; return; }
            uint64_t keep = UINT64_MAX;
            cudaMemPoolSetAttribute(p, cudaMemPoolAttrReleaseThreshold, &keep);
            pools[dev] = p;
        });
        return pools[dev];
    }
    explicit AsyncTmp(cudaStream_t s) : st(s), pool(pool_of_current_device()) {}
    ~AsyncTmp() { for (void *p : ptrs) cudaFreeAsync(p, st); }
    int alloc(size_t bytes, void **d)
    {
        if (pool) CUDA_TRY(cudaMallocFromPoolAsync(d, bytes ? bytes : 16, pool, st));
        else CUDA_TRY(cudaMallocAsync(d, bytes ? bytes : 16, st));
        ptrs.push_back(*d);
        return KG_OK;
    }
    // device view of an input: the pointer itself, or a stream-ordered copy of host memory
    int get(const void *src, size_t bytes, const void **dev)
    {
        if (!src) { *dev = nullptr; return KG_OK; }
        if (is_device_ptr(src)) { *dev = src; return KG_OK; }
        void *d = nullptr;
        int rc = alloc(bytes, &d);
        if (rc) return rc;
        CUDA_TRY(cudaMemcpyAsync(d, src, bytes, cudaMemcpyHostToDevice, st));
        *dev = d;
        return KG_OK;
    }
};

extern "C" int kg_create_hamiltonian(kg_hamiltonian **out, int64_t n, int32_t kmax, const int32_t *nn,
                                     const int32_t *nl, const double *hop_eV, const double *onsite_eV,
                                     const double *x_nm, double period_x_nm, double e0_eV,
                                     double scale_eV, void *stream)
{
    return guarded([&]() -> int {
    int rc = check_create_args(out, n, kmax, nn, nl, hop_eV, x_nm, period_x_nm, e0_eV, scale_eV);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    TmpDev tmp;
    const void *d_nn, *d_nl, *d_hop, *d_ons, *d_x;
    if ((rc = tmp.get(nn, (size_t)n * 4, st, &d_nn)) || (rc = tmp.get(nl, (size_t)n * kmax * 4, st, &d_nl)) ||
        (rc = tmp.get(hop_eV, (size_t)n * kmax * 8, st, &d_hop)) || (rc = tmp.get(onsite_eV, (size_t)n * 8, st, &d_ons)) ||
        (rc = tmp.get(x_nm, (size_t)n * 8, st, &d_x)))
        return rc;
    return create_from_device_list(out, n, kmax, (const int32_t *)d_nn, (const int32_t *)d_nl,
                                   (const double *)d_hop, (const double *)d_ons, (const double *)d_x,
                                   period_x_nm, e0_eV, scale_eV, st);
    });
}

extern "C" int kg_create_hamiltonian_csr(kg_hamiltonian **out, int64_t n, const int64_t *rowptr,
                                         const int32_t *col, const double *hop_eV,
                                         const double *onsite_eV, const double *x_nm,
                                         double period_x_nm, double e0_eV, double scale_eV, void *stream)
{
    return guarded([&]() -> int {
    int rc = check_create_args(out, n, 1, rowptr, col, hop_eV, x_nm, period_x_nm, e0_eV, scale_eV);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    TmpDev tmp;
    const void *d_rp, *d_col, *d_val, *d_ons, *d_x;
    if ((rc = tmp.get(rowptr, (size_t)(n + 1) * 8, st, &d_rp))) return rc;
    int64_t nnz = 0;
    CUDA_TRY(cudaMemcpyAsync(&nnz, (const int64_t *)d_rp + n, 8, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (nnz < 0 || nnz > n * 32) return fail(KG_EINVAL, "rowptr[n] = %lld is not a valid nnz", (long long)nnz);
    const size_t nz = (size_t)(nnz > 0 ? nnz : 1);
    if ((rc = tmp.get(col, nz * 4, st, &d_col)) || (rc = tmp.get(hop_eV, nz * 8, st, &d_val)) ||
        (rc = tmp.get(onsite_eV, (size_t)n * 8, st, &d_ons)) || (rc = tmp.get(x_nm, (size_t)n * 8, st, &d_x)))
        return rc;
    int *d_max = nullptr;
    CUDA_TRY(cudaMalloc(&d_max, 8));
    tmp.ptrs.push_back(d_max);
    CUDA_TRY(cudaMemsetAsync(d_max, 0, 8, st));
    const int grid = (int)std::min<int64_t>((n + 255) / 256, 1184);
    kg_csr_max_row<<<grid, 256, 0, st>>>(n, (const int64_t *)d_rp, d_max, (unsigned int *)(d_max + 1));
    int hostv[2];
    CUDA_TRY(cudaMemcpyAsync(hostv, d_max, 8, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (hostv[1]) return fail(KG_EINVAL, "CSR row length outside [0, 32]");
    const int kmax = hostv[0] > 0 ? hostv[0] : 1;
    int32_t *d_nn = nullptr, *d_nl = nullptr;
    double *d_hop = nullptr;
    CUDA_TRY(cudaMalloc(&d_nn, (size_t)n * 4)); tmp.ptrs.push_back(d_nn);
    CUDA_TRY(cudaMalloc(&d_nl, (size_t)n * kmax * 4)); tmp.ptrs.push_back(d_nl);
    CUDA_TRY(cudaMalloc(&d_hop, (size_t)n * kmax * 8)); tmp.ptrs.push_back(d_hop);
    kg_csr_to_ell<<<grid, 256, 0, st>>>(n, (const int64_t *)d_rp, (const int32_t *)d_col,
                                        (const double *)d_val, kmax, d_nn, d_nl, d_hop);
    CUDA_TRY(cudaGetLastError());
    return create_from_device_list(out, n, kmax, d_nn, d_nl, d_hop, (const double *)d_ons,
                                   (const double *)d_x, period_x_nm, e0_eV, scale_eV, st);
    });
}

extern "C" int kg_destroy_hamiltonian(kg_hamiltonian *h)
{
    if (!h) return KG_OK;
    for (auto &g : h->graphs) cudaGraphExecDestroy(g.exec);
    cudaFree(h->nl); cudaFree(h->nlp); cudaFree(h->hop); cudaFree(h->xhop); cudaFree(h->onsite);
    cudaFree(h->perm); cudaFree(h->iperm); cudaFree(h->d_flag);
    for (auto &tp : h->tbp) { cudaFree(tp.tinfo); cudaFree(tp.rows); cudaFree(tp.hid); cudaFree(tp.hons); }
    for (int i = 0; i < WS_COUNT; ++i) cudaFree(h->ws[i]);
    delete h;
    return KG_OK;
}

extern "C" size_t kg_workspace_bytes(const kg_hamiltonian *h)
{
    if (!h) return 0;
    size_t t = h->matrix_bytes + h->tbp[0].bytes + h->tbp[1].bytes;
    for (int i = 0; i < WS_COUNT; ++i) t += h->ws_bytes[i];
    return t;
}

extern "C" int64_t kg_num_sites(const kg_hamiltonian *h) { return h ? h->n : 0; }
extern "C" int64_t kg_launch_count(const kg_hamiltonian *h) { return h ? h->launches : 0; }

extern "C" int kg_set_option(kg_hamiltonian *h, int option, int64_t value)
{
    return guarded([&]() -> int {
    if (!h) return fail(KG_EINVAL, "NULL handle");
    switch (option) {
    case KG_OPT_USE_GRAPHS: h->use_graphs = (int)value; break;
    case KG_OPT_BLOCKS_PER_SM:
        if (value < 1 || value > 32) return fail(KG_EINVAL, "blocks per SM must be in [1, 32]");
        h->blocks_per_sm = (int)value; break;
    case KG_OPT_THREADS:
        if (value != 64 && value != 128 && value != 256) return fail(KG_EINVAL, "threads must be 64, 128 or 256");
        h->threads = (int)value; break;
    case KG_OPT_STAGED: h->staged = value != 0; break;
    case KG_OPT_STAGES:
        if (value < 0 || value > SG_MAX_STAGES) return fail(KG_EINVAL, "stages must be in [0, %d]", SG_MAX_STAGES);
        h->stages = (int)value; break;
    case KG_OPT_STAGED_CTAS:
        if (value < 0 || value > 8) return fail(KG_EINVAL, "staged CTAs per SM must be in [0, 8]");
        h->staged_ctas = (int)value; break;
    case KG_OPT_ALTERNATE: h->alternate = value != 0; break;
    case KG_OPT_DOUBLING: h->doubling = value != 0; break;
    case KG_OPT_CLENSHAW: h->clenshaw = value != 0; break;
    case KG_OPT_PDL: h->pdl = value < 0 ? -1 : (value != 0); break;
    case KG_OPT_TWO_STEP: h->tb2 = value < 0 ? -1 : (value != 0); break;
    case KG_OPT_CHECK_INPUT: h->check_input = value != 0; break;
    case KG_OPT_ONE_LAUNCH: h->one_launch = value < 0 ? -1 : (value != 0); break;
    case KG_OPT_DICT:
        if (value != 0) return fail(KG_EINVAL, "the dictionary can only be switched off");
        h->ndict = 0; break;
    default: return fail(KG_EINVAL, "unknown option %d", option);
    }
    for (auto &g : h->graphs) cudaGraphExecDestroy(g.exec);
    h->graphs.clear();
    return KG_OK;
    });
}

// --------------------------------------------------------------------------------------
// device-level drivers (all pointers are device pointers here)
// --------------------------------------------------------------------------------------

// enqueue the M-1 fused recursion+dot kernels of Alg. 5 (a2+a3); partials [M][grid][R]
// mode MODE_MOM: literal Alg. 5, R columns.  MODE_MOM2 (phi_L = phi_R) and MODE_MOMX (phiR is the
// batch [phi_L | phi_R], R = total columns, partial rows R/2 wide): step m produces T_m and the
// partials of moments 2m-1 and 2m, so the loop stops at m = M/2
// (2 T_a T_b = T_{a+b} + T_{|a-b|}; kg_reduce_partials finishes it).
static int enqueue_moment_steps(kg_hamiltonian *h, const c128 *phiL, int ldL, const c128 *phiR, int ldR,
                                int R, int M, c128 *ta, c128 *tb, c128 *part, int grid,
                                const StagedPlan &sp, int mode, cudaStream_t st)
{
    const bool dbl = mode != MODE_MOM;
    const int m_end = dbl ? M / 2 + 1 : M;
    const size_t prow = (size_t)grid * (mode == MODE_MOMX ? R / 2 : R);
    StagedArgs sa = staged_base_args(h, sp);
    sa.aux = phiL;
    StepArgs a = base_args(h);
    a.phiL = phiL; a.ld_L = ldL;
    // m = 1: T_1 = H~ T_0, partial rows 0 and 1
    a.alpha = 1.0;
    a.cur = phiR; a.ld_cur = ldR; a.next = ta;
    a.partial0 = part; a.partial = part + prow; a.partial2 = part + 2 * prow;
    CUDA_TRY(launch_step(h, mode, true, R, a, grid, st));
    a.alpha = 2.0; a.partial0 = nullptr;
    for (int m = 2; m < m_end; ++m) {
        a.partial = part + (size_t)(dbl ? 2 * m - 1 : m) * prow;
        a.partial2 = part + (size_t)(2 * m) * prow;
        if (m == 2) { a.cur = ta; a.ld_cur = R; a.prev = phiR; a.ld_prev = ldR; a.next = tb; }
        else if (m & 1) { a.cur = tb; a.ld_cur = R; a.prev = ta; a.ld_prev = R; a.next = ta; }
        else { a.cur = ta; a.ld_cur = R; a.prev = tb; a.ld_prev = R; a.next = tb; }
        if (sp.ok && ldL == R && a.ld_cur == R && a.ld_prev == R) {
            // tuned form of the same step: TMA-staged streams, alternating sweep direction
            sa.cur = a.cur; sa.prev = a.prev; sa.next = a.next; sa.partial = a.partial; sa.partial2 = a.partial2;
            sa.reverse = h->alternate ? (m & 1) : 0;
            CUDA_TRY(staged_launch(h, mode, R, sa, sp, st));
        } else {
            CUDA_TRY(launch_step(h, mode, false, R, a, grid, st));
        }
    }
    return KG_OK;
}

static bool want_graph(const kg_hamiltonian *h, int64_t elems, cudaStream_t st)
{
    // the legacy default stream cannot be captured
    if (st == nullptr || st == cudaStreamLegacy || h->use_graphs == 0) return false;
    if (h->use_graphs > 0) return true;
    return elems <= (int64_t)1 << 21;      // auto: launch-bound sizes only
}

static int copy_cols(kg_hamiltonian *h, const c128 *src, int ld_src, c128 *dst, int ld_dst, int ncols, cudaStream_t st);

// mu[r*mu_rstride + m] = <phiL_r | T_m(H~) | phiR_r>, m < M
// cross = true: phiL == phiR is the batch [phi_L | phi_R] with R columns in total (MODE_MOMX);
// mu gets R/2 rows.
static int moments_device(kg_hamiltonian *h, const c128 *phiL, int ldL, const c128 *phiR, int ldR, int R,
                          int M, c128 *mu, int64_t mu_rstride, cudaStream_t st, bool cross = false)
{
    const int64_t elems = h->n * R;
    const bool dbl = cross || (h->doubling && phiL == phiR && ldL == ldR);
    const int mode = cross ? MODE_MOMX : dbl ? MODE_MOM2 : MODE_MOM;
    const int PR = cross ? R / 2 : R;                        // columns of a partial row / rows of mu
    const StagedPlan sp = staged_plan(h, mode, R);
    int rc;
    // two Chebyshev steps per pass (kg_tb2.cuh) when the vectors are contiguous [n][R].  The kernel keeps a
    // matrix row and its columns in per-thread registers, which stops at two columns: a wider batch is split
    // into column-pair PLANES [n][2] — (2p, 2p+1) for phi_L = phi_R, (phi_L,r, phi_R,r) for the cross form — that
    // ONE launch per pass serves side by side, each plane on its share of the CTAs.
    Tb2Launch tl;
    tl.ok = false;
    const int CP = R <= 2 ? R : 2;                                  // columns per plane
    const int nplanes = R / CP;
    if (dbl && ldL == R && ldR == R && M / 2 >= 3 && (R <= 2 || R % 2 == 0) &&
        (rc = tb2_plan(h, mode, CP, nplanes, st, &tl)))
        return rc;
    const int grid = tl.ok ? tl.grid : sp.ok ? sp.grid : grid_for(h, elems);   // one partial row shape for all kernels of the call
    void *ta, *tb, *part;
    if ((rc = ws_get(h, WS_TA, (size_t)elems * 16, &ta)) || (rc = ws_get(h, WS_TB, (size_t)elems * 16, &tb)) ||
        (rc = ws_get(h, WS_PART, (size_t)(M + 1) * grid * R * 16, &part)))
        return rc;
    if (tl.ok) {
        void *tc, *td;
        if ((rc = ws_get(h, WS_TC, (size_t)elems * 16, &tc)) || (rc = ws_get(h, WS_TD, (size_t)elems * 16, &td))) return rc;
        const size_t prow = (size_t)grid * PR;                      // partial rows [grid = CTAs per plane][PR], plane-major columns
        c128 *P = (c128 *)part;
        // m = 1: T_1 = H~ T_0 and the partials of moments 0, 1, 2 (one-thread-per-element kernel, whole batch)
        StepArgs a = base_args(h);
        a.phiL = phiL; a.ld_L = ldL; a.alpha = 1.0;
        a.cur = phiR; a.ld_cur = ldR; a.next = (c128 *)ta;
        a.partial0 = P; a.partial = P + prow; a.partial2 = P + 2 * prow;
        CUDA_TRY(launch_step(h, mode, true, R, a, grid, st));
        // steps m = 2 .. M/2 in pairs; step m makes T_m and the partials of moments 2m - 1 and 2m
        Tb2Args ta2 = tb2_base_args(h, CP);
        ta2.nstages = tl.nst;
        ta2.nplanes = nplanes; ta2.plane_stride = nplanes > 1 ? h->n * CP : 0;
        const c128 *prev = phiR, *cur = (const c128 *)ta;
        std::vector<c128 *> freeb = {(c128 *)tb, (c128 *)tc, (c128 *)td};
        if (nplanes > 1) {
            // T_0 and T_1 from [n][R] into planes [nplanes][n][2]
            void *p0;
            if ((rc = ws_get(h, WS_PLANE, (size_t)elems * 16, &p0))) return rc;
            c128 *P0 = (c128 *)p0, *P1 = (c128 *)tb;
            const int Rh = R / 2;
            for (int p = 0; p < nplanes; ++p) {
                c128 *d0 = P0 + (size_t)p * h->n * 2, *d1 = P1 + (size_t)p * h->n * 2;
                if (cross) {
                    if ((rc = copy_cols(h, phiR + p, R, d0, 2, 1, st)) || (rc = copy_cols(h, phiR + Rh + p, R, d0 + 1, 2, 1, st)) ||
                        (rc = copy_cols(h, (const c128 *)ta + p, R, d1, 2, 1, st)) ||
                        (rc = copy_cols(h, (const c128 *)ta + Rh + p, R, d1 + 1, 2, 1, st)))
                        return rc;
                } else if ((rc = copy_cols(h, phiR + 2 * p, R, d0, 2, 2, st)) || (rc = copy_cols(h, (const c128 *)ta + 2 * p, R, d1, 2, 2, st))) {
                    return rc;
                }
            }
            prev = P0; cur = P1;
            freeb = {(c128 *)ta, (c128 *)tc, (c128 *)td};
        }
        const c128 *keep_in = nplanes > 1 ? nullptr : phiR;          // the caller's phi_R is never written
        const int m_end = M / 2 + 1;
        int pass = 0;
        for (int m = 2; m < m_end; ++pass) {
            const int nstep = (m + 1 < m_end) ? 2 : 1;
            ta2.cur = cur; ta2.prev = prev;
            ta2.next1 = freeb[0]; ta2.next2 = nstep == 2 ? freeb[1] : nullptr;
            ta2.p1 = P + (size_t)(2 * m - 1) * prow; ta2.p2 = P + (size_t)(2 * m) * prow;
            ta2.p3 = P + (size_t)(2 * m + 1) * prow; ta2.p4 = P + (size_t)(2 * m + 2) * prow;
            ta2.reverse = h->alternate ? (pass & 1) : 0;
            h->launches++;
            CUDA_TRY(kg_tb2_launch(h->kmax, mode, CP, h->has_onsite, nstep, ta2, grid * nplanes, tl.smem, h->device, st));
            // rotate: the two oldest vectors become free
            c128 *old_prev = const_cast<c128 *>(prev), *old_cur = const_cast<c128 *>(cur);
            if (nstep == 2) {
                prev = freeb[0]; cur = freeb[1];
                freeb.erase(freeb.begin(), freeb.begin() + 2);
                if (old_prev != keep_in) freeb.push_back(old_prev);
                freeb.push_back(old_cur);
            } else {
                prev = cur; cur = freeb[0];
                freeb.erase(freeb.begin());
                if (old_prev != keep_in) freeb.push_back(old_prev);
            }
            m += nstep;
        }
    } else if (h->one_launch != 0 && sp.ok && sp.grid == sp.ntiles && ldL == R && ldR == R && R <= 8 && h->kmax <= 12 &&
               (sp.ntiles + SM_MAX_CLUSTER - 1) / SM_MAX_CLUSTER <= 255 &&
               (sp.ntiles + SM_MAX_CLUSTER - 1) / SM_MAX_CLUSTER * sm_tile_bytes(R, h->kmax, mode == MODE_MOM) <= (size_t)200 * 1024) {
        // launch-bound sizes: first step, then ALL further steps in one cluster kernel whose CTAs keep their
        // tiles in (distributed) shared memory (kg_small.cuh); bitwise equal to the one-launch-per-step path
        const size_t prow = (size_t)grid * PR;
        c128 *P = (c128 *)part;
        StepArgs a = base_args(h);
        a.phiL = phiL; a.ld_L = ldL; a.alpha = 1.0;
        a.cur = phiR; a.ld_cur = ldR; a.next = (c128 *)ta;
        a.partial0 = P; a.partial = P + prow; a.partial2 = P + 2 * prow;
        CUDA_TRY(launch_step(h, mode, true, R, a, grid, st));
        const int m_end = dbl ? M / 2 + 1 : M;
        if (m_end > 2) {
            SmallArgs sa;
            memset(&sa, 0, sizeof(sa));
            sa.nl = h->nl; sa.hop = h->hop; sa.onsite = h->onsite; sa.n = h->n; sa.ns = h->ns; sa.K = h->kmax;
            sa.ons = h->has_onsite ? 1 : 0;
            sa.t0 = phiR; sa.t1 = (const c128 *)ta; sa.phiL = phiL; sa.part = P; sa.m_end = m_end;
            sa.ntiles = sp.ntiles;
            sa.alternate = h->alternate;
            h->launches++;
            // 9-16 tiles: one tile per CTA in a 16-CTA cluster (non-portable size) when the device takes it,
            // else two tiles per CTA in the portable 8-CTA cluster — same arithmetic, same partial slots
            cudaError_t e = cudaErrorInvalidValue;
            if (sp.ntiles > SM_MAX_CLUSTER && sp.ntiles <= SM_BIG_CLUSTER && h->big_cluster != 0) {
                sa.vt = 1;
                e = kg_small_launch(mode, R, sa, sp.ntiles, sm_tile_bytes(R, h->kmax, mode == MODE_MOM), h->device, st);
                if (e != cudaSuccess) { (void)cudaGetLastError(); h->big_cluster = 0; }
            }
            if (e != cudaSuccess) {
                sa.vt = (sp.ntiles + SM_MAX_CLUSTER - 1) / SM_MAX_CLUSTER;
                const int ncta = (sp.ntiles + sa.vt - 1) / sa.vt;
                CUDA_TRY(kg_small_launch(mode, R, sa, ncta, (size_t)sa.vt * sm_tile_bytes(R, h->kmax, mode == MODE_MOM), h->device, st));
            }
        }
    } else if (want_graph(h, elems, st)) {
        cudaGraphExec_t exec = nullptr;
        for (auto &g : h->graphs)
            if (g.phiL == phiL && g.phiR == phiR && g.ldL == ldL && g.ldR == ldR && g.R == R && g.M == M &&
                g.grid == grid && g.threads == h->threads && g.dbl == mode)
                exec = g.exec;
        if (!exec) {
            cudaGraph_t graph;
            CUDA_TRY(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
            const int64_t before = h->launches;
            rc = enqueue_moment_steps(h, phiL, ldL, phiR, ldR, R, M, (c128 *)ta, (c128 *)tb, (c128 *)part, grid, sp, mode, st);
            h->launches = before;
            cudaError_t e = cudaStreamEndCapture(st, &graph);
            if (rc) { if (e == cudaSuccess) cudaGraphDestroy(graph); return rc; }
            if (e != cudaSuccess) return fail(KG_ECUDA, "graph capture: %s", cudaGetErrorString(e));
            e = cudaGraphInstantiate(&exec, graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) return fail(KG_ECUDA, "graph instantiate: %s", cudaGetErrorString(e));
            if (h->graphs.size() >= 8) { cudaGraphExecDestroy(h->graphs.front().exec); h->graphs.erase(h->graphs.begin()); }
            h->graphs.push_back(GraphEntry{phiL, phiR, ldL, ldR, R, M, grid, h->threads, mode, exec});
        }
        CUDA_TRY(cudaGraphLaunch(exec, st));
        h->launches += dbl ? M / 2 : M - 1;
    } else {
        if ((rc = enqueue_moment_steps(h, phiL, ldL, phiR, ldR, R, M, (c128 *)ta, (c128 *)tb, (c128 *)part, grid, sp, mode, st)))
            return rc;
    }
    const int warps = M * PR;
    kg_reduce_partials<<<(warps * 32 + 255) / 256, 256, 0, st>>>((const c128 *)part, M, grid, PR, mu, mu_rstride, dbl ? 1 : 0);
    h->launches++;
    CUDA_TRY(cudaGetLastError());
    return KG_OK;
}

// out = U(dt) in  (Alg. 6): in [n] with row stride ld_in, out [n][R]
static int evolve_device(kg_hamiltonian *h, const c128 *in, int ld_in, c128 *out, int R, double dt_fs,
                         double eps, cudaStream_t st)
{
    const int64_t elems = h->n * R;
    const int grid = grid_for(h, elems);
    const StagedPlan sp = staged_plan(h, MODE_EVO, R);
    StagedArgs sa = staged_base_args(h, sp);
    sa.aux = out; sa.out = out;
    void *ta, *tb;
    int rc;
    if ((rc = ws_get(h, WS_TA, (size_t)elems * 16, &ta)) || (rc = ws_get(h, WS_TB, (size_t)elems * 16, &tb))) return rc;
    std::vector<c128> c;
    series_coefficients(h, dt_fs, eps, c);
    const int np = (int)c.size();
    const StagedPlan cp = staged_plan(h, MODE_CLEN, R);
    if (h->clenshaw && cp.ok && ld_in == R && np >= 4) {
        // Clenshaw's backward recurrence for sum_m c_m T_m(H~) phi (same series as Alg. 6, eq 36):
        //   b_m = c_m phi + 2 H~ b_{m+1} - b_{m+2}  (b_np = b_{np+1} = 0),  U phi = c_0 phi + H~ b_1 - b_2.
        // np - 1 staged sweeps, no accumulator stream.  The first two sweeps fold b_{np-1} = c_{np-1} phi
        // into their coefficients so that it is never written.
        StagedArgs ca = staged_base_args(h, cp);
        ca.aux = in;
        c128 *buf[2] = {(c128 *)ta, (c128 *)tb};
        const c128 one = make_double2(1.0, 0.0);
        for (int m = np - 2, k = 0; m >= 0; --m, ++k) {
            ca.alpha = m == 0 ? 1.0 : 2.0;
            ca.next = m == 0 ? out : buf[k & 1];
            if (k == 0) {            // b_{np-2} = c_{np-2} phi + 2 c_{np-1} H~ phi
                ca.cur = in; ca.prev = in; ca.c1 = c[m]; ca.cpre = c[np - 1]; ca.use_prev = 0;
            } else if (k == 1) {     // b_{np-3} = (c_{np-3} - c_{np-1}) phi + 2 H~ b_{np-2}
                ca.cur = buf[0]; ca.prev = buf[0]; ca.cpre = one; ca.use_prev = 0;
                ca.c1 = make_double2(c[m].x - c[np - 1].x, c[m].y - c[np - 1].y);
            } else {
                ca.cur = buf[(k - 1) & 1]; ca.prev = buf[k & 1]; ca.c1 = c[m]; ca.cpre = one; ca.use_prev = 1;
            }
            ca.reverse = h->alternate ? (k & 1) : 0;
            CUDA_TRY(staged_launch(h, MODE_CLEN, R, ca, cp, st));
        }
        return KG_OK;
    }
    StepArgs a = base_args(h);
    a.out = out;
    a.alpha = 1.0;
    a.cur = in; a.ld_cur = ld_in; a.next = (c128 *)ta;
    a.c0 = c[0]; a.c1 = np > 1 ? c[1] : make_double2(0.0, 0.0);
    CUDA_TRY(launch_step(h, MODE_EVO, true, R, a, grid, st));
    a.alpha = 2.0;
    for (int m = 2; m < np; ++m) {
        a.c1 = c[m];
        if (m == 2) { a.cur = (c128 *)ta; a.ld_cur = R; a.prev = in; a.ld_prev = ld_in; a.next = (c128 *)tb; }
        else if (m & 1) { a.cur = (c128 *)tb; a.prev = (c128 *)ta; a.ld_prev = R; a.next = (c128 *)ta; }
        else { a.cur = (c128 *)ta; a.prev = (c128 *)tb; a.ld_prev = R; a.next = (c128 *)tb; }
        if (sp.ok && a.ld_cur == R && a.ld_prev == R) {
            sa.cur = a.cur; sa.prev = a.prev; sa.next = a.next; sa.c1 = a.c1;
            sa.reverse = h->alternate ? (m & 1) : 0;
            CUDA_TRY(staged_launch(h, MODE_EVO, R, sa, sp, st));
        } else {
            CUDA_TRY(launch_step(h, MODE_EVO, false, R, a, grid, st));
        }
    }
    return KG_OK;
}

// (psi_out, psix_out) = (U psi, U psix + [X,U] psi)  (eq 44 via the (a,d) pair recursion)
static int pair_device(kg_hamiltonian *h, const c128 *psi, const c128 *psix, c128 *psi_out, c128 *psix_out,
                       int R, double dt_fs, double eps, cudaStream_t st)
{
    const int64_t elems = h->n * R;
    const int grid = grid_for(h, elems);
    void *ta, *tb, *da, *db;
    int rc;
    if ((rc = ws_get(h, WS_TA, (size_t)elems * 16, &ta)) || (rc = ws_get(h, WS_TB, (size_t)elems * 16, &tb)) ||
        (rc = ws_get(h, WS_DA, (size_t)elems * 16, &da)) || (rc = ws_get(h, WS_DB, (size_t)elems * 16, &db)))
        return rc;
    std::vector<c128> c;
    series_coefficients(h, dt_fs, eps, c);
    const int np = (int)c.size();
    const StagedPlan cp = staged_plan(h, MODE_PCLEN, R);
    if (h->clenshaw && cp.ok && np >= 4) {
        // Clenshaw form of the pair recursion (see evolve_device): b and e chains, np - 1 sweeps,
        // no accumulator streams; psi_out / psix_out are written by the last sweep.
        StagedArgs ca = staged_base_args(h, cp);
        ca.aux = psi; ca.daux = psix;
        c128 *bb[2] = {(c128 *)ta, (c128 *)tb}, *ee[2] = {(c128 *)da, (c128 *)db};
        const c128 one = make_double2(1.0, 0.0);
        for (int m = np - 2, k = 0; m >= 0; --m, ++k) {
            ca.alpha = m == 0 ? 1.0 : 2.0;
            ca.next = m == 0 ? psi_out : bb[k & 1];
            ca.dnext = m == 0 ? psix_out : ee[k & 1];
            if (k == 0) {
                ca.cur = psi; ca.prev = psi; ca.dcur = psix; ca.dprev = psix;
                ca.c1 = c[m]; ca.cpre = c[np - 1]; ca.use_prev = 0;
            } else if (k == 1) {
                ca.cur = bb[0]; ca.prev = bb[0]; ca.dcur = ee[0]; ca.dprev = ee[0]; ca.cpre = one; ca.use_prev = 0;
                ca.c1 = make_double2(c[m].x - c[np - 1].x, c[m].y - c[np - 1].y);
            } else {
                ca.cur = bb[(k - 1) & 1]; ca.prev = bb[k & 1]; ca.dcur = ee[(k - 1) & 1]; ca.dprev = ee[k & 1];
                ca.c1 = c[m]; ca.cpre = one; ca.use_prev = 1;
            }
            ca.reverse = h->alternate ? (k & 1) : 0;
            CUDA_TRY(staged_launch(h, MODE_PCLEN, R, ca, cp, st));
        }
        return KG_OK;
    }
    const StagedPlan sp = staged_plan(h, MODE_PAIR, R);
    StagedArgs sa = staged_base_args(h, sp);
    sa.aux = psi_out; sa.out = psi_out; sa.daux = psix_out; sa.outd = psix_out;
    StepArgs a = base_args(h);
    a.out = psi_out; a.outd = psix_out;
    a.alpha = 1.0;
    a.cur = psi; a.ld_cur = R; a.next = (c128 *)ta;
    a.dcur = psix; a.ld_dcur = R; a.dnext = (c128 *)da;
    a.c0 = c[0]; a.c1 = np > 1 ? c[1] : make_double2(0.0, 0.0);
    CUDA_TRY(launch_step(h, MODE_PAIR, true, R, a, grid, st));
    a.alpha = 2.0;
    a.ld_prev = R; a.ld_dprev = R;
    for (int m = 2; m < np; ++m) {
        a.c1 = c[m];
        if (m == 2) {
            a.cur = (c128 *)ta; a.prev = psi; a.next = (c128 *)tb;
            a.dcur = (c128 *)da; a.dprev = psix; a.dnext = (c128 *)db;
        } else if (m & 1) {
            a.cur = (c128 *)tb; a.prev = (c128 *)ta; a.next = (c128 *)ta;
            a.dcur = (c128 *)db; a.dprev = (c128 *)da; a.dnext = (c128 *)da;
        } else {
            a.cur = (c128 *)ta; a.prev = (c128 *)tb; a.next = (c128 *)tb;
            a.dcur = (c128 *)da; a.dprev = (c128 *)db; a.dnext = (c128 *)db;
        }
        if (sp.ok) {
            sa.cur = a.cur; sa.prev = a.prev; sa.next = a.next; sa.c1 = a.c1;
            sa.dcur = a.dcur; sa.dprev = a.dprev; sa.dnext = a.dnext;
            sa.reverse = h->alternate ? (m & 1) : 0;
            CUDA_TRY(staged_launch(h, MODE_PAIR, R, sa, sp, st));
        } else {
            CUDA_TRY(launch_step(h, MODE_PAIR, false, R, a, grid, st));
        }
    }
    return KG_OK;
}

static int velocity_device(kg_hamiltonian *h, const c128 *in, int ld_in, c128 *out, int ld_out, int R,
                           cudaStream_t st)
{
    StepArgs a = base_args(h);
    a.cur = in; a.ld_cur = ld_in; a.vout = out; a.ld_vout = ld_out;
    a.vscale = h->s / KG_HBAR;
    CUDA_TRY(launch_step(h, MODE_VEL, true, R, a, grid_for(h, h->n * R), st));
    return KG_OK;
}

static int copy_cols(kg_hamiltonian *h, const c128 *src, int ld_src, c128 *dst, int ld_dst, int ncols,
                     cudaStream_t st)
{
    kg_copy_cols<<<grid_for(h, h->n * ncols), h->threads, 0, st>>>(src, ld_src, dst, ld_dst, ncols, h->n);
    h->launches++;
    CUDA_TRY(cudaGetLastError());
    return KG_OK;
}

// output staging: device buffer to compute into, copied to the caller's host array afterwards
struct OutStage { void *user; void *dev; size_t bytes; bool host; };
static int stage_out(kg_hamiltonian *h, int slot, void *p, size_t bytes, OutStage *o)
{
    o->user = p; o->bytes = bytes; o->host = !is_device_ptr(p);
    if (!o->host) { o->dev = p; return KG_OK; }
    return ws_get(h, slot, bytes, &o->dev);
}
static int finish_out(const OutStage &o, cudaStream_t st)
{
    if (o.host) CUDA_TRY(cudaMemcpyAsync(o.user, o.dev, o.bytes, cudaMemcpyDeviceToHost, st));
    return KG_OK;
}

// --------------------------------------------------------------------------------------
// public calls
// --------------------------------------------------------------------------------------
extern "C" int kg_moments(kg_hamiltonian *h, const kg_c128 *phiL, const kg_c128 *phiR, int R, int M,
                          kg_c128 *mu, void *stream)
{
    return guarded([&]() -> int {
    if (!h || !phiL || !phiR || !mu) return fail(KG_EINVAL, "kg_moments: NULL argument");
    if (!r_ok(R, true)) return fail(KG_EUNSUPPORTED, "R must be 1, 2, 4, 8 or 16");
    if (M < 2) return fail(KG_EINVAL, "M must be >= 2");
    cudaStream_t st = (cudaStream_t)stream;
    const void *dL, *dR;
    int rc;
    if ((rc = vec_in(h, WS_IN0, phiL, R, st, &dL))) return rc;
    if (phiR == phiL) dR = dL;
    else if ((rc = vec_in(h, WS_IN1, phiR, R, st, &dR))) return rc;
    OutStage o;
    if ((rc = stage_out(h, WS_MU, mu, (size_t)R * M * 16, &o))) return rc;
    if ((rc = moments_device(h, (const c128 *)dL, R, (const c128 *)dR, R, R, M, (c128 *)o.dev, M, st))) return rc;
    return finish_out(o, st);
    });
}

extern "C" int kg_dos_moments(kg_hamiltonian *h, const kg_c128 *phi, int R, int M, kg_c128 *mu, void *stream)
{
    return guarded([&]() -> int {
    return kg_moments(h, phi, phi, R, M, mu, stream);
    });
}

extern "C" int kg_evolve(kg_hamiltonian *h, const kg_c128 *in, kg_c128 *out, int R, double dt_fs,
                         double bessel_eps, void *stream)
{
    return guarded([&]() -> int {
    if (!h || !in || !out) return fail(KG_EINVAL, "kg_evolve: NULL argument");
    if (in == out) return fail(KG_EINVAL, "kg_evolve: out must not alias in");
    if (!r_ok(R, true)) return fail(KG_EUNSUPPORTED, "R must be 1, 2, 4, 8 or 16");
    if (dt_fs == 0.0 || !std::isfinite(dt_fs)) return fail(KG_EINVAL, "dt_fs must be finite and non-zero");
    cudaStream_t st = (cudaStream_t)stream;
    const void *din;
    VecOut o;
    int rc;
    if ((rc = vec_in(h, WS_IN0, in, R, st, &din)) || (rc = vec_out(h, WS_OUT0, out, R, &o))) return rc;
    if ((rc = evolve_device(h, (const c128 *)din, R, (c128 *)o.dev, R, dt_fs, bessel_eps, st))) return rc;
    return vec_out_finish(h, o, st);
    });
}

extern "C" int kg_apply_velocity(kg_hamiltonian *h, const kg_c128 *in, kg_c128 *out, int R, void *stream)
{
    return guarded([&]() -> int {
    if (!h || !in || !out) return fail(KG_EINVAL, "kg_apply_velocity: NULL argument");
    if (in == out) return fail(KG_EINVAL, "kg_apply_velocity: out must not alias in");
    if (!r_ok(R, true)) return fail(KG_EUNSUPPORTED, "R must be 1, 2, 4, 8 or 16");
    cudaStream_t st = (cudaStream_t)stream;
    const void *din;
    VecOut o;
    int rc;
    if ((rc = vec_in(h, WS_IN0, in, R, st, &din)) || (rc = vec_out(h, WS_OUT0, out, R, &o))) return rc;
    if ((rc = velocity_device(h, (const c128 *)din, R, (c128 *)o.dev, R, R, st))) return rc;
    return vec_out_finish(h, o, st);
    });
}

extern "C" int kg_evolve_x(kg_hamiltonian *h, kg_c128 *psi, kg_c128 *psix, int R, double dt_fs,
                           double bessel_eps, void *stream)
{
    return guarded([&]() -> int {
    if (!h || !psi || !psix) return fail(KG_EINVAL, "kg_evolve_x: NULL argument");
    if (psi == psix) return fail(KG_EINVAL, "kg_evolve_x: psi and psix must be distinct");
    if (!r_ok(R, true)) return fail(KG_EUNSUPPORTED, "R must be 1, 2, 4, 8 or 16");
    if (!(dt_fs > 0.0) || !std::isfinite(dt_fs)) return fail(KG_EINVAL, "dt_fs must be finite and positive");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t vbytes = (size_t)h->n * R * 16;
    const void *dpsi, *dpsix;
    void *o0, *o1;
    int rc;
    if ((rc = vec_in(h, WS_IN0, psi, R, st, &dpsi)) || (rc = vec_in(h, WS_IN1, psix, R, st, &dpsix)) ||
        (rc = ws_get(h, WS_OUT0, vbytes, &o0)) || (rc = ws_get(h, WS_OUT1, vbytes, &o1)))
        return rc;
    if ((rc = pair_device(h, (const c128 *)dpsi, (const c128 *)dpsix, (c128 *)o0, (c128 *)o1, R, dt_fs, bessel_eps, st)))
        return rc;
    // back into the caller's arrays (in place for the caller): inverse permutation and / or copy
    void *user[2] = {psi, psix}, *res[2] = {o0, o1};
    for (int q = 0; q < 2; ++q) {
        const bool on_dev = is_device_ptr(user[q]);
        const void *src = res[q];
        if (h->perm) {
            void *dst = user[q];
            if (!on_dev && (rc = ws_get(h, WS_RAW0 + q, vbytes, &dst))) return rc;
            kg_permute_rows<<<grid_for(h, h->n * R), 256, 0, st>>>((const c128 *)res[q], (c128 *)dst, h->iperm, h->n, R);
            h->launches++;
            CUDA_TRY(cudaGetLastError());
            src = dst;
        }
        if (src != user[q]) CUDA_TRY(cudaMemcpyAsync(user[q], src, vbytes, cudaMemcpyDefault, st));
    }
    return KG_OK;
    });
}

static int check_corr_args(kg_hamiltonian *h, const void *phi, int R, int M, int n_steps, double dt_fs, void *mu, bool allow16)
{
    if (!h || !phi || !mu) return fail(KG_EINVAL, "NULL argument");
    if (!r_ok(R, allow16))
        return fail(KG_EUNSUPPORTED, allow16 ? "R must be 1, 2, 4, 8 or 16"
                                             : "R must be 1, 2, 4 or 8 (kg_vac advances a batch of 2R columns)");
    if (M < 2) return fail(KG_EINVAL, "M must be >= 2");
    if (n_steps < 0) return fail(KG_EINVAL, "n_steps must be >= 0");
    if (!(dt_fs > 0.0) || !std::isfinite(dt_fs)) return fail(KG_EINVAL, "dt_fs must be finite and positive");
    return KG_OK;
}

extern "C" int kg_vac(kg_hamiltonian *h, const kg_c128 *phi, int R, int M, int n_steps, double dt_fs,
                      double bessel_eps, kg_c128 *mu, void *stream)
{
    return guarded([&]() -> int {
    int rc = check_corr_args(h, phi, R, M, n_steps, dt_fs, mu, false);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t vbytes = (size_t)h->n * R * 16;
    const int R2 = 2 * R;
    const void *dphi;
    void *s0, *s1, *pl;
    OutStage o;
    if ((rc = vec_in(h, WS_IN0, phi, R, st, &dphi)) || (rc = ws_get(h, WS_S0, 2 * vbytes, &s0)) ||
        (rc = ws_get(h, WS_S1, 2 * vbytes, &s1)) || (rc = ws_get(h, WS_PHIL, 2 * vbytes, &pl)) ||
        (rc = stage_out(h, WS_MU, mu, (size_t)R * (n_steps + 1) * M * 16, &o)))
        return rc;
    // state S = [psi | chi] as one [n][2R] batch: psi_0 = phi, chi_0 = V phi  (Alg. 2)
    c128 *S = (c128 *)s0, *Sn = (c128 *)s1;
    if ((rc = copy_cols(h, (const c128 *)dphi, R, S, R2, R, st)) ||
        (rc = velocity_device(h, (const c128 *)dphi, R, S + R, R2, R, st)))
        return rc;
    const int64_t rstride = (int64_t)(n_steps + 1) * M;
    for (int k = 0; k <= n_steps; ++k) {
        // phi_L = V psi_k, phi_R = chi_k
        if (h->doubling && k == 0) {
            // t = 0: V psi_0 = V phi = chi_0, so phi_L = phi_R and the one-column doubling form applies
            // (half the work of the cross form; C_m^VAC(0) = <V phi|T_m|V phi>)
            c128 *X0 = (c128 *)pl;
            if ((rc = copy_cols(h, S + R, R2, X0, R, R, st)) ||
                (rc = moments_device(h, X0, R, X0, R, R, M, (c128 *)o.dev, rstride, st)))
                return rc;
        } else if (h->doubling) {
            // cross-doubling: [V psi_k | chi_k] advanced as one 2R-wide batch, two moments per sweep
            c128 *X0 = (c128 *)pl;
            if ((rc = velocity_device(h, S, R2, X0, R2, R, st)) || (rc = copy_cols(h, S + R, R2, X0 + R, R2, R, st)) ||
                (rc = moments_device(h, X0, R2, X0, R2, R2, M, (c128 *)o.dev + (size_t)k * M, rstride, st, true)))
                return rc;
        } else if ((rc = velocity_device(h, S, R2, (c128 *)pl, R, R, st)) ||
                   (rc = moments_device(h, (const c128 *)pl, R, S + R, R2, R, M, (c128 *)o.dev + (size_t)k * M, rstride, st)))
            return rc;
        if (k == n_steps) break;
        // [psi | chi] <- U(-dt) [psi | chi]   (eqs 42-43), one 2R-wide batch
        if ((rc = evolve_device(h, S, R2, Sn, R2, -dt_fs, bessel_eps, st))) return rc;
        c128 *t = S; S = Sn; Sn = t;
    }
    return finish_out(o, st);
    });
}

extern "C" int kg_msd(kg_hamiltonian *h, const kg_c128 *phi, int R, int M, int n_steps, double dt_fs,
                      double bessel_eps, kg_c128 *mu, void *stream)
{
    return guarded([&]() -> int {
    int rc = check_corr_args(h, phi, R, M, n_steps, dt_fs, mu, true);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t vbytes = (size_t)h->n * R * 16;
    const void *dphi;
    void *p0, *p1, *x0, *x1;
    OutStage o;
    if ((rc = vec_in(h, WS_IN0, phi, R, st, &dphi)) || (rc = ws_get(h, WS_S0, vbytes, &p0)) ||
        (rc = ws_get(h, WS_S1, vbytes, &p1)) || (rc = ws_get(h, WS_X0, vbytes, &x0)) ||
        (rc = ws_get(h, WS_X1, vbytes, &x1)) ||
        (rc = stage_out(h, WS_MU, mu, (size_t)R * (n_steps + 1) * M * 16, &o)))
        return rc;
    c128 *P = (c128 *)p0, *Pn = (c128 *)p1, *X = (c128 *)x0, *Xn = (c128 *)x1;
    CUDA_TRY(cudaMemcpyAsync(P, dphi, vbytes, cudaMemcpyDeviceToDevice, st));   // psi_0 = phi
    CUDA_TRY(cudaMemsetAsync(X, 0, vbytes, st));                                // psix_0 = 0
    const int64_t rstride = (int64_t)(n_steps + 1) * M;
    // row k = 0: psix_0 = 0, so C_m^MSD(0) = 0 exactly (eq 44 starts from zero) — written, not computed
    CUDA_TRY(cudaMemset2DAsync(o.dev, (size_t)rstride * 16, 0, (size_t)M * 16, (size_t)R, st));
    for (int k = 0; k <= n_steps; ++k) {
        if (k > 0 && (rc = moments_device(h, X, R, X, R, R, M, (c128 *)o.dev + (size_t)k * M, rstride, st))) return rc;
        if (k == n_steps) break;
        if ((rc = pair_device(h, P, X, Pn, Xn, R, dt_fs, bessel_eps, st))) return rc;
        c128 *t = P; P = Pn; Pn = t;
        t = X; X = Xn; Xn = t;
    }
    return finish_out(o, st);
    });
}

// --------------------------------------------------------------------------------------
// KPM reconstruction (SUPPORT row R1/R2 of SURVEY 2.2): handle-free, temporary device buffers
// --------------------------------------------------------------------------------------
extern "C" int kg_kpm_reconstruct(const kg_c128 *mu, int64_t rows, int M, int jackson, double e0_eV,
                                  double scale_eV, const double *energies_eV, int n_energies, double *f,
                                  void *stream)
{
    return guarded([&]() -> int {
    if (!mu || !energies_eV || !f) return fail(KG_EINVAL, "kg_kpm_reconstruct: NULL argument");
    if (rows <= 0 || rows > 65535 || M < 1 || n_energies < 1)
        return fail(KG_EINVAL, "kg_kpm_reconstruct: need 1 <= rows <= 65535, M >= 1, n_energies >= 1");
    if (!(scale_eV > 0.0) || !std::isfinite(scale_eV) || !std::isfinite(e0_eV))
        return fail(KG_EINVAL, "kg_kpm_reconstruct: scale must be positive and finite");
    cudaStream_t st = (cudaStream_t)stream;
    // |x_j| < 1 is checked here when the grid is host memory; a device grid is not read back (no
    // synchronisation): energies outside (E0 - s, E0 + s) then give NaN, from sqrt(1 - x^2)
    if (!is_device_ptr(energies_eV))
        for (int j = 0; j < n_energies; ++j)
            if (!(std::fabs((energies_eV[j] - e0_eV) / scale_eV) < 1.0))
                return fail(KG_EINVAL, "kg_kpm_reconstruct: energy %.6g eV is outside (E0 - s, E0 + s)", energies_eV[j]);
    AsyncTmp tmp(st);
    const void *d_mu, *d_en;
    int rc;
    if ((rc = tmp.get(mu, (size_t)rows * M * 16, &d_mu)) || (rc = tmp.get(energies_eV, (size_t)n_energies * 8, &d_en)))
        return rc;
    void *d_w = nullptr, *d_f = f;
    if ((rc = tmp.alloc((size_t)M * 8, &d_w))) return rc;
    const bool f_dev = is_device_ptr(f);
    if (!f_dev && (rc = tmp.alloc((size_t)rows * n_energies * 8, &d_f))) return rc;
    kg_kpm_weights<<<(M + 255) / 256, 256, 0, st>>>(M, jackson, (double *)d_w);
    dim3 grid((n_energies + 127) / 128, (unsigned)rows);
    kg_kpm_reconstruct_kernel<<<grid, 128, 0, st>>>((const c128 *)d_mu, rows, M, (const double *)d_w, e0_eV, scale_eV,
                                                    (const double *)d_en, n_energies, (double *)d_f);
    CUDA_TRY(cudaGetLastError());
    if (!f_dev) CUDA_TRY(cudaMemcpyAsync(f, d_f, (size_t)rows * n_energies * 8, cudaMemcpyDeviceToHost, st));
    return KG_OK;
    });
}

extern "C" int kg_transport(int n_steps, int n_energies, double dt_fs, double dens_per_nm2, double width_nm,
                            const double *rho, const double *fvac, const double *fmsd, double *sigma_gk,
                            double *sigma_e1, double *sigma_e2, double *length_nm, double *conductance,
                            void *stream)
{
    return guarded([&]() -> int {
    if (n_steps < 0 || n_energies < 1) return fail(KG_EINVAL, "kg_transport: n_steps >= 0, n_energies >= 1");
    if (!(dt_fs > 0.0) || !std::isfinite(dt_fs) || !std::isfinite(dens_per_nm2) || !std::isfinite(width_nm))
        return fail(KG_EINVAL, "kg_transport: dt_fs must be positive; dens and width finite");
    if (sigma_gk && !fvac) return fail(KG_EINVAL, "kg_transport: sigma_gk needs fvac");
    if ((sigma_e1 || sigma_e2 || length_nm || conductance) && !fmsd)
        return fail(KG_EINVAL, "kg_transport: sigma_e1 / sigma_e2 / length / conductance need fmsd");
    if ((length_nm || conductance) && !rho) return fail(KG_EINVAL, "kg_transport: length / conductance need rho");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t tbytes = (size_t)(n_steps + 1) * n_energies * 8;
    AsyncTmp tmp(st);
    const void *d_rho, *d_vac, *d_msd;
    int rc;
    if ((rc = tmp.get(rho, (size_t)n_energies * 8, &d_rho)) || (rc = tmp.get(sigma_gk ? fvac : nullptr, tbytes, &d_vac)) ||
        (rc = tmp.get(fmsd, tbytes, &d_msd)))
        return rc;
    double *user[5] = {sigma_gk, sigma_e1, sigma_e2, length_nm, conductance};
    double *dev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    for (int q = 0; q < 5; ++q) {
        if (!user[q]) continue;
        if (is_device_ptr(user[q])) { dev[q] = user[q]; continue; }
        void *d;
        if ((rc = tmp.alloc(tbytes, &d))) return rc;
        dev[q] = (double *)d;
    }
    kg_transport_kernel<<<(n_energies + 127) / 128, 128, 0, st>>>(n_steps, n_energies, dt_fs,
        2.0 * 3.14159265358979323846 * KG_HBAR * dens_per_nm2, width_nm, (const double *)d_rho,
        (const double *)d_vac, (const double *)d_msd, dev[0], dev[1], dev[2], dev[3], dev[4]);
    CUDA_TRY(cudaGetLastError());
    for (int q = 0; q < 5; ++q)
        if (user[q] && dev[q] != user[q]) CUDA_TRY(cudaMemcpyAsync(user[q], dev[q], tbytes, cudaMemcpyDeviceToHost, st));
    return KG_OK;
    });
}

// --------------------------------------------------------------------------------------
// Fourier-transform method: Alg. 4 = kg_evolve in a loop + inner products
// --------------------------------------------------------------------------------------
static int dot_device(kg_hamiltonian *h, const c128 *a, int ld_a, const c128 *b, int R, c128 *partial,
                      int grid, cudaStream_t st)
{
    switch (R) {
    case 1: kg_dot_kernel<1><<<grid, 256, 0, st>>>(a, ld_a, b, h->n, partial); break;
    case 2: kg_dot_kernel<2><<<grid, 256, 0, st>>>(a, ld_a, b, h->n, partial); break;
    case 4: kg_dot_kernel<4><<<grid, 256, 0, st>>>(a, ld_a, b, h->n, partial); break;
    case 8: kg_dot_kernel<8><<<grid, 256, 0, st>>>(a, ld_a, b, h->n, partial); break;
    case 16: kg_dot_kernel<16><<<grid, 256, 0, st>>>(a, ld_a, b, h->n, partial); break;
    default: return fail(KG_EUNSUPPORTED, "R must be 1, 2, 4, 8 or 16");
    }
    h->launches++;
    CUDA_TRY(cudaGetLastError());
    return KG_OK;
}

extern "C" int kg_fourier_moments(kg_hamiltonian *h, const kg_c128 *phiL, const kg_c128 *phiR, int R, int Nm,
                                  double dtau_fs, double bessel_eps, kg_c128 *F, void *stream)
{
    return guarded([&]() -> int {
    if (!h || !phiL || !phiR || !F) return fail(KG_EINVAL, "kg_fourier_moments: NULL argument");
    if (!r_ok(R, true)) return fail(KG_EUNSUPPORTED, "R must be 1, 2, 4, 8 or 16");
    if (Nm < 0) return fail(KG_EINVAL, "Nm must be >= 0");
    if (!(dtau_fs > 0.0) || !std::isfinite(dtau_fs)) return fail(KG_EINVAL, "dtau_fs must be finite and positive");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t vbytes = (size_t)h->n * R * 16;
    const int rows = 2 * Nm + 1;
    const int grid = grid_for(h, h->n * R);
    const void *dL, *dR;
    void *b0, *b1, *part;
    OutStage o;
    int rc;
    if ((rc = vec_in(h, WS_IN0, phiL, R, st, &dL))) return rc;
    if (phiR == phiL) dR = dL;
    else if ((rc = vec_in(h, WS_IN1, phiR, R, st, &dR))) return rc;
    if ((rc = ws_get(h, WS_S0, vbytes, &b0)) || (rc = ws_get(h, WS_S1, vbytes, &b1)) ||
        (rc = ws_get(h, WS_PART, (size_t)rows * grid * R * 16, &part)) ||
        (rc = stage_out(h, WS_MU, F, (size_t)R * rows * 16, &o)))
        return rc;
    const size_t prow = (size_t)grid * R;
    c128 *P = (c128 *)part;
    if ((rc = dot_device(h, (const c128 *)dL, R, (const c128 *)dR, R, P + (size_t)Nm * prow, grid, st))) return rc;   // l.2
    for (int dir = +1; dir >= -1; dir -= 2) {
        const c128 *cur = (const c128 *)dR;                                       // l.1 / l.7
        c128 *nxt = (c128 *)b0;
        for (int m = 1; m <= Nm; ++m) {
            if ((rc = evolve_device(h, cur, R, nxt, R, dir * dtau_fs, bessel_eps, st)) ||             // l.4 / l.9
                (rc = dot_device(h, (const c128 *)dL, R, nxt, R, P + (size_t)(Nm + dir * m) * prow, grid, st)))   // l.5 / l.10
                return rc;
            cur = nxt;
            nxt = (nxt == (c128 *)b0) ? (c128 *)b1 : (c128 *)b0;
        }
    }
    kg_reduce_partials<<<(rows * R * 32 + 255) / 256, 256, 0, st>>>(P, rows, grid, R, (c128 *)o.dev, rows, 0);
    h->launches++;
    CUDA_TRY(cudaGetLastError());
    return finish_out(o, st);
    });
}

extern "C" int kg_ftm_reconstruct(const kg_c128 *F, int64_t rows, int Nm, int window, double dtau_fs,
                                  const double *energies_eV, int n_energies, double *f, void *stream)
{
    return guarded([&]() -> int {
    if (!F || !energies_eV || !f) return fail(KG_EINVAL, "kg_ftm_reconstruct: NULL argument");
    if (rows <= 0 || rows > 65535 || Nm < 0 || n_energies < 1)
        return fail(KG_EINVAL, "kg_ftm_reconstruct: need 1 <= rows <= 65535, Nm >= 0, n_energies >= 1");
    if (!(dtau_fs > 0.0) || !std::isfinite(dtau_fs)) return fail(KG_EINVAL, "dtau_fs must be finite and positive");
    cudaStream_t st = (cudaStream_t)stream;
    AsyncTmp tmp(st);
    const void *d_F, *d_en;
    int rc;
    if ((rc = tmp.get(F, (size_t)rows * (2 * Nm + 1) * 16, &d_F)) ||
        (rc = tmp.get(energies_eV, (size_t)n_energies * 8, &d_en)))
        return rc;
    void *d_f = f;
    const bool f_dev = is_device_ptr(f);
    if (!f_dev && (rc = tmp.alloc((size_t)rows * n_energies * 8, &d_f))) return rc;
    dim3 grid((n_energies + 127) / 128, (unsigned)rows);
    kg_ftm_reconstruct_kernel<<<grid, 128, 0, st>>>((const c128 *)d_F, rows, Nm, window, dtau_fs / KG_HBAR,
                                                    (const double *)d_en, n_energies, (double *)d_f);
    CUDA_TRY(cudaGetLastError());
    if (!f_dev) CUDA_TRY(cudaMemcpyAsync(f, d_f, (size_t)rows * n_energies * 8, cudaMemcpyDeviceToHost, st));
    return KG_OK;
    });
}

// --------------------------------------------------------------------------------------
// kg_kpm_reconstruct_noalloc — the KPM reconstruction for callers that must not allocate.
//
// kg_kpm_reconstruct keeps the damped weights (2 - delta_m0) g_m in a temporary device buffer
// taken from the stream-ordered pool.  Some users of this library cannot afford that: a host
// application that has handed every byte of HBM to its own arena (a framework's caching
// allocator, or a job whose Chebyshev vectors were sized to fill the 180 GB) gets an
// out-of-memory error from any further cudaMalloc / pool growth, and a service that reconstructs
// spectra inside a latency-bound loop cannot take the device-wide stall a fresh allocation may
// cost.  For them the weights live in the fixed array below, which is part of the library image:
// KG_KPM_NOALLOC_MAX_M doubles = 128 KiB on every GPU that loads libkg, held until the process
// exits.  The call path underneath issues two kernel launches and nothing else — no cudaMalloc,
// cudaMallocAsync, cudaFree, no copy, no std::vector.
//
// The array is ONE per device, shared by every call and every stream: a call overwrites entries
// 0..M-1 (entries beyond M keep whatever an earlier call left and are never read, so nothing has
// to be cleared first), and two calls that overlap on the GPU — different streams, or different
// host threads — race on it.
//
// In host code `g_kpm_noalloc_w` is only a stand-in for the symbol; the device address is fetched
// with cudaGetSymbolAddress once per device (with that device current) the first time the entry
// point is called there, and cached.  That first call loads the module's data on the device, so
// it should be made outside any stream capture.
// --------------------------------------------------------------------------------------
static __device__ __align__(256) double g_kpm_noalloc_w[KG_KPM_NOALLOC_MAX_M];

#define KG_NOALLOC_MAX_DEVICES 64
static std::mutex g_noalloc_lock;
static double *g_noalloc_w_dev[KG_NOALLOC_MAX_DEVICES];   // device address of the array, per device ordinal

static int noalloc_weights(double **w)
{
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= KG_NOALLOC_MAX_DEVICES)
        return fail(KG_EUNSUPPORTED, "kg_kpm_reconstruct_noalloc: device ordinal %d is beyond the %d this entry point tracks",
                    dev, KG_NOALLOC_MAX_DEVICES);
    std::lock_guard<std::mutex> hold(g_noalloc_lock);
    if (!g_noalloc_w_dev[dev]) {
        void *p = nullptr;
        CUDA_TRY(cudaGetSymbolAddress(&p, g_kpm_noalloc_w));
        if (!p) return fail(KG_ECUDA, "kg_kpm_reconstruct_noalloc: cudaGetSymbolAddress returned a null address");
        g_noalloc_w_dev[dev] = (double *)p;
    }
    *w = g_noalloc_w_dev[dev];
    return KG_OK;
}

extern "C" int kg_kpm_reconstruct_noalloc(const kg_c128 *mu, int64_t rows, int M, int jackson, double e0_eV,
                                          double scale_eV, const double *energies_eV, int n_energies,
                                          double *f, void *stream)
{
    return guarded([&]() -> int {
    if (!mu || !energies_eV || !f) return fail(KG_EINVAL, "kg_kpm_reconstruct_noalloc: NULL argument");
    if (rows <= 0 || rows > 65535 || M < 1 || n_energies < 1)
        return fail(KG_EINVAL, "kg_kpm_reconstruct_noalloc: need 1 <= rows <= 65535, M >= 1, n_energies >= 1");
    if (M > KG_KPM_NOALLOC_MAX_M)
        return fail(KG_EINVAL, "kg_kpm_reconstruct_noalloc: M = %d exceeds the fixed weight table of "
                    "KG_KPM_NOALLOC_MAX_M = %d entries; use kg_kpm_reconstruct (which allocates) for longer series",
                    M, KG_KPM_NOALLOC_MAX_M);
    if (!(scale_eV > 0.0) || !std::isfinite(scale_eV) || !std::isfinite(e0_eV))
        return fail(KG_EINVAL, "kg_kpm_reconstruct_noalloc: scale must be positive and finite");
    // a host array would have to be staged in device memory, i.e. allocated: not here
    if (!is_device_ptr(mu) || !is_device_ptr(energies_eV) || !is_device_ptr(f))
        return fail(KG_EINVAL, "kg_kpm_reconstruct_noalloc: mu, energies_eV and f must be device memory "
                    "(staging a host array needs an allocation; kg_kpm_reconstruct does that)");
    double *d_w = nullptr;
    int rc;
    if ((rc = noalloc_weights(&d_w))) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    kg_kpm_weights<<<(M + 255) / 256, 256, 0, st>>>(M, jackson, d_w);
    dim3 grid((n_energies + 127) / 128, (unsigned)rows);
    kg_kpm_reconstruct_kernel<<<grid, 128, 0, st>>>((const c128 *)mu, rows, M, d_w, e0_eV, scale_eV, energies_eV,
                                                    n_energies, f);
    CUDA_TRY(cudaGetLastError());
    return KG_OK;
    });
}
