// kg_common.cuh — types, argument blocks and device helpers shared by the kernels of libkg
// (sm_100a): kg_kernels.cuh (one thread per element) and kg_staged.cuh (TMA-staged).
//
// One fused kernel family implements every step of the hot path:
//
//   MODE_MOM   T_{m+1} = alpha H~ T_m - beta T_{m-1}  (eq 38)  + per-block partial of
//              <phi_L|T_{m+1}>  (Alg. 5 l.6-7 P:363-365; the paper's K3 and K5 in one pass)
//   MODE_MOM2  the same recursion for phi_L = phi_R = phi with the product identity
//              2 T_a T_b = T_{a+b} + T_{|a-b|}: per-block partials of <T_m|T_{m+1}> (moment
//              2m+1) and <T_{m+1}|T_{m+1}> (moment 2m+2) — two moments per sweep, no phi_L read
//   MODE_MOMX  the same identity for phi_L != phi_R: the batch holds [phi_L | phi_R] as its two
//              column halves, both are advanced by the recursion, and the partials are the CROSS
//              products <T_m L|T_{m+1} R> (moment 2m+1) and <T_{m+1} L|T_{m+1} R> (moment 2m+2);
//              one matrix read serves both chains and there is no separate phi_L stream (VAC)
//   MODE_EVO   same recursion + out (+)= c_{m+1} T_{m+1}              (Alg. 6 l.5-6 P:383-385)
//   MODE_CLEN  (staged kernel only) the same series summed by Clenshaw's backward recurrence
//              b_m = c_m phi + 2 H~ b_{m+1} - b_{m+2}: no accumulator stream
//   MODE_PCLEN (staged kernel only) Clenshaw form of the pair recursion (eq 44):
//              e_m = c_m psix + 2 H~ e_{m+1} + 2 [X,H~] b_{m+1} - e_{m+2} next to b_m
//   MODE_PAIR  (a, d) pair recursion: a = T_m psi, d = T_m psix + [X,T_m] psi,
//              d_{m+1} = alpha([X,H~] a_m + H~ d_m) - beta d_{m-1}    (eq 39, Alg. 7 l.7-8)
//              + both series accumulations                            (eq 44)
//   MODE_VEL   out = V in = -(i s/hbar) [X,H~] in                     (eq 15)
//
// Layout: vectors [n][R] complex128 (double2), one THREAD PER ELEMENT (site i, vector r),
// e = i*R + r, so the R lanes of a site read R consecutive 16-byte values: every own-element
// access is a fully coalesced ld.global.v2.f64, every gather reads R*16 contiguous bytes, and
// the matrix row (index, hopping, on-site) is fetched once per site and broadcast to R lanes.
// The matrix is the paper's k-major neighbour list with row stride `ns` (n rounded up
// to 32 so that each k-slab is 128-byte aligned).
//
// Determinism: a thread's elements are fixed by (grid, block), per-thread sums run in index
// order, the warp/block reduction is a fixed tree, and kg_reduce_partials adds the per-block
// partials in block order: moments are bitwise reproducible.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

typedef double2 c128;

enum { MODE_MOM = 0, MODE_EVO = 1, MODE_PAIR = 2, MODE_VEL = 3, MODE_MOM2 = 4, MODE_MOMX = 5, MODE_CLEN = 6, MODE_PCLEN = 7 };

struct StepArgs {
    // matrix (device, library-owned)
    const int32_t *nl;    // [kmax][ns]
    const double *hop;    // [kmax][ns]  H_ik / s
    const double *xhop;   // [kmax][ns]  (X_i - X_m)_minimg H_ik / s   ([X,H~] weights)
    const double *onsite; // [ns]        (H_ii - E0)/s
    int64_t n;            // sites
    int64_t ns;           // row stride of the k-major arrays
    int kmax;
    double alpha;         // 1 for the first step (T_1 = H~ T_0), 2 afterwards
    // a-chain: element (i, r) of X at X[i*ld + r]
    const c128 *cur;  int ld_cur;    // T_m      (gathered + own)
    const c128 *prev; int ld_prev;   // T_{m-1}  (own element; unused when FIRST)
    c128 *next;                      // T_{m+1}  (ld = R); may alias prev
    // MODE_MOM
    const c128 *phiL; int ld_L;
    c128 *partial;                   // [grid][R] for moment m+1
    c128 *partial0;                  // FIRST only: [grid][R] for moment 0
    c128 *partial2;                  // MODE_MOM2: [grid][R] for moment 2m+2 (partial: 2m+1)
    // MODE_EVO / MODE_PAIR: series accumulators (ld = R)
    c128 *out;
    c128 c0, c1;                     // FIRST: out = c0 cur + c1 next; else out += c1 next
    // MODE_PAIR d-chain
    const c128 *dcur; int ld_dcur;
    const c128 *dprev; int ld_dprev;
    c128 *dnext;
    c128 *outd;
    // MODE_VEL
    c128 *vout; int ld_vout;
    double vscale;                   // s / hbar
};

__device__ __forceinline__ c128 ld_nc(const c128 *p)
{
    return __ldg(reinterpret_cast<const double2 *>(p));
}
__device__ __forceinline__ c128 cmul(c128 a, c128 b)
{
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ void cfma_r(c128 &acc, double h, c128 v)
{
    acc.x = fma(h, v.x, acc.x);
    acc.y = fma(h, v.y, acc.y);
}

// Sum `v` over the lanes of a warp that share (lane % R), then over warps; thread tid < R of
// the block ends up with the block total for vector r = tid.  Fixed tree => deterministic.
template <int R>
__device__ __forceinline__ c128 block_reduce_per_r(c128 v, c128 *smem /* [32][R] */)
{
#pragma unroll
    for (int off = 16; off >= R; off >>= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, off);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, off);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nwarps = blockDim.x >> 5;
    if (lane < R) smem[warp * R + lane] = v;
    __syncthreads();
    c128 tot = make_double2(0.0, 0.0);
    if (threadIdx.x < R) {
        for (int w = 0; w < nwarps; ++w) {
            tot.x += smem[w * R + threadIdx.x].x;
            tot.y += smem[w * R + threadIdx.x].y;
        }
    }
    __syncthreads();
    return tot;
}

