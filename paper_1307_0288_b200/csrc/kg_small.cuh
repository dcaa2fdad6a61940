// kg_small.cuh — the whole moment loop of Alg. 5 (eq 38, eq 46) in ONE launch
// for launch-bound sizes (sm_100a): a single thread-block cluster keeps T_m, T_{m-1}, the matrix rows
// and phi_L of every tile in (distributed) shared memory and runs steps m = 2 .. on the device, one
// cluster barrier per Chebyshev step; neighbours that live in another CTA's tile are read through
// DSMEM.  BASELINE config 1 (4096 sites: 64 KB per vector, 0.1 us of bandwidth work per step) spends
// 2.8-4.1 us per step when every step is a kernel launch.
//
// Bitwise equal to the multi-launch path (kg_staged.cuh with grid = number of tiles): the same
// 512-element tiles, the same element -> thread assignment (le = tid + q * 256), the same arithmetic
// per element, the same per-thread summation order, the same block tree, and the per-tile partial
// of step m is written to the slot the staged CTA of that tile writes (tiles are swept in reverse
// order on odd steps there).  The first step (T_1, moments 0-2) and the final fixed-order reduction
// stay the launches they are in the multi-launch path.
#pragma once
#include <cooperative_groups.h>

#include "kg_common.cuh"

#define SM_TILE_E 512
#define SM_THREADS 256
#define SM_MAX_CLUSTER 8        // portable cluster size
#define SM_BIG_CLUSTER 16       // non-portable size B200 schedules inside one GPC (tried first for 9-16 tiles)

struct SmallArgs {
    const int32_t *nl;       // [K][ns]
    const double *hop;       // [K][ns]  H_ik / s
    const double *onsite;    // [ns]
    int64_t n, ns;
    int K, ons;
    const c128 *t0, *t1;     // T_0 (phi_R) and T_1, [n][R]
    const c128 *phiL;        // MODE_MOM: phi_L
    c128 *part;              // partial rows [row][ntiles][PR]
    int m_end;               // steps m = 2 .. m_end - 1
    int ntiles, vt;          // tiles in total, tiles per CTA (CTA c owns tiles c*vt .. c*vt + vt - 1)
    int alternate;
};

// shared memory of one tile: cur, prev (16 B x 512 each), aux (MODE_MOM), idx [K][CS], hop [K][CS], ons [CS]
__host__ __device__ constexpr size_t sm_tile_bytes(int R, int K, bool aux)
{
    return (size_t)SM_TILE_E * 16 * (aux ? 3 : 2) + (size_t)(SM_TILE_E / R) * (K * 12 + 8);
}

// Sum `v` and `v2` over the lanes of a warp that share (lane % R), then over the warps: the same tree as
// block_reduce_per_r (kg_common.cuh) for each value, with one pair of barriers for both.
template <int R>
__device__ __forceinline__ void sm_reduce2(c128 &v, c128 &v2, c128 *red /* [2][32][R] */)
{
#pragma unroll
    for (int off = 16; off >= R; off >>= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, off);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, off);
        v2.x += __shfl_xor_sync(0xffffffffu, v2.x, off);
        v2.y += __shfl_xor_sync(0xffffffffu, v2.y, off);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int NW = SM_THREADS / 32;
    if (lane < R) { red[warp * R + lane] = v; red[(32 + warp) * R + lane] = v2; }
    __syncthreads();
    c128 tot = make_double2(0.0, 0.0), tot2 = make_double2(0.0, 0.0);
    if (threadIdx.x < R) {
        for (int w = 0; w < NW; ++w) {
            tot.x += red[w * R + threadIdx.x].x; tot.y += red[w * R + threadIdx.x].y;
            tot2.x += red[(32 + w) * R + threadIdx.x].x; tot2.y += red[(32 + w) * R + threadIdx.x].y;
        }
    }
    __syncthreads();
    v = tot; v2 = tot2;
}

// KU: compile-time bound of the neighbour loop (rows are K <= KU wide; slots k >= K are skipped)
template <int R, int MODE, int KU>
__global__ void __launch_bounds__(SM_THREADS) kg_small_kernel(const SmallArgs a)
{
    namespace cg = cooperative_groups;
    constexpr int CS = SM_TILE_E / R;
    constexpr bool AUX = MODE == MODE_MOM;
    constexpr int RH = (MODE == MODE_MOMX && R > 1) ? R / 2 : 0;
    constexpr int PR = R - RH;
    extern __shared__ __align__(128) unsigned char sm_smem[];
    __shared__ c128 red[64 * R];
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    const int tid = threadIdx.x;
    const int r = tid & (R - 1);
    const int K = a.K;
    const size_t tb = sm_tile_bytes(R, K, AUX);
    const int64_t total = a.n * R;

    auto vec = [&](unsigned char *base, int lvt, int which) {    // which: 0 / 1 = the two Chebyshev buffers, 2 = aux
        return reinterpret_cast<c128 *>(base + (size_t)lvt * tb + (size_t)which * SM_TILE_E * 16);
    };
    auto idx_of = [&](int lvt) { return reinterpret_cast<int32_t *>(sm_smem + (size_t)lvt * tb + (size_t)SM_TILE_E * 16 * (AUX ? 3 : 2)); };

    // ---- load: T_1 -> buffer 0, T_0 -> buffer 1, phi_L, matrix rows ----
    for (int lvt = 0; lvt < a.vt; ++lvt) {
        const int t = rank * a.vt + lvt;
        if (t >= a.ntiles) break;
        const int64_t e0 = (int64_t)t * SM_TILE_E, site0 = (int64_t)t * CS;
        for (int le = tid; le < SM_TILE_E; le += SM_THREADS) {
            const bool in = e0 + le < total;
            const c128 z = make_double2(0.0, 0.0);
            vec(sm_smem, lvt, 0)[le] = in ? a.t1[e0 + le] : z;
            vec(sm_smem, lvt, 1)[le] = in ? a.t0[e0 + le] : z;
            if (AUX) vec(sm_smem, lvt, 2)[le] = in ? a.phiL[e0 + le] : z;
        }
        int32_t *ix = idx_of(lvt);
        double *hp = reinterpret_cast<double *>(ix + K * CS);
        double *on = hp + K * CS;
        for (int q = tid; q < K * CS; q += SM_THREADS) {
            const int k = q / CS, ls = q - k * CS;
            // where the neighbour lives: (owner CTA << 24) | (its tile slot there << 16) | site offset in that tile
            const int m = a.nl[(int64_t)k * a.ns + site0 + ls];  // rows beyond n are padding (index 0, hopping 0)
            const int tt = m / CS, owner = tt / a.vt;
            ix[q] = (owner << 24) | ((tt - owner * a.vt) << 16) | (m - tt * CS);
            hp[q] = a.hop[(int64_t)k * a.ns + site0 + ls];
        }
        for (int ls = tid; ls < CS; ls += SM_THREADS) on[ls] = a.onsite[site0 + ls];
    }
    cluster.sync();

    int cur_b = 0;                                               // buffer holding T_{m-1} ("cur" of step m)
    for (int m = 2; m < a.m_end; ++m) {
        const bool dbl = MODE != MODE_MOM;
        const size_t prow = (size_t)a.ntiles * PR;
        c128 *p1 = a.part + (size_t)(dbl ? 2 * m - 1 : m) * prow, *p2 = a.part + (size_t)(2 * m) * prow;
        const int reverse = a.alternate ? (m & 1) : 0;
        for (int lvt = 0; lvt < a.vt; ++lvt) {
            const int t = rank * a.vt + lvt;
            if (t >= a.ntiles) break;
            const int64_t e0 = (int64_t)t * SM_TILE_E;
            const int64_t rem = total - e0;
            const int ne = (int)(rem < SM_TILE_E ? rem : SM_TILE_E);
            const c128 *cur = vec(sm_smem, lvt, cur_b);
            c128 *prev = vec(sm_smem, lvt, cur_b ^ 1);
            const c128 *aux = vec(sm_smem, lvt, 2);
            const int32_t *ix = idx_of(lvt);
            const double *hp = reinterpret_cast<const double *>(ix + K * CS);
            const double *on = hp + K * CS;
            c128 sum = make_double2(0.0, 0.0), sum2 = make_double2(0.0, 0.0);
#pragma unroll
            for (int q = 0; q < SM_TILE_E / SM_THREADS; ++q) {
                const int le = tid + q * SM_THREADS;
                const int ls = le / R;
                c128 acc = make_double2(0.0, 0.0);
                if (a.ons) {
                    const double eps = on[ls];
                    const c128 self = cur[le];
                    acc.x = eps * self.x; acc.y = eps * self.y;
                }
                c128 v[KU];
                double hk[KU];
#pragma unroll
                for (int k = 0; k < KU; ++k) {
                    if (k < K) {
                        const int w = ix[k * CS + ls];
                        const int owner = w >> 24;
                        const c128 *src = vec(sm_smem, (w >> 16) & 0xFF, cur_b) + (w & 0xFFFF) * R + r;
                        if (owner != rank) src = cluster.map_shared_rank(src, owner);
                        v[k] = *src;
                        hk[k] = hp[k * CS + ls];
                    }
                }
#pragma unroll
                for (int k = 0; k < KU; ++k)
                    if (k < K) cfma_r(acc, hk[k], v[k]);
                const c128 p = prev[le];
                const c128 tt2 = make_double2(fma(2.0, acc.x, -p.x), fma(2.0, acc.y, -p.y));
                c128 tl = make_double2(0.0, 0.0);
                if (MODE == MODE_MOMX) {
                    const int src = (tid - (R > 1 ? R / 2 : 1)) & 31;
                    tl.x = __shfl_sync(0xffffffffu, tt2.x, src);
                    tl.y = __shfl_sync(0xffffffffu, tt2.y, src);
                }
                if (le < ne) {
                    prev[le] = tt2;                                          // T_{m+1} over T_{m-1} (own element only)
                    if (MODE == MODE_MOM) {
                        const c128 Lv = aux[le];
                        sum.x = fma(Lv.x, tt2.x, fma(Lv.y, tt2.y, sum.x));
                        sum.y = fma(Lv.x, tt2.y, fma(-Lv.y, tt2.x, sum.y));
                    } else if (MODE == MODE_MOMX) {
                        constexpr int RHH = R > 1 ? R / 2 : 1;
                        if (r >= RHH) {
                            const c128 sl = cur[le - RHH];
                            sum.x = fma(sl.x, tt2.x, fma(sl.y, tt2.y, sum.x));
                            sum.y = fma(sl.x, tt2.y, fma(-sl.y, tt2.x, sum.y));
                            sum2.x = fma(tl.x, tt2.x, fma(tl.y, tt2.y, sum2.x));
                            sum2.y = fma(tl.x, tt2.y, fma(-tl.y, tt2.x, sum2.y));
                        }
                    } else {
                        const c128 sv = cur[le];
                        sum.x = fma(sv.x, tt2.x, fma(sv.y, tt2.y, sum.x));
                        sum.y = fma(sv.x, tt2.y, fma(-sv.y, tt2.x, sum.y));
                        sum2.x = fma(tt2.x, tt2.x, fma(tt2.y, tt2.y, sum2.x));
                    }
                }
            }
            // the slot the staged CTA of this tile writes: CTA b sweeps tile b, or ntiles - 1 - b on reversed steps
            const int64_t slot = (int64_t)(reverse ? a.ntiles - 1 - t : t) * PR + (tid - RH);
            const bool writer = tid >= RH && tid < R;
            sm_reduce2<R>(sum, sum2, red);
            if (writer) {
                p1[slot] = sum;
                if (dbl) p2[slot] = sum2;
            }
        }
        cur_b ^= 1;
        cluster.sync();                                          // T_m complete everywhere before anyone overwrites T_{m-1}
    }
}


// ---------------------------------------------------------------------------------------------------
// Register-resident form for the smallest batches (VT <= 2 tiles per CTA, <= 8192 elements in all):
// everything that does not change from step to step — where each neighbour lives (a shared::cluster
// address, own or remote CTA), its hopping, the on-site energy — is decoded ONCE into registers, so a
// Chebyshev step is a handful of loads and FMAs per element; the cross-warp part of the moment sums is
// done for SM_BATCH steps at a time (same fixed tree), and the cluster barrier is split into arrive (right
// after the last shared-memory write of the step) and wait (before the first remote read of the next).
// Same arithmetic, same summation order, same partial slots as kg_small_kernel / kg_staged_kernel.
// ---------------------------------------------------------------------------------------------------
#define SM_BATCH 8

__device__ __forceinline__ uint32_t sm_mapa(uint32_t addr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ c128 sm_ld_cluster(uint32_t addr)
{
    c128 v;
    asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory");
    return v;
}

template <int R, int MODE, int KU, int VT>
__global__ void __launch_bounds__(SM_THREADS) kg_small_reg_kernel(const SmallArgs a)
{
    namespace cg = cooperative_groups;
    constexpr int CS = SM_TILE_E / R;
    constexpr bool AUX = MODE == MODE_MOM;
    constexpr bool DBL = MODE != MODE_MOM;
    constexpr int RH = (MODE == MODE_MOMX && R > 1) ? R / 2 : 0;
    constexpr int PR = R - RH;
    constexpr int EPT = SM_TILE_E / SM_THREADS;
    constexpr int NW = SM_THREADS / 32;
    extern __shared__ __align__(128) unsigned char sm_smem[];
    __shared__ c128 ring[SM_BATCH][2][NW][R];
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r = tid & (R - 1);
    const int K = a.K;
    const size_t tb = sm_tile_bytes(R, K, AUX);
    const int64_t total = a.n * R;
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(sm_smem);

    // ---- load (as kg_small_kernel): T_1 -> buffer 0, T_0 -> buffer 1, phi_L -> buffer 2 ----
#pragma unroll
    for (int lvt = 0; lvt < VT; ++lvt) {
        const int t = rank * VT + lvt;
        if (t >= a.ntiles) break;
        const int64_t e0 = (int64_t)t * SM_TILE_E;
        c128 *b0 = reinterpret_cast<c128 *>(sm_smem + (size_t)lvt * tb);
        for (int le = tid; le < SM_TILE_E; le += SM_THREADS) {
            const bool in = e0 + le < total;
            const c128 z = make_double2(0.0, 0.0);
            b0[le] = in ? a.t1[e0 + le] : z;
            b0[SM_TILE_E + le] = in ? a.t0[e0 + le] : z;
            if (AUX) b0[2 * SM_TILE_E + le] = in ? a.phiL[e0 + le] : z;
        }
    }
    // ---- per-element constants ----
    uint32_t nb[VT][EPT][KU], own[VT][EPT];
    double hk[VT][EPT][KU], eps[VT][EPT];
    c128 Lv[VT][EPT];
    bool live[VT][EPT];
#pragma unroll
    for (int lvt = 0; lvt < VT; ++lvt) {
        const int t = rank * VT + lvt;
        const int64_t e0 = (int64_t)t * SM_TILE_E, site0 = (int64_t)t * CS;
#pragma unroll
        for (int q = 0; q < EPT; ++q) {
            const int le = tid + q * SM_THREADS, ls = le / R;
            live[lvt][q] = t < a.ntiles && e0 + le < total;
            own[lvt][q] = base + (uint32_t)((size_t)lvt * tb) + (uint32_t)le * 16u;
            eps[lvt][q] = (t < a.ntiles && a.ons) ? a.onsite[site0 + ls] : 0.0;
            Lv[lvt][q] = (AUX && live[lvt][q]) ? a.phiL[e0 + le] : make_double2(0.0, 0.0);
#pragma unroll
            for (int k = 0; k < KU; ++k) {
                nb[lvt][q][k] = own[lvt][q];
                hk[lvt][q][k] = 0.0;
                if (k < K && t < a.ntiles) {
                    const int m = a.nl[(int64_t)k * a.ns + site0 + ls];
                    const int tt = m / CS, owner = tt / VT;
                    const uint32_t la = base + (uint32_t)((size_t)(tt - owner * VT) * tb) + (uint32_t)((m - tt * CS) * R + r) * 16u;
                    nb[lvt][q][k] = sm_mapa(la, (uint32_t)owner);
                    hk[lvt][q][k] = a.hop[(int64_t)k * a.ns + site0 + ls];
                }
            }
        }
    }
    cluster.sync();

    uint32_t cur_off = 0, prev_off = SM_TILE_E * 16;              // byte offsets of the two Chebyshev buffers
    const size_t prow = (size_t)a.ntiles * PR;
    int pending = 0, first_pending = 2;
    auto flush = [&](int m_first, int count) {
        // cross-warp sums of `count` steps m_first .. : thread (j * R + rr) finishes step j, column rr of each tile
        __syncthreads();
        for (int lvt = 0; lvt < VT; ++lvt) {
            const int t = rank * VT + lvt;
            if (t >= a.ntiles) break;
            for (int j = tid / R; j < count; j += SM_THREADS / R) {
                const int rr = tid & (R - 1), m = m_first + j;
                // ring rows are per (step, tile): [j][lvt]
                c128 tot = make_double2(0.0, 0.0), tot2 = make_double2(0.0, 0.0);
                for (int w = 0; w < NW; ++w) {
                    const c128 x = ring[(j * VT + lvt) % SM_BATCH][0][w][rr], y = ring[(j * VT + lvt) % SM_BATCH][1][w][rr];
                    tot.x += x.x; tot.y += x.y; tot2.x += y.x; tot2.y += y.y;
                }
                if (rr >= RH) {
                    const int reverse = a.alternate ? (m & 1) : 0;
                    const int64_t slot = (int64_t)(reverse ? a.ntiles - 1 - t : t) * PR + (rr - RH);
                    a.part[(size_t)(DBL ? 2 * m - 1 : m) * prow + slot] = tot;
                    if (DBL) a.part[(size_t)(2 * m) * prow + slot] = tot2;
                }
            }
        }
        __syncthreads();
    };
    constexpr int STEPS_PER_FLUSH = SM_BATCH / VT;

    for (int m = 2; m < a.m_end; ++m) {
#pragma unroll
        for (int lvt = 0; lvt < VT; ++lvt) {
            c128 sum = make_double2(0.0, 0.0), sum2 = make_double2(0.0, 0.0);
#pragma unroll
            for (int q = 0; q < EPT; ++q) {
                c128 v[KU];
#pragma unroll
                for (int k = 0; k < KU; ++k)
                    if (k < K) v[k] = sm_ld_cluster(nb[lvt][q][k] + cur_off);
                c128 self, p;
                asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(self.x), "=d"(self.y) : "r"(own[lvt][q] + cur_off) : "memory");
                asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(p.x), "=d"(p.y) : "r"(own[lvt][q] + prev_off) : "memory");
                c128 acc = make_double2(0.0, 0.0);
                if (a.ons) { acc.x = eps[lvt][q] * self.x; acc.y = eps[lvt][q] * self.y; }
#pragma unroll
                for (int k = 0; k < KU; ++k)
                    if (k < K) cfma_r(acc, hk[lvt][q][k], v[k]);
                const c128 tt2 = make_double2(fma(2.0, acc.x, -p.x), fma(2.0, acc.y, -p.y));
                c128 tl = make_double2(0.0, 0.0), sl = make_double2(0.0, 0.0);
                if (MODE == MODE_MOMX) {
                    const int src = (tid - (R > 1 ? R / 2 : 1)) & 31;
                    tl.x = __shfl_sync(0xffffffffu, tt2.x, src); tl.y = __shfl_sync(0xffffffffu, tt2.y, src);
                    sl.x = __shfl_sync(0xffffffffu, self.x, src); sl.y = __shfl_sync(0xffffffffu, self.y, src);
                }
                if (live[lvt][q]) {
                    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(own[lvt][q] + prev_off), "d"(tt2.x), "d"(tt2.y) : "memory");
                    if (MODE == MODE_MOM) {
                        sum.x = fma(Lv[lvt][q].x, tt2.x, fma(Lv[lvt][q].y, tt2.y, sum.x));
                        sum.y = fma(Lv[lvt][q].x, tt2.y, fma(-Lv[lvt][q].y, tt2.x, sum.y));
                    } else if (MODE == MODE_MOMX) {
                        if (r >= (R > 1 ? R / 2 : 1)) {
                            sum.x = fma(sl.x, tt2.x, fma(sl.y, tt2.y, sum.x));
                            sum.y = fma(sl.x, tt2.y, fma(-sl.y, tt2.x, sum.y));
                            sum2.x = fma(tl.x, tt2.x, fma(tl.y, tt2.y, sum2.x));
                            sum2.y = fma(tl.x, tt2.y, fma(-tl.y, tt2.x, sum2.y));
                        }
                    } else {
                        sum.x = fma(self.x, tt2.x, fma(self.y, tt2.y, sum.x));
                        sum.y = fma(self.x, tt2.y, fma(-self.y, tt2.x, sum.y));
                        sum2.x = fma(tt2.x, tt2.x, fma(tt2.y, tt2.y, sum2.x));
                    }
                }
            }
            if (lvt == VT - 1) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
            // warp part of the block tree (as block_reduce_per_r), then park the warp totals in the ring
#pragma unroll
            for (int off = 16; off >= R; off >>= 1) {
                sum.x += __shfl_xor_sync(0xffffffffu, sum.x, off); sum.y += __shfl_xor_sync(0xffffffffu, sum.y, off);
                if (DBL) { sum2.x += __shfl_xor_sync(0xffffffffu, sum2.x, off); sum2.y += __shfl_xor_sync(0xffffffffu, sum2.y, off); }
            }
            if (lane < R) {
                ring[(pending * VT + lvt) % SM_BATCH][0][warp][lane] = sum;
                ring[(pending * VT + lvt) % SM_BATCH][1][warp][lane] = sum2;
            }
        }
        if (++pending == STEPS_PER_FLUSH) { flush(first_pending, pending); first_pending = m + 1; pending = 0; }
        const uint32_t x = cur_off; cur_off = prev_off; prev_off = x;
        asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
    }
    if (pending) flush(first_pending, pending);
}
