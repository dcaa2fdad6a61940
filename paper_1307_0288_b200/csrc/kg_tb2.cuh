// kg_tb2.cuh — TWO Chebyshev steps per pass over the vectors (sm_100a): the moment sweeps of
// Alg. 5 (eq 38, eq 46) in their doubling forms (MODE_MOM2 / MODE_MOMX, see
// kg_common.cuh), blocked in time inside the SM.
//
// Why: the one-step sweep (kg_staged.cuh) sits on the DRAM line (profiles/r02b_tb2.md: 272 MB must move per
// sweep of config 4 and it takes the time a copy of that size takes): T_m and T_{m-1} are read and T_{m+1}
// written for every
// step, 48 B + the matrix row per site-update.  Here a tile of CS consecutive sites — a compact patch
// of the lattice after the re-ordering of kg_partition.h — is brought into shared memory together with
// its two rings of halo sites
//     H1 = neighbours of the tile outside it,   H2 = neighbours of H1 outside tile + H1,
// T_{m+1} = 2 H~ T_m - T_{m-1} is formed on tile + H1 (the H1 part redundantly: the neighbouring tiles
// compute it too), and T_{m+2} = 2 H~ T_{m+1} - T_m on the tile, without leaving the SM.  Per site and
// PAIR of steps: T_m, T_{m-1} read, T_{m+1}, T_{m+2} written (64 B) + ~10 B of tile-local matrix +
// the halo (~11 %), i.e. ~45 B per site-update instead of ~80.  The four inner products of a pass
//     <T_m|T_{m+1}>, <T_{m+1}|T_{m+1}>, <T_{m+1}|T_{m+2}>, <T_{m+2}|T_{m+2}>     (moments 2m+1 .. 2m+4)
// are accumulated on the tile's own sites.
//
// Per-tile PLAN, built on the host at first use (kg.cu: tb2_build_plan) from the packed list:
//   tinfo[t]              {n1, n2} = |H1|, |H2|
//   hid[t][cap1 + cap2]   internal site index of the H1 sites, then (dense, from n1) of the H2 sites
//   hons[t][cap1]         on-site energy (H_ii - E0)/s of the H1 rows
//   rows[t][CS + cap1][KP] tile-LOCAL matrix rows of the own sites [0, CS) and the H1 sites [CS, CS+n1):
//                         (dictionary id << 12) | local slot;  slots: own j, H1 CS + j, H2 CS + n1 + j
// Everything contiguous of a tile (own T_m, T_{m-1}, on-site energies, hid, hons, rows) is fetched by
// TMA bulk copies completing on one mbarrier; the halo values are 16-byte gathers (L2 hits: they are the
// neighbouring tiles' own elements).  Needs the hopping dictionary (<= 15 distinct H_ik/s, one in the
// paper's model eq 13) and C = 1 or 2 columns per site.  NSTEP = 1 is the same kernel doing a
// single step (odd step counts), so that one call uses one grid and one shape of moment partials.
//
// Wider batches: a launch can serve `nplanes` independent [n][C] batches (column pairs of an [n][R] batch,
// kg.cu: moments_device) side by side — gridDim.x = nplanes * cpp, CTA (plane, bl) sweeps the tiles bl,
// bl + cpp, ... of its plane with the SAME per-tile plan, and writes its partial into the plane's columns of
// the common row [cpp][nplanes * PR], which is the layout of the first-step kernel and of kg_reduce_partials.
//
// Determinism: tile -> CTA -> thread -> row assignment is a pure function of the launch shape, sums run
// in a fixed order, the block tree is fixed, kg_reduce_partials adds the CTA partials in CTA order.
#pragma once
#include "kg_common.cuh"
#include "kg_staged.cuh"

#define TB_CONSUMERS 512       // consumer threads (arithmetic)
#define TB_THREADS (TB_CONSUMERS + 64)   // + a TMA issuer warp (one lane) and a halo gatherer warp (32 lanes)
#define TB_SITES 1024          // C * CS: elements (site, column) of a tile
#define TB_SLOT_MASK 0x0FFF    // local slot in bits 0..11, dictionary id in 12..15
#define TB_MAX_STAGES 4
#define TB_HEADER 2048         // barriers + reduction scratch

__host__ __device__ constexpr int tb_kp(int K) { return (K + 3) / 4 * 4; }
__host__ __device__ constexpr int tb_cs(int C) { return TB_SITES / C; }
// bytes of one shared-memory stage: T_m on own + H1 + H2, T_{m-1} on own + H1, on-site energies of the
// own and H1 rows, halo ids, tile-local rows
__host__ __device__ constexpr size_t tb_stage_bytes(int C, int K, int cap1, int cap2)
{
    return ((size_t)(tb_cs(C) + cap1 + cap2) * C * 16 + (size_t)(tb_cs(C) + cap1) * C * 16 + (size_t)tb_cs(C) * 8 +
            (size_t)cap1 * 8 + (size_t)(cap1 + cap2) * 4 + (size_t)(tb_cs(C) + cap1) * tb_kp(K) * 2 + 127) / 128 * 128;
}

struct Tb2Args {
    const int2 *tinfo;
    const uint16_t *rows;
    const int32_t *hid;
    const double *hons;
    const double *onsite;    // [ns] (H_ii - E0)/s, internal order
    double dict[16];
    int64_t n;
    int cap1, cap2, ntiles, reverse, nstages;
    int nplanes;             // independent [n][C] batches served by one launch (CTAs are split evenly among them)
    int64_t plane_stride;    // elements between consecutive planes in cur / prev / next1 / next2
    const c128 *cur, *prev;  // T_m, T_{m-1}   [n][C]
    c128 *next1, *next2;     // T_{m+1}, T_{m+2}
    c128 *p1, *p2, *p3, *p4; // moment partials [grid][PR] of moments 2m+1 .. 2m+4 (p3, p4: NSTEP = 2)
};

// total over the CTA, valid in thread 0 (fixed tree: xor-shuffles, then the warps in order)
__device__ __forceinline__ c128 tb_block_sum(c128 v, c128 *red)
{
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, off);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, off);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) red[warp] = v;
    __syncthreads();
    c128 tot = make_double2(0.0, 0.0);
    if (threadIdx.x == 0)
        for (int w = 0; w < TB_THREADS / 32; ++w) { tot.x += red[w].x; tot.y += red[w].y; }
    __syncthreads();
    return tot;
}

__device__ __forceinline__ void tb_cdot(c128 &s, c128 a, c128 b)     // s += conj(a) * b
{
    s.x = fma(a.x, b.x, fma(a.y, b.y, s.x));
    s.y = fma(a.x, b.y, fma(-a.y, b.x, s.y));
}
// 16-byte asynchronous copy global -> shared (LDGSTS, L2 only) and its completion on an mbarrier
__device__ __forceinline__ void tb_cp_async16(uint32_t dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void tb_cp_async_arrive(uint32_t bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}

// T_{m+1} / T_{m+2} go out with an L2 evict_last hint: they are what the next pass (which sweeps the tiles
// in the opposite direction) reads first, the streams read by this pass are dead (one-column pass: -2 %)
__device__ __forceinline__ uint64_t tb_keep_policy()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void tb_store_keep(c128 *p, c128 v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}

// one matrix row from shared memory: KP packed uint16 as KP/2 words
template <int KP>
__device__ __forceinline__ void tb_load_row(const uint16_t *rows_s, int row, uint32_t (&w)[KP / 2])
{
    if (KP == 4) {
        const uint2 v = reinterpret_cast<const uint2 *>(rows_s)[row];
        w[0] = v.x; w[1] = v.y;
    } else {
        const uint4 v = reinterpret_cast<const uint4 *>(rows_s)[row];
        w[0] = v.x; w[1] = v.y; w[2] = v.z; w[3] = v.w;
    }
}
template <int KP>
__device__ __forceinline__ uint32_t tb_row_entry(const uint32_t (&w)[KP / 2], int k)
{
    return (k & 1) ? (w[k >> 1] >> 16) : (w[k >> 1] & 0xFFFFu);
}

template <int C, int K, int MODE, bool ONS, int NSTEP>
__global__ void __launch_bounds__(TB_THREADS, 1) kg_tb2_kernel(const Tb2Args a)
{
    constexpr int CS = tb_cs(C), KP = tb_kp(K), RPT = CS / TB_CONSUMERS;     // own rows per consumer thread
    constexpr int PR = MODE == MODE_MOMX ? C / 2 : C;                        // columns of a partial row
    static_assert(MODE == MODE_MOM2 || (MODE == MODE_MOMX && C == 2), "modes of the two-step kernel");
    static_assert(KP == 4 || KP == 8, "row widths up to 8");
    extern __shared__ __align__(128) unsigned char tb_smem[];
    const int cap1 = a.cap1, cap2 = a.cap2, nst = a.nstages;
    uint64_t *bars = reinterpret_cast<uint64_t *>(tb_smem);
    volatile int2 *sinfo = reinterpret_cast<volatile int2 *>(tb_smem + 192);   // {n1, n2} of the tile in each stage
    c128 *red = reinterpret_cast<c128 *>(tb_smem + 256);
    // C = 2: lanes 4-7 of every 8 take the two columns of a site in the other order, so that the 8 lanes of a
    // quarter-warp touch 8 different 16-byte bank groups (site stride 32 B would otherwise collide 2-way)
    const int sw = C == 2 ? ((threadIdx.x >> 2) & 1) : 0;
    const size_t stage_bytes = tb_stage_bytes(C, K, cap1, cap2);
    // offsets inside a stage
    const size_t off_tp = (size_t)(CS + cap1 + cap2) * C * 16;
    const size_t off_ons = off_tp + (size_t)(CS + cap1) * C * 16;
    const size_t off_hons = off_ons + (size_t)CS * 8;
    const size_t off_hid = off_hons + (size_t)cap1 * 8;
    const size_t off_rows = off_hid + (size_t)(cap1 + cap2) * 4;

    const int tid = threadIdx.x;
    const uint64_t keep = tb_keep_policy();
    const uint32_t fa0 = sg_smem_u32(bars), fb0 = sg_smem_u32(bars + TB_MAX_STAGES), em0 = sg_smem_u32(bars + 2 * TB_MAX_STAGES),
                   fh0 = sg_smem_u32(bars + 3 * TB_MAX_STAGES);
    if (tid == 0) {
        for (int s = 0; s < nst; ++s) {
            sg_mbar_init(fh0 + 8 * s, 1);                       // halo ids of the stage (small, lands first)
            sg_mbar_init(fa0 + 8 * s, 1);                       // the other TMA bytes of the stage
            sg_mbar_init(fb0 + 8 * s, 32);                      // halo gathers of the 32 gatherer lanes
            sg_mbar_init(em0 + 8 * s, TB_CONSUMERS / 32);       // consumer warps done with the stage
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // planes: gridDim.x = nplanes * cpp; CTA (plane, bl) sweeps the tiles bl, bl + cpp, ... of its plane
    const int cpp = (int)gridDim.x / a.nplanes, plane = (int)blockIdx.x / cpp, bl = (int)blockIdx.x - plane * cpp;
    const c128 *const cur_p = a.cur + plane * a.plane_stride, *const prev_p = a.prev + plane * a.plane_stride;
    c128 *const next1_p = a.next1 + plane * a.plane_stride;
    c128 *const next2_p = NSTEP == 2 ? a.next2 + plane * a.plane_stride : nullptr;
    const int my_tiles = (bl < a.ntiles) ? (a.ntiles - 1 - bl) / cpp + 1 : 0;
    c128 s1[PR], s2[PR], s3[PR], s4[PR];
#pragma unroll
    for (int c = 0; c < PR; ++c) s1[c] = s2[c] = s3[c] = s4[c] = make_double2(0.0, 0.0);

    auto tile_of = [&](int j) { int t = bl + j * cpp; return a.reverse ? a.ntiles - 1 - t : t; };

    if (tid == TB_CONSUMERS) {
        // ---------------- warp 8, one lane: TMA bulk copies of everything contiguous ----------------
        int s = 0; uint32_t ph = 0;
        int2 info = my_tiles > 0 ? __ldg(a.tinfo + tile_of(0)) : make_int2(0, 0);
        for (int j = 0; j < my_tiles; ++j, ++s) {
            if (s == nst) { s = 0; ph ^= 1u; }
            const int t = tile_of(j);
            const int2 cur_info = info;
            if (j + 1 < my_tiles) info = __ldg(a.tinfo + tile_of(j + 1));     // in flight while this tile is issued
            const int64_t site0 = (int64_t)t * CS, left = a.n - site0;
            const int nown = (int)(left < CS ? left : CS);
            const int n1 = cur_info.x, n2 = cur_info.y;
            const int nh = NSTEP == 2 ? n1 + n2 : n1;
            // always all CS own rows: the plan zero-fills the rows behind a ragged last tile (slot 0, dictionary
            // id 0), so threads with row >= nown gather inside the stage instead of decoding what an earlier
            // tile left there
            const int nrow = NSTEP == 2 ? CS + ((n1 + 1) & ~1) : CS;
            const uint32_t vb = (uint32_t)nown * C * 16u;
            const uint32_t hb = (uint32_t)((nh + 3) & ~3) * 4u;
            const uint32_t rb = (uint32_t)nrow * KP * 2u;
            const uint32_t ob = ONS ? (uint32_t)((nown + 1) & ~1) * 8u : 0u;
            const uint32_t gb = (ONS && NSTEP == 2) ? (uint32_t)((n1 + 1) & ~1) * 8u : 0u;
            while (!sg_mbar_try_wait(em0 + 8 * s, ph ^ 1u)) __nanosleep(32);
            // the stage was written through the generic proxy (halo values, T_{m+1} in place)
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            const uint32_t sb = sg_smem_u32(tb_smem + TB_HEADER + (size_t)s * stage_bytes), fa = fa0 + 8 * s;
            const uint32_t fh = fh0 + 8 * s;
            sinfo[s].x = n1; sinfo[s].y = n2;                    // released by the arrive below
            if (hb) {
                sg_mbar_expect_tx(fh, hb);
                sg_bulk_g2s(sb + (uint32_t)off_hid, a.hid + (size_t)t * (cap1 + cap2), hb, fh);
            } else {
                sg_mbar_arrive(fh);
            }
            sg_mbar_expect_tx(fa, 2u * vb + rb + ob + gb);
            sg_bulk_g2s(sb, cur_p + site0 * C, vb, fa);
            sg_bulk_g2s(sb + (uint32_t)off_tp, prev_p + site0 * C, vb, fa);
            sg_bulk_g2s(sb + (uint32_t)off_rows, a.rows + (size_t)t * (CS + cap1) * KP, rb, fa);
            if (ONS) sg_bulk_g2s(sb + (uint32_t)off_ons, a.onsite + site0, ob, fa);
            if (gb) sg_bulk_g2s(sb + (uint32_t)off_hons, a.hons + (size_t)t * cap1, gb, fa);
        }
    } else if (tid >= TB_CONSUMERS + 32) {
        // ---------------- warp 9: halo values, 16-byte asynchronous gathers (L2 hits) ----------------
        const int lane = tid & 31;
        int s = 0; uint32_t ph = 0;
        for (int j = 0; j < my_tiles; ++j, ++s) {
            if (s == nst) { s = 0; ph ^= 1u; }
            unsigned char *sb = tb_smem + TB_HEADER + (size_t)s * stage_bytes;
            const int32_t *hid_s = reinterpret_cast<const int32_t *>(sb + off_hid);
            const uint32_t tm_s = sg_smem_u32(sb), tp_s = sg_smem_u32(sb + off_tp);
            sg_mbar_wait(fh0 + 8 * s, ph);
            const int n1 = sinfo[s].x, nh = NSTEP == 2 ? n1 + sinfo[s].y : n1;
            for (int q = lane; q < nh; q += 32) {
                const int64_t g = (int64_t)hid_s[q] * C;
#pragma unroll
                for (int c = 0; c < C; ++c) {
                    tb_cp_async16(tm_s + (uint32_t)((CS + q) * C + c) * 16u, cur_p + g + c);
                    if (NSTEP == 2 && q < n1) tb_cp_async16(tp_s + (uint32_t)((CS + q) * C + c) * 16u, prev_p + g + c);
                }
            }
            tb_cp_async_arrive(fb0 + 8 * s);
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
    } else if (tid < TB_CONSUMERS) {
        // ---------------- consumers ----------------
        int s = 0; uint32_t ph = 0;
        for (int j = 0; j < my_tiles; ++j, ++s) {
            if (s == nst) { s = 0; ph ^= 1u; }
            const int t = tile_of(j);
            const int64_t site0 = (int64_t)t * CS, left = a.n - site0;
            const int nown = (int)(left < CS ? left : CS);
            unsigned char *sb = tb_smem + TB_HEADER + (size_t)s * stage_bytes;
            c128 *Tm = reinterpret_cast<c128 *>(sb);
            c128 *Tp = reinterpret_cast<c128 *>(sb + off_tp);
            const double *ons_s = reinterpret_cast<const double *>(sb + off_ons);
            const double *hons_s = reinterpret_cast<const double *>(sb + off_hons);
            const uint16_t *rows_s = reinterpret_cast<const uint16_t *>(sb + off_rows);
            sg_mbar_wait(fa0 + 8 * s, ph);
            sg_mbar_wait(fb0 + 8 * s, ph);
            const int n1 = sinfo[s].x;

            // ---- step 1 on the own rows: RPT rows per thread, all loads first ----
            uint32_t w[RPT][KP / 2];
            double eps[RPT];
            c128 self[RPT][C], t1[RPT][C];
            {
                c128 v[RPT][K][C], p[RPT][C];
#pragma unroll
                for (int q = 0; q < RPT; ++q) {
                    const int row = tid + q * TB_CONSUMERS;
                    tb_load_row<KP>(rows_s, row, w[q]);
                    eps[q] = ONS ? ons_s[row] : 0.0;
#pragma unroll
                    for (int c = 0; c < C; ++c) { self[q][c] = Tm[(size_t)row * C + (c ^ sw)]; p[q][c] = Tp[(size_t)row * C + (c ^ sw)]; }
                }
#pragma unroll
                for (int q = 0; q < RPT; ++q)
#pragma unroll
                    for (int k = 0; k < K; ++k) {
                        const int sl = (int)(tb_row_entry<KP>(w[q], k) & TB_SLOT_MASK);
#pragma unroll
                        for (int c = 0; c < C; ++c) v[q][k][c] = Tm[(size_t)sl * C + (c ^ sw)];
                    }
#pragma unroll
                for (int q = 0; q < RPT; ++q) {
                    const int row = tid + q * TB_CONSUMERS;
#pragma unroll
                    for (int c = 0; c < C; ++c) {
                        c128 acc = make_double2(eps[q] * self[q][c].x, eps[q] * self[q][c].y);
#pragma unroll
                        for (int k = 0; k < K; ++k) cfma_r(acc, a.dict[tb_row_entry<KP>(w[q], k) >> 12], v[q][k][c]);
                        t1[q][c] = make_double2(fma(2.0, acc.x, -p[q][c].x), fma(2.0, acc.y, -p[q][c].y));
                    }
                    if (row < nown) {
#pragma unroll
                        for (int c = 0; c < C; ++c) {
                            if (NSTEP == 2) Tp[(size_t)row * C + (c ^ sw)] = t1[q][c];
                            tb_store_keep(next1_p + (site0 + row) * C + (c ^ sw), t1[q][c], keep);
                        }
                        if (MODE == MODE_MOM2) {
                            // (C = 2: register slot c holds column c ^ sw; the per-column sums are un-swizzled at the end)
#pragma unroll
                            for (int c = 0; c < C; ++c) {
                                tb_cdot(s1[c], self[q][c], t1[q][c]);                                        // <T_m|T_{m+1}>
                                s2[c].x = fma(t1[q][c].x, t1[q][c].x, fma(t1[q][c].y, t1[q][c].y, s2[c].x));   // |T_{m+1}|^2
                            }
                        } else {
                            const c128 sL = sw ? self[q][C - 1] : self[q][0];
                            const c128 tL = sw ? t1[q][C - 1] : t1[q][0], tR = sw ? t1[q][0] : t1[q][C - 1];
                            tb_cdot(s1[0], sL, tR);                                                          // <T_m L|T_{m+1} R>
                            tb_cdot(s2[0], tL, tR);                                                          // <T_{m+1} L|T_{m+1} R>
                        }
                    }
                }
            }
            if (NSTEP == 2) {
                // ---- step 1 on the H1 rows (redundant with the neighbouring tiles), in place over T_{m-1} ----
                for (int row = CS + tid; row < CS + n1; row += TB_CONSUMERS) {
                    uint32_t wr[KP / 2];
                    tb_load_row<KP>(rows_s, row, wr);
                    const double e1 = ONS ? hons_s[row - CS] : 0.0;
#pragma unroll
                    for (int c = 0; c < C; ++c) {
                        const int cc = c ^ sw;
                        const c128 sv = Tm[(size_t)row * C + cc], pv = Tp[(size_t)row * C + cc];
                        c128 acc = make_double2(e1 * sv.x, e1 * sv.y);
#pragma unroll
                        for (int k = 0; k < K; ++k) {
                            const uint32_t e = tb_row_entry<KP>(wr, k);
                            cfma_r(acc, a.dict[e >> 12], Tm[(size_t)(e & TB_SLOT_MASK) * C + cc]);
                        }
                        Tp[(size_t)row * C + cc] = make_double2(fma(2.0, acc.x, -pv.x), fma(2.0, acc.y, -pv.y));
                    }
                }
                asm volatile("bar.sync 1, %0;" ::"n"(TB_CONSUMERS) : "memory");      // T_{m+1} complete on own + H1
                // ---- step 2: T_{m+2} = 2 H~ T_{m+1} - T_m on the own rows (matrix row, T_m, T_{m+1} kept in registers) ----
                c128 v[RPT][K][C];
#pragma unroll
                for (int q = 0; q < RPT; ++q)
#pragma unroll
                    for (int k = 0; k < K; ++k) {
                        const int sl = (int)(tb_row_entry<KP>(w[q], k) & TB_SLOT_MASK);
#pragma unroll
                        for (int c = 0; c < C; ++c) v[q][k][c] = Tp[(size_t)sl * C + (c ^ sw)];
                    }
#pragma unroll
                for (int q = 0; q < RPT; ++q) {
                    const int row = tid + q * TB_CONSUMERS;
                    c128 t2[C];
#pragma unroll
                    for (int c = 0; c < C; ++c) {
                        c128 acc = make_double2(eps[q] * t1[q][c].x, eps[q] * t1[q][c].y);
#pragma unroll
                        for (int k = 0; k < K; ++k) cfma_r(acc, a.dict[tb_row_entry<KP>(w[q], k) >> 12], v[q][k][c]);
                        t2[c] = make_double2(fma(2.0, acc.x, -self[q][c].x), fma(2.0, acc.y, -self[q][c].y));
                    }
                    if (row < nown) {
#pragma unroll
                        for (int c = 0; c < C; ++c) tb_store_keep(next2_p + (site0 + row) * C + (c ^ sw), t2[c], keep);
                        if (MODE == MODE_MOM2) {
#pragma unroll
                            for (int c = 0; c < C; ++c) {
                                tb_cdot(s3[c], t1[q][c], t2[c]);                                             // <T_{m+1}|T_{m+2}>
                                s4[c].x = fma(t2[c].x, t2[c].x, fma(t2[c].y, t2[c].y, s4[c].x));             // |T_{m+2}|^2
                            }
                        } else {
                            const c128 tL = sw ? t1[q][C - 1] : t1[q][0];
                            const c128 uL = sw ? t2[C - 1] : t2[0], uR = sw ? t2[0] : t2[C - 1];
                            tb_cdot(s3[0], tL, uR);                                                          // <T_{m+1} L|T_{m+2} R>
                            tb_cdot(s4[0], uL, uR);                                                          // <T_{m+2} L|T_{m+2} R>
                        }
                    }
                }
            }
            __syncwarp();
            if ((tid & 31) == 0) sg_mbar_arrive(em0 + 8 * s);
        }
    }
    if (MODE == MODE_MOM2 && C == 2 && sw) {         // register slot c held column c ^ 1 in these lanes
        c128 x;
        x = s1[0]; s1[0] = s1[PR - 1]; s1[PR - 1] = x;
        x = s2[0]; s2[0] = s2[PR - 1]; s2[PR - 1] = x;
        x = s3[0]; s3[0] = s3[PR - 1]; s3[PR - 1] = x;
        x = s4[0]; s4[0] = s4[PR - 1]; s4[PR - 1] = x;
    }
#pragma unroll
    for (int c = 0; c < PR; ++c) {
        const int64_t slot = ((int64_t)bl * a.nplanes + plane) * PR + c;      // [cpp][nplanes * PR]: plane-major columns
        c128 tot = tb_block_sum(s1[c], red);
        if (tid == 0) a.p1[slot] = tot;
        tot = tb_block_sum(s2[c], red);
        if (tid == 0) a.p2[slot] = tot;
        if (NSTEP == 2) {
            tot = tb_block_sum(s3[c], red);
            if (tid == 0) a.p3[slot] = tot;
            tot = tb_block_sum(s4[c], red);
            if (tid == 0) a.p4[slot] = tot;
        }
    }
}
