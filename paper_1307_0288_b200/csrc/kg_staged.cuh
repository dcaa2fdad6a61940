// kg_staged.cuh — the bandwidth-tuned form of the hot kernels (sm_100a): the fused Chebyshev
// step  T_{m+1} = 2 H~ T_m - T_{m-1}  (eq 38; Alg. 5 l.6 P:363) with, folded into the
// same pass, the moment inner product <phi_L|T_{m+1}> (Alg. 5 l.7 P:365, eq 46), or the
// series accumulation out += c_{m+1} T_{m+1} (Alg. 6 l.6 P:385, eq 36), or the commutator
// recursion of eq 39 (Alg. 7) on the (a, d) pair with both accumulations (eq 44).
//
// Same arithmetic as kg_step_kernel<MODE_MOM / MODE_EVO / MODE_PAIR> (kg_kernels.cuh), steps
// m >= 2 with contiguous vectors; what differs is how the bytes move:
//
//  * every CONTIGUOUS stream of a tile — the tile's own T_m, T_{m-1} and phi_L elements, its
//    neighbour indices and its on-site energies — is fetched by the TMA engine with 1-D bulk
//    copies (cp.async.bulk.shared.global, completion on an mbarrier) into a ring of shared-
//    memory stages, issued by one producer lane several tiles ahead of the consumers.  The
//    stream loads therefore cost no registers and no warp stalls; DRAM requests stay in
//    flight independently of occupancy.
//  * the only loads left in the consumer warps are the GATHERS T_m[NL_ik].  Neighbours that
//    lie inside the tile are read from the staged copy of T_m in shared memory; the others
//    (the lattice rows above / below) are 16-byte ld.global.nc hits in L2, brought there by
//    the neighbouring tiles' streams.
//  * the matrix stream is compressed when the hoppings allow it (DICT): a hopping that takes
//    at most 15 distinct non-zero values — one value, -gamma_0/s, in the paper's model, eq 13
//    is stored as a 4-bit dictionary id in the top bits of the int32 neighbour index
//    (n <= 2^28), so a row costs 12 B of indices + 8 B on-site instead of 44 B.  Otherwise the
//    fp64 hoppings are staged like the indices (general Alg. 8 matrix).
//  * persistent grid, tiles interleaved over the CTAs; the sweep direction alternates from
//    one Chebyshev step to the next (`reverse`), so that the tail of step m — the last ~L2-size
//    worth of T_{m+1}, T_m, phi_L and matrix — is what step m+1 touches first and is served
//    from the 126 MB L2 instead of HBM.
//
// Determinism: tile -> CTA -> thread -> element assignment is a pure function of the launch
// shape; per-thread sums run in a fixed order, the block tree is fixed, kg_reduce_partials
// adds the per-CTA partials in CTA order.  Moments are bitwise reproducible run to run.
#pragma once
#include "kg_common.cuh"

#define SG_TILE_E 512          // largest tile, elements (site, vector); row stride ns is a multiple
#define SG_CONSUMERS 256       // consumer threads; + one producer warp
#define SG_THREADS (SG_CONSUMERS + 32)
#define SG_IDX_MASK 0x0FFFFFFF // DICT: neighbour index in bits 0..27, dictionary id in 28..31
#define SG_MAX_STAGES 8

struct StagedArgs {
    const int32_t *idx;    // [K][ns]  DICT: (id << 28) | NL_ik ; else NL_ik
    const double *hop;     // [K][ns]  H_ik / s              (used when !DICT)
    const double *xhop;    // [K][ns]  (X_i - X_m) H_ik / s  (MODE_PAIR)
    const double *onsite;  // [ns]     (H_ii - E0)/s         (used when ONS)
    double dict[16];       // DICT: hopping value per id, dict[0] = 0 (read from the constant bank)
    int64_t n, ns;
    const c128 *cur;       // T_m      [n][R]
    const c128 *prev;      // T_{m-1}  [n][R]
    c128 *next;            // T_{m+1}  [n][R]; may alias prev
    const c128 *aux;       // MODE_MOM: phi_L ; MODE_EVO / MODE_PAIR: the accumulator `out` (read side)
    c128 *partial;         // MODE_MOM: [grid][R] ; MODE_MOM2: <T_m|T_{m+1}> (moment 2m+1)
    c128 *partial2;        // MODE_MOM2: <T_{m+1}|T_{m+1}> (moment 2m+2)
    c128 *out;             // MODE_EVO / MODE_PAIR: out += c1 T_{m+1}
    c128 c1;
    c128 cpre;             // MODE_CLEN: next = c1 aux + cpre (alpha H~ cur) - (use_prev ? prev : 0)
    double alpha;
    int use_prev;
    const c128 *dcur, *dprev, *daux;   // MODE_PAIR d-chain (daux = outd, read side)
    c128 *dnext, *outd;
    int ntiles;
    int reverse;           // sweep the tiles from the last to the first
    int nstages;
};

__device__ __forceinline__ uint32_t sg_smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void sg_mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void sg_mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void sg_mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool sg_mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void sg_mbar_wait(uint32_t bar, uint32_t parity)
{
    while (!sg_mbar_try_wait(bar, parity)) {}
}
// 1-D bulk copy global -> shared through the TMA engine; bytes % 16 == 0, 16-byte aligned ends
__device__ __forceinline__ void sg_bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

// Tile size per mode: the pair recursion stages six vector streams, so its tile is half as long
// to keep >= 2 stages x 3 CTAs per SM in shared memory.
__host__ __device__ constexpr bool sg_is_pair(int mode) { return mode == MODE_PAIR || mode == MODE_PCLEN; }
__host__ __device__ constexpr int sg_tile_e(int mode) { return sg_is_pair(mode) ? 256 : 512; }
__host__ __device__ constexpr int sg_nvec(int mode) { return sg_is_pair(mode) ? 6 : (mode == MODE_MOM2 || mode == MODE_MOMX) ? 2 : 3; }
// bytes of one stage / of the header (host planning and device layout use the same formulas)
__host__ __device__ constexpr int sg_stage_bytes(int R, int K, int mode, bool ons, bool dict)
{
    return (sg_nvec(mode) * sg_tile_e(mode) * 16 + (sg_tile_e(mode) / R) * (4 * K + (ons ? 8 : 0) +
            (sg_is_pair(mode) ? 8 * K : 0) + (dict ? 0 : 8 * K)) + 127) / 128 * 128;
}
// row widths the staged kernels are compiled for (others run kg_step_kernel)
__host__ __device__ constexpr bool sg_k_supported(int K) { return K == 2 || K == 3 || K == 4 || K == 6 || K == 9; }
__host__ __device__ constexpr int sg_header_bytes(int R)
{
    return (2 * SG_MAX_STAGES * 8 + 16 * 8 + 32 * R * 16 + 127) / 128 * 128;
}

// byte offsets inside one stage.  Vector slots: 0 self (T_m of the tile), 1 prev (T_{m-1}),
// 2 aux (phi_L for moments, the series accumulator for evolve / pair), 3-5 the same for the
// d-chain of the pair recursion.
template <int R, int K, int MODE, bool ONS, bool DICT>
struct SgLayout {
    static constexpr int TE = sg_tile_e(MODE);
    static constexpr int CS = TE / R;                        // sites per tile
    static constexpr int VEC = TE * 16;
    static constexpr int OFF_IDX = sg_nvec(MODE) * VEC;
    static constexpr int OFF_ONS = OFF_IDX + K * CS * 4;
    static constexpr int OFF_XHOP = OFF_ONS + (ONS ? CS * 8 : 0);
    static constexpr int OFF_HOP = OFF_XHOP + (sg_is_pair(MODE) ? K * CS * 8 : 0);
    static constexpr int STAGE = sg_stage_bytes(R, K, MODE, ONS, DICT);
    static constexpr int OFF_DICT = 2 * SG_MAX_STAGES * 8;
    static constexpr int OFF_RED = OFF_DICT + 16 * 8;
    static constexpr int HEADER = sg_header_bytes(R);
    static_assert(OFF_HOP + (DICT ? 0 : K * CS * 8) <= STAGE, "stage layout");
};

// MODE_MOM   next = 2 H~ cur - prev ; partial += <phiL|next>            (Alg. 5 l.6-7)
// MODE_MOM2  next = 2 H~ cur - prev ; partial += <cur|next>, partial2 += <next|next>
//            (phi_L = phi_R: moments 2m+1 and 2m+2 from one sweep, see kg_kernels.cuh)
// MODE_MOMX  the batch is [phi_L | phi_R] (R/2 columns each), both halves are advanced;
//            partial += <cur_L|next_R>, partial2 += <next_L|next_R>, rows [grid][R/2]
// MODE_EVO   next = 2 H~ cur - prev ; out += c1 next                     (Alg. 6 l.5-6)
// MODE_CLEN  next = c1 phi + cpre (alpha H~ cur) - prev : Clenshaw's backward recurrence for the
//            series of eq 36, b_m = c_m phi + 2 H~ b_{m+1} - b_{m+2}, U phi = c_0 phi + H~ b_1 - b_2
//            (aux = phi; three read streams and one write instead of evolve's three and two)
// MODE_PCLEN the same for the pair of eq 44: b as above and
//            e_m = c_m psix + 2 H~ e_{m+1} + 2 [X,H~] b_{m+1} - e_{m+2}   (the derivation [X, .] of
//            Clenshaw's recurrence), psix' = c_0 psix + H~ e_1 + [X,H~] b_1 - e_2; daux = psix
// MODE_PAIR  the same on the a-chain, and on the d-chain
//            dnext = 2([X,H~] cur + H~ dcur) - dprev ; outd += c1 dnext  (eq 39, Alg. 7 l.7-8)
template <int R, int K, int MODE, bool ONS, bool DICT>
__global__ void __launch_bounds__(SG_THREADS) kg_staged_kernel(const StagedArgs a)
{
    typedef SgLayout<R, K, MODE, ONS, DICT> L;
    constexpr int CS = L::CS, TE = L::TE, EPT = TE / SG_CONSUMERS;
    constexpr bool PAIR = sg_is_pair(MODE);
    constexpr bool CLEN = MODE == MODE_CLEN || MODE == MODE_PCLEN;
    extern __shared__ __align__(128) unsigned char sg_smem[];
    uint64_t *bars = reinterpret_cast<uint64_t *>(sg_smem);
    c128 *red = reinterpret_cast<c128 *>(sg_smem + L::OFF_RED);
    unsigned char *stages = sg_smem + L::HEADER;

    const int tid = threadIdx.x;
    const int nst = a.nstages;
    const uint32_t full0 = sg_smem_u32(bars), empty0 = sg_smem_u32(bars + SG_MAX_STAGES);
    // Programmatic dependent launch: let the next sweep's CTAs be scheduled as ours drain, and do
    // our own set-up (barrier init) while the previous sweep is still finishing; nothing that the
    // previous kernel wrote is touched before griddepcontrol.wait.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (tid == 0) {
        for (int s = 0; s < nst; ++s) {
            sg_mbar_init(full0 + 8 * s, 1);
            sg_mbar_init(empty0 + 8 * s, SG_CONSUMERS / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    asm volatile("griddepcontrol.wait;" ::: "memory");

    const int64_t total = a.n * R;
    const int my_tiles = ((int)blockIdx.x < a.ntiles) ? (a.ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
    c128 sum = make_double2(0.0, 0.0), sum2 = make_double2(0.0, 0.0);

    if (tid >= SG_CONSUMERS) {
        // ---------------- producer warp: one lane feeds the ring ----------------
        if (tid == SG_CONSUMERS) {
            int s = 0;
            uint32_t ph = 0;
            for (int j = 0; j < my_tiles; ++j, ++s) {
                if (s == nst) { s = 0; ph ^= 1u; }
                int t = (int)blockIdx.x + j * (int)gridDim.x;
                if (a.reverse) t = a.ntiles - 1 - t;
                const int64_t site0 = (int64_t)t * CS, e0 = site0 * R;
                const int64_t rem = total - e0;
                const uint32_t vbytes = (uint32_t)(rem < TE ? rem : TE) * 16u;
                const uint32_t full = full0 + 8 * s;
                while (!sg_mbar_try_wait(empty0 + 8 * s, ph ^ 1u)) __nanosleep(64);   // ring full: back off
                const uint32_t sb = sg_smem_u32(stages + (size_t)s * L::STAGE);
                uint32_t tx = (uint32_t)sg_nvec(MODE) * vbytes + (uint32_t)K * CS * 4u;
                if (ONS) tx += CS * 8u;
                if (PAIR) tx += (uint32_t)K * CS * 8u;
                if (!DICT) tx += (uint32_t)K * CS * 8u;
                sg_mbar_expect_tx(full, tx);
                sg_bulk_g2s(sb + 0 * L::VEC, a.cur + e0, vbytes, full);
                sg_bulk_g2s(sb + 1 * L::VEC, a.prev + e0, vbytes, full);
                if (sg_nvec(MODE) > 2) sg_bulk_g2s(sb + 2 * L::VEC, a.aux + e0, vbytes, full);
                if (PAIR) {
                    sg_bulk_g2s(sb + 3 * L::VEC, a.dcur + e0, vbytes, full);
                    sg_bulk_g2s(sb + 4 * L::VEC, a.dprev + e0, vbytes, full);
                    sg_bulk_g2s(sb + 5 * L::VEC, a.daux + e0, vbytes, full);
                }
#pragma unroll
                for (int k = 0; k < K; ++k)
                    sg_bulk_g2s(sb + L::OFF_IDX + k * CS * 4, a.idx + k * a.ns + site0, CS * 4u, full);
                if (ONS) sg_bulk_g2s(sb + L::OFF_ONS, a.onsite + site0, CS * 8u, full);
                if (PAIR) {
#pragma unroll
                    for (int k = 0; k < K; ++k)
                        sg_bulk_g2s(sb + L::OFF_XHOP + k * CS * 8, a.xhop + k * a.ns + site0, CS * 8u, full);
                }
                if (!DICT) {
#pragma unroll
                    for (int k = 0; k < K; ++k)
                        sg_bulk_g2s(sb + L::OFF_HOP + k * CS * 8, a.hop + k * a.ns + site0, CS * 8u, full);
                }
            }
        }
    } else {
        // ---------------- consumers: gathers + arithmetic ----------------
        const int r = tid & (R - 1);
        int s = 0;
        uint32_t ph = 0;
        for (int j = 0; j < my_tiles; ++j, ++s) {
            if (s == nst) { s = 0; ph ^= 1u; }
            int t = (int)blockIdx.x + j * (int)gridDim.x;
            if (a.reverse) t = a.ntiles - 1 - t;
            const int32_t site0 = t * CS;                    // n < 2^31: site indices fit 32 bits
            const int64_t e0 = (int64_t)site0 * R;
            const int64_t rem = total - e0;
            const int ne = (int)(rem < TE ? rem : TE);
            const unsigned char *sb = stages + (size_t)s * L::STAGE;
            const c128 *self_s = reinterpret_cast<const c128 *>(sb + 0 * L::VEC);
            const c128 *prev_s = reinterpret_cast<const c128 *>(sb + 1 * L::VEC);
            const c128 *aux_s = reinterpret_cast<const c128 *>(sb + 2 * L::VEC);
            const c128 *dself_s = reinterpret_cast<const c128 *>(sb + 3 * L::VEC);
            const c128 *dprev_s = reinterpret_cast<const c128 *>(sb + 4 * L::VEC);
            const c128 *daux_s = reinterpret_cast<const c128 *>(sb + 5 * L::VEC);
            const int32_t *idx_s = reinterpret_cast<const int32_t *>(sb + L::OFF_IDX);
            const double *ons_s = reinterpret_cast<const double *>(sb + L::OFF_ONS);
            const double *xhop_s = reinterpret_cast<const double *>(sb + L::OFF_XHOP);
            const double *hop_s = reinterpret_cast<const double *>(sb + L::OFF_HOP);
            sg_mbar_wait(full0 + 8 * s, ph);

            c128 v[EPT][K], dv[PAIR ? EPT : 1][K];
            double hk[EPT][K];
#pragma unroll
            for (int q = 0; q < EPT; ++q) {
                const int le = tid + q * SG_CONSUMERS;
                const int ls = le / R;
#pragma unroll
                for (int k = 0; k < K; ++k) {
                    const int32_t w = idx_s[k * CS + ls];
                    int32_t m;
                    if (DICT) {
                        m = w & SG_IDX_MASK;
                        hk[q][k] = a.dict[(uint32_t)w >> 28];      // constant bank (LDC), not shared memory
                    } else {
                        m = w;
                        hk[q][k] = hop_s[k * CS + ls];
                    }
                    const uint32_t d = (uint32_t)(m - site0);
                    if (d < (uint32_t)CS) {
                        v[q][k] = self_s[d * R + r];
                        if (PAIR) dv[q][k] = dself_s[d * R + r];
                    } else {
                        const int64_t g = (int64_t)m * R + r;
                        v[q][k] = ld_nc(a.cur + g);
                        if (PAIR) dv[q][k] = ld_nc(a.dcur + g);
                    }
                }
            }
#pragma unroll
            for (int q = 0; q < EPT; ++q) {
                const int le = tid + q * SG_CONSUMERS;
                const int ls = le / R;
                c128 acc = make_double2(0.0, 0.0), dacc = make_double2(0.0, 0.0);
                if (ONS) {
                    const double eps = ons_s[ls];
                    const c128 self = self_s[le];
                    acc.x = eps * self.x; acc.y = eps * self.y;
                    if (PAIR) {
                        const c128 dself = dself_s[le];
                        dacc.x = eps * dself.x; dacc.y = eps * dself.y;
                    }
                }
#pragma unroll
                for (int k = 0; k < K; ++k) {
                    cfma_r(acc, hk[q][k], v[q][k]);
                    if (PAIR) {
                        cfma_r(dacc, xhop_s[k * CS + ls], v[q][k]);     // [X,H~] a_m
                        cfma_r(dacc, hk[q][k], dv[q][k]);               // H~ d_m
                    }
                }
                c128 tl = make_double2(0.0, 0.0);
                if (MODE == MODE_MOMX) {
                    // the left-chain partner (column r - R/2 of the same site) is lane - R/2;
                    // every lane of the warp takes part (tail lanes carry unused values)
                    const c128 p = prev_s[le];
                    const int src = (tid - (R > 1 ? R / 2 : 1)) & 31;
                    tl.x = __shfl_sync(0xffffffffu, fma(2.0, acc.x, -p.x), src);
                    tl.y = __shfl_sync(0xffffffffu, fma(2.0, acc.y, -p.y), src);
                }
                if (le < ne) {
                    const c128 p = prev_s[le];
                    c128 tt;
                    if (CLEN) {
                        const c128 g = cmul(a.cpre, make_double2(a.alpha * acc.x, a.alpha * acc.y));
                        const c128 ca = cmul(a.c1, aux_s[le]);
                        tt = make_double2(ca.x + g.x, ca.y + g.y);
                        if (a.use_prev) { tt.x -= p.x; tt.y -= p.y; }
                    } else {
                        tt = make_double2(fma(2.0, acc.x, -p.x), fma(2.0, acc.y, -p.y));
                    }
                    a.next[e0 + le] = tt;
                    if (CLEN) {
                    } else if (MODE == MODE_MOM) {
                        const c128 Lv = aux_s[le];
                        sum.x = fma(Lv.x, tt.x, fma(Lv.y, tt.y, sum.x));      // conj(L) * t
                        sum.y = fma(Lv.x, tt.y, fma(-Lv.y, tt.x, sum.y));
                    } else if (MODE == MODE_MOMX) {
                        constexpr int RH = R > 1 ? R / 2 : 1;
                        if (r >= RH) {
                            const c128 sl = self_s[le - RH];
                            sum.x = fma(sl.x, tt.x, fma(sl.y, tt.y, sum.x));      // conj(T_m L) * T_{m+1} R
                            sum.y = fma(sl.x, tt.y, fma(-sl.y, tt.x, sum.y));
                            sum2.x = fma(tl.x, tt.x, fma(tl.y, tt.y, sum2.x));    // conj(T_{m+1} L) * T_{m+1} R
                            sum2.y = fma(tl.x, tt.y, fma(-tl.y, tt.x, sum2.y));
                        }
                    } else if (MODE == MODE_MOM2) {
                        const c128 sv = self_s[le];
                        sum.x = fma(sv.x, tt.x, fma(sv.y, tt.y, sum.x));      // conj(T_m) * T_{m+1}
                        sum.y = fma(sv.x, tt.y, fma(-sv.y, tt.x, sum.y));
                        sum2.x = fma(tt.x, tt.x, fma(tt.y, tt.y, sum2.x));    // |T_{m+1}|^2
                    } else {
                        const c128 o = aux_s[le], ct = cmul(a.c1, tt);
                        a.out[e0 + le] = make_double2(o.x + ct.x, o.y + ct.y);
                    }
                    if (MODE == MODE_PCLEN) {
                        const c128 dp = dprev_s[le];
                        const c128 g = cmul(a.cpre, make_double2(a.alpha * dacc.x, a.alpha * dacc.y));
                        const c128 ca = cmul(a.c1, daux_s[le]);
                        c128 dt = make_double2(ca.x + g.x, ca.y + g.y);
                        if (a.use_prev) { dt.x -= dp.x; dt.y -= dp.y; }
                        a.dnext[e0 + le] = dt;
                    } else if (PAIR) {
                        const c128 dp = dprev_s[le];
                        const c128 dt = make_double2(fma(2.0, dacc.x, -dp.x), fma(2.0, dacc.y, -dp.y));
                        a.dnext[e0 + le] = dt;
                        const c128 o = daux_s[le], ct = cmul(a.c1, dt);
                        a.outd[e0 + le] = make_double2(o.x + ct.x, o.y + ct.y);
                    }
                }
            }
            __syncwarp();
            if ((tid & 31) == 0) sg_mbar_arrive(empty0 + 8 * s);
        }
    }
    if (MODE == MODE_MOM || MODE == MODE_MOM2 || MODE == MODE_MOMX) {
        // block total per column (the producer warp adds zeros); MODE_MOMX keeps the right-chain
        // columns only: partial rows are [grid][R/2]
        constexpr int RH = (MODE == MODE_MOMX && R > 1) ? R / 2 : 0;
        constexpr int PR = R - RH;
        const bool writer = tid >= RH && tid < R;
        const int64_t slot = (int64_t)blockIdx.x * PR + (tid - RH);
        c128 tot = block_reduce_per_r<R>(sum, red);
        if (writer) a.partial[slot] = tot;
        if (MODE != MODE_MOM) {
            c128 tot2 = block_reduce_per_r<R>(sum2, red);
            if (writer) a.partial2[slot] = tot2;
        }
    }
}

