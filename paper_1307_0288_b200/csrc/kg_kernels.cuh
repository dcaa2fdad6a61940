// kg_kernels.cuh — device kernels of libkg (sm_100a) compiled into kg.cu: the one-thread-per-
// element recursion kernel family, reductions, create-time kernels, post-processing.
// (Shared types and helpers: kg_common.cuh; the TMA-staged kernels: kg_staged.cuh.)
#pragma once
#include "kg_common.cuh"

// R = 16 or 32 lanes would leave nothing to shuffle for R = 32; supported R: 1, 2, 4, 8, 16.
template <int R, int MODE, bool FIRST, bool ONS, int KMAX>
__global__ void __launch_bounds__(256) kg_step_kernel(const StepArgs a)
{
    const int64_t total = a.n * R;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int r = threadIdx.x & (R - 1);
    const int kmax = KMAX > 0 ? KMAX : a.kmax;

    c128 sum = make_double2(0.0, 0.0), sum0 = make_double2(0.0, 0.0), sum2 = make_double2(0.0, 0.0);

    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += stride) {
        const int64_t i = e / R;   // R is a power of two: a shift
        c128 acc = make_double2(0.0, 0.0);
        c128 dacc = make_double2(0.0, 0.0);
        c128 self = make_double2(0.0, 0.0), dself = make_double2(0.0, 0.0);
        if (MODE != MODE_VEL && (ONS || FIRST || MODE == MODE_MOM2 || MODE == MODE_MOMX)) {
            self = ld_nc(a.cur + i * a.ld_cur + r);
            if (MODE == MODE_PAIR) dself = ld_nc(a.dcur + i * a.ld_dcur + r);
        }
        if (MODE != MODE_VEL && ONS) {
            const double eps = __ldg(a.onsite + i);
            acc.x = eps * self.x; acc.y = eps * self.y;
            if (MODE == MODE_PAIR) { dacc.x = eps * dself.x; dacc.y = eps * dself.y; }
        }
#pragma unroll
        for (int k = 0; k < kmax; ++k) {
            const int64_t m = __ldg(a.nl + k * a.ns + i);
            if (MODE == MODE_VEL) {
                const double w = __ldg(a.xhop + k * a.ns + i);
                cfma_r(acc, w, ld_nc(a.cur + m * a.ld_cur + r));
            } else {
                const double h = __ldg(a.hop + k * a.ns + i);
                const c128 v = ld_nc(a.cur + m * a.ld_cur + r);
                cfma_r(acc, h, v);
                if (MODE == MODE_PAIR) {
                    const double w = __ldg(a.xhop + k * a.ns + i);
                    cfma_r(dacc, w, v);                                   // [X,H~] a_m
                    cfma_r(dacc, h, ld_nc(a.dcur + m * a.ld_dcur + r));   // H~ d_m
                }
            }
        }
        if (MODE == MODE_VEL) {
            // V = -(i s/hbar)[X,H~]:  -i (x + i y) = y - i x
            a.vout[i * a.ld_vout + r] = make_double2(a.vscale * acc.y, -a.vscale * acc.x);
            continue;
        }
        c128 t;
        if (FIRST) {
            t = acc;
        } else {
            const c128 p = a.prev[i * a.ld_prev + r];
            t = make_double2(fma(a.alpha, acc.x, -p.x), fma(a.alpha, acc.y, -p.y));
        }
        a.next[e] = t;
        if (MODE == MODE_MOM) {
            const c128 L = ld_nc(a.phiL + i * a.ld_L + r);
            sum.x = fma(L.x, t.x, fma(L.y, t.y, sum.x));      // conj(L) * t
            sum.y = fma(L.x, t.y, fma(-L.y, t.x, sum.y));
            if (FIRST) {
                sum0.x = fma(L.x, self.x, fma(L.y, self.y, sum0.x));
                sum0.y = fma(L.x, self.y, fma(-L.y, self.x, sum0.y));
            }
        }
        if (MODE == MODE_MOM2) {
            sum.x = fma(self.x, t.x, fma(self.y, t.y, sum.x));        // conj(T_m) * T_{m+1}
            sum.y = fma(self.x, t.y, fma(-self.y, t.x, sum.y));
            sum2.x = fma(t.x, t.x, fma(t.y, t.y, sum2.x));            // |T_{m+1}|^2
            if (FIRST) sum0.x = fma(self.x, self.x, fma(self.y, self.y, sum0.x));
        }
        if (MODE == MODE_MOMX) {
            // column r >= R/2 (right chain) pairs with column r - R/2 (left chain) of the same
            // site, held by lane - R/2 of the same warp
            constexpr int RH = R > 1 ? R / 2 : 1;
            const unsigned mask = __activemask();
            const int src = (threadIdx.x - RH) & 31;
            c128 tl, sl;
            tl.x = __shfl_sync(mask, t.x, src); tl.y = __shfl_sync(mask, t.y, src);
            sl.x = __shfl_sync(mask, self.x, src); sl.y = __shfl_sync(mask, self.y, src);
            if (r >= RH) {
                sum.x = fma(sl.x, t.x, fma(sl.y, t.y, sum.x));        // conj(T_m L) * T_{m+1} R
                sum.y = fma(sl.x, t.y, fma(-sl.y, t.x, sum.y));
                sum2.x = fma(tl.x, t.x, fma(tl.y, t.y, sum2.x));      // conj(T_{m+1} L) * T_{m+1} R
                sum2.y = fma(tl.x, t.y, fma(-tl.y, t.x, sum2.y));
                if (FIRST) {
                    sum0.x = fma(sl.x, self.x, fma(sl.y, self.y, sum0.x));
                    sum0.y = fma(sl.x, self.y, fma(-sl.y, self.x, sum0.y));
                }
            }
        }
        if (MODE == MODE_EVO || MODE == MODE_PAIR) {
            c128 o;
            if (FIRST) o = cmul(a.c0, self); else o = a.out[e];
            const c128 ct = cmul(a.c1, t);
            a.out[e] = make_double2(o.x + ct.x, o.y + ct.y);
        }
        if (MODE == MODE_PAIR) {
            c128 dt;
            if (FIRST) {
                dt = dacc;
            } else {
                const c128 p = a.dprev[i * a.ld_dprev + r];
                dt = make_double2(fma(a.alpha, dacc.x, -p.x), fma(a.alpha, dacc.y, -p.y));
            }
            a.dnext[e] = dt;
            c128 o;
            if (FIRST) o = cmul(a.c0, dself); else o = a.outd[e];
            const c128 ct = cmul(a.c1, dt);
            a.outd[e] = make_double2(o.x + ct.x, o.y + ct.y);
        }
    }

    if (MODE == MODE_MOM || MODE == MODE_MOM2 || MODE == MODE_MOMX) {
        __shared__ c128 red[32 * R];
        // MODE_MOMX: only the right-chain columns carry sums; partial rows are [grid][R/2]
        constexpr int RH = (MODE == MODE_MOMX && R > 1) ? R / 2 : 0;
        constexpr int PR = R - RH;
        const bool writer = (int)threadIdx.x >= RH && (int)threadIdx.x < R;
        const int64_t slot = (int64_t)blockIdx.x * PR + ((int)threadIdx.x - RH);
        c128 tot = block_reduce_per_r<R>(sum, red);
        if (writer) a.partial[slot] = tot;
        if (MODE == MODE_MOM2 || MODE == MODE_MOMX) {
            c128 tot2 = block_reduce_per_r<R>(sum2, red);
            if (writer) a.partial2[slot] = tot2;
        }
        if (FIRST) {
            c128 tot0 = block_reduce_per_r<R>(sum0, red);
            if (writer) a.partial0[slot] = tot0;
        }
    }
}

// Fixed-order final sum of the per-block partials (a8): one warp per (moment m, vector r).
// partials [M][B][R]  ->  mu[r*mu_rstride + m]
// `doubling`: rows m >= 2 hold <T_a|T_b> with a + b = m, |a - b| = m & 1, and
// mu_m = 2 <T_a|T_b> - mu_{m&1}  (2 T_a T_b = T_{a+b} + T_{|a-b|}).
__global__ void kg_reduce_partials(const c128 *__restrict__ partials, int M, int B, int R,
                                   c128 *__restrict__ mu, int64_t mu_rstride, int doubling)
{
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (warp >= M * R) return;
    const int m = warp / R, r = warp % R;
    const c128 *p = partials + (int64_t)m * B * R + r;
    double sx = 0.0, sy = 0.0;
    for (int b = lane; b < B; b += 32) {
        const c128 v = p[(int64_t)b * R];
        sx += v.x; sy += v.y;
    }
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        sx += __shfl_xor_sync(0xffffffffu, sx, off);
        sy += __shfl_xor_sync(0xffffffffu, sy, off);
    }
    if (doubling && m >= 2) {
        const c128 *p0 = partials + (int64_t)(m & 1) * B * R + r;
        double bx = 0.0, by = 0.0;
        for (int b = lane; b < B; b += 32) {
            const c128 v = p0[(int64_t)b * R];
            bx += v.x; by += v.y;
        }
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) {
            bx += __shfl_xor_sync(0xffffffffu, bx, off);
            by += __shfl_xor_sync(0xffffffffu, by, off);
        }
        sx = 2.0 * sx - bx; sy = 2.0 * sy - by;
    }
    if (lane == 0) mu[(int64_t)r * mu_rstride + m] = make_double2(sx, sy);
}

// dst[i*ld_dst + c] = src[i*ld_src + c], c < ncols (column-block copy between [n][ld] layouts)
__global__ void kg_copy_cols(const c128 *__restrict__ src, int ld_src, c128 *__restrict__ dst,
                             int ld_dst, int ncols, int64_t n)
{
    const int64_t total = n * ncols;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = e / ncols;
        const int c = (int)(e - i * ncols);
        dst[i * ld_dst + c] = src[i * ld_src + c];
    }
}

// ---------------------------------------------------------------------------------------
// create: validate + scale (a1).  flags[0] bit0: index out of range, bit1: nn out of range,
// bit2: non-finite value, bit3: asymmetric H.  gersh[0] = max_i (|H_ii - E0| + sum_k |H_ik|)
// as an ordered-int encoded double (all values >= 0 so the bit pattern is monotone).
// ---------------------------------------------------------------------------------------
__global__ void kg_build_matrix(int64_t n, int64_t ns, int kmax, const int32_t *__restrict__ nn,
                                const int32_t *__restrict__ nl_in, const double *__restrict__ hop_in,
                                const double *__restrict__ onsite_in, const double *__restrict__ x,
                                double period, double e0, double s, const int32_t *__restrict__ perm,
                                const int32_t *__restrict__ iperm, int32_t *__restrict__ nl,
                                double *__restrict__ hop, double *__restrict__ xhop,
                                double *__restrict__ onsite, unsigned int *flags,
                                unsigned long long *gersh)
{
    // perm / iperm (may be NULL): internal row i is the caller's row perm[i]; the caller's site m is
    // internal site iperm[m] (site re-ordering, kg_partition.h)
    unsigned int bad = 0;
    double gmax = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < ns;
         i += (int64_t)gridDim.x * blockDim.x) {
        if (i >= n) {   // padding rows of the stride
            for (int k = 0; k < kmax; ++k) { nl[k * ns + i] = 0; hop[k * ns + i] = 0.0; xhop[k * ns + i] = 0.0; }
            onsite[i] = 0.0;
            continue;
        }
        const int64_t io = perm ? perm[i] : i;              // the caller's index of this row
        int cnt = nn[io];
        if (cnt < 0 || cnt > kmax) { bad |= 2u; cnt = 0; }
        const double xi = x[io];
        if (!isfinite(xi)) bad |= 4u;
        const double eps = onsite_in ? onsite_in[io] : 0.0;
        if (!isfinite(eps)) bad |= 4u;
        double g = fabs(eps - e0);
        onsite[i] = (eps - e0) / s;
        for (int k = 0; k < kmax; ++k) {
            int32_t m = (int32_t)i;
            double h = 0.0, w = 0.0;
            if (k < cnt) {
                int32_t mo = nl_in[k * n + io];
                h = hop_in[k * n + io];
                if (mo < 0 || mo >= n) { bad |= 1u; mo = (int32_t)io; h = 0.0; }
                if (!isfinite(h)) { bad |= 4u; h = 0.0; }
                double d = x[mo] - xi;                      // Delta = X_m - X_i, minimum image
                if (period > 0.0) {
                    if (d > 0.5 * period) d -= period;
                    if (d < -0.5 * period) d += period;
                }
                w = (-d) * h / s;                           // (X_i - X_m) H_im / s
                g += fabs(h);
                if (mo != io) {                             // symmetry: H_mi must equal H_im
                    bool found = false;
                    int cm = nn[mo];
                    if (cm < 0 || cm > kmax) cm = 0;
                    for (int q = 0; q < cm; ++q)
                        if (nl_in[q * n + mo] == (int32_t)io && hop_in[q * n + mo] == h) found = true;
                    if (!found) bad |= 8u;
                } else {
                    bad |= 8u;                              // diagonal belongs in onsite_eV
                }
                m = iperm ? iperm[mo] : mo;
            }
            nl[k * ns + i] = m;
            hop[k * ns + i] = h / s;
            xhop[k * ns + i] = w;
        }
        gmax = fmax(gmax, g);
    }
    if (bad) atomicOr(flags, bad);
    atomicMax(gersh, (unsigned long long)__double_as_longlong(gmax));
}

// flag |= 1 if any of the `count` doubles is NaN or Inf (KG_OPT_CHECK_INPUT)
__global__ void kg_check_finite(const double *__restrict__ v, int64_t count, unsigned int *flag)
{
    bool bad = false;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < count; e += (int64_t)gridDim.x * blockDim.x)
        bad |= !isfinite(v[e]);
    if (bad) atomicOr(flag, 1u);
}

// dst[i*R + r] = src[map[i]*R + r]: caller order -> internal order with map = perm, and back with
// map = iperm (one thread per element, coalesced writes, 16-byte gathers)
__global__ void kg_permute_rows(const c128 *__restrict__ src, c128 *__restrict__ dst,
                                const int32_t *__restrict__ map, int64_t n, int R)
{
    const int64_t total = n * R;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = e / R;
        const int r = (int)(e - i * R);
        dst[e] = src[(int64_t)map[i] * R + r];
    }
}

// CSR -> k-major list (rows become columns of the ELL slabs)
__global__ void kg_csr_to_ell(int64_t n, const int64_t *__restrict__ rowptr,
                              const int32_t *__restrict__ col, const double *__restrict__ val,
                              int kmax, int32_t *__restrict__ nn, int32_t *__restrict__ nl,
                              double *__restrict__ hop)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t b = rowptr[i], e = rowptr[i + 1];
        int cnt = (int)(e - b);
        if (cnt < 0) cnt = -1;           // flagged as bad nn by kg_build_matrix
        if (cnt > kmax) cnt = kmax + 1;
        nn[i] = cnt;
        for (int k = 0; k < kmax; ++k) {
            const bool ok = cnt >= 0 && k < cnt && k < kmax;
            nl[(int64_t)k * n + i] = ok ? col[b + k] : (int32_t)i;
            hop[(int64_t)k * n + i] = ok ? val[b + k] : 0.0;
        }
    }
}

__global__ void kg_csr_max_row(int64_t n, const int64_t *__restrict__ rowptr, int *maxrow, unsigned int *flags)
{
    int mx = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t c = rowptr[i + 1] - rowptr[i];
        if (c < 0 || c > 32) atomicOr(flags, 2u);
        else mx = max(mx, (int)c);
    }
    atomicMax(maxrow, mx);
}

// ---------------------------------------------------------------------------------------
// KPM reconstruction (eqs 29-31, Jackson damping eq 35).
// w[m] = g_m (2 - delta_m0),  g_m = (1 - m a) cos(pi m a) + a sin(pi m a) cot(pi a), a = 1/(M+1)
// ---------------------------------------------------------------------------------------
__global__ void kg_kpm_weights(int M, int jackson, double *__restrict__ w)
{
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= M) return;
    double g = 1.0;
    if (jackson) {
        const double a = 1.0 / (M + 1.0);
        double sn, cs, sa, ca;
        sincospi(m * a, &sn, &cs);
        sincospi(a, &sa, &ca);
        g = (1.0 - m * a) * cs + a * sn * (ca / sa);
    }
    w[m] = (m == 0 ? 1.0 : 2.0) * g;
}

// f[row][j] = 1/(pi s sqrt(1 - x_j^2)) sum_m w[m] T_m(x_j) Re mu[row][m],  x_j = (E_j - E0)/s,
// T_m by the three-term recurrence; one thread per (row, energy).
__global__ void kg_kpm_reconstruct_kernel(const c128 *__restrict__ mu, int64_t rows, int M,
                                          const double *__restrict__ w, double e0, double s,
                                          const double *__restrict__ energies, int ne,
                                          double *__restrict__ f)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t row = blockIdx.y;
    if (j >= ne || row >= rows) return;
    const double x = (energies[j] - e0) / s;
    const c128 *mr = mu + row * (int64_t)M;
    double t0 = 1.0, t1 = x;
    double sum = w[0] * mr[0].x, comp = 0.0;           // Kahan-compensated
    for (int m = 1; m < M; ++m) {
        const double term = w[m] * t1 * mr[m].x - comp;
        const double ns = sum + term;
        comp = (ns - sum) - term;
        sum = ns;
        const double t2 = fma(2.0 * x, t1, -t0);
        t0 = t1; t1 = t2;
    }
    // outside (-1, 1) the reconstruction is undefined: NaN (a device grid is not validated on the host)
    f[row * (int64_t)ne + j] = fabs(x) < 1.0 ? sum / (3.14159265358979323846 * s * sqrt(1.0 - x * x))
                                             : __longlong_as_double(0x7ff8000000000000LL);
}

// ---------------------------------------------------------------------------------------
// Running conductivities (eqs 6, 9, 11 P:61-78) and ballistic length / conductance (eqs 50-51
// P:496-501) from reconstructed rho~(E_j), rho~C_vv(E_j,t_k), rho~DX2(E_j,t_k); one thread per
// energy, time loop in order.  Trapezoid integral; central differences, second-order one-sided
// at the two ends (reading g14).  Units of e^2/h: pref = 2 pi hbar * dens.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ double kg_ddt(const double *f, int k, int nt, int ne, int j, double dt)
{
    if (nt < 1) return 0.0;
    if (nt == 1) return (f[ne + j] - f[j]) / dt;
    if (k == 0) return (-3.0 * f[j] + 4.0 * f[ne + j] - f[2 * ne + j]) / (2.0 * dt);
    if (k == nt)
        return (3.0 * f[(int64_t)nt * ne + j] - 4.0 * f[(int64_t)(nt - 1) * ne + j] + f[(int64_t)(nt - 2) * ne + j]) / (2.0 * dt);
    return (f[(int64_t)(k + 1) * ne + j] - f[(int64_t)(k - 1) * ne + j]) / (2.0 * dt);
}

__global__ void kg_transport_kernel(int nt, int ne, double dt, double pref, double width,
                                    const double *__restrict__ rho, const double *__restrict__ fvac,
                                    const double *__restrict__ fmsd, double *sigma_gk, double *sigma_e1,
                                    double *sigma_e2, double *length_nm, double *conductance)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= ne) return;
    double integral = 0.0, comp = 0.0;
    for (int k = 0; k <= nt; ++k) {
        const int64_t o = (int64_t)k * ne + j;
        if (sigma_gk) {
            if (k > 0) {
                const double term = 0.5 * (fvac[o - ne] + fvac[o]) * dt - comp;
                const double ns = integral + term;
                comp = (ns - integral) - term;
                integral = ns;
            }
            sigma_gk[o] = pref * integral;
        }
        if (!fmsd) continue;
        const double e1 = pref * 0.5 * kg_ddt(fmsd, k, nt, ne, j, dt);
        if (sigma_e1) sigma_e1[o] = e1;
        if (sigma_e2) sigma_e2[o] = k == 0 ? 0.0 : pref * fmsd[o] / (2.0 * k * dt);
        if (!length_nm && !conductance) continue;
        const double dx2 = fmsd[o] / rho[j];
        const double len = 2.0 * sqrt(dx2 > 0.0 ? dx2 : 0.0);
        if (length_nm) length_nm[o] = len;
        if (conductance) conductance[o] = len > 0.0 ? width / len * e1 : 0.0;
    }
}

// ---------------------------------------------------------------------------------------
// Inner product kernel of Alg. 4 (l.2, 5, 10 P:325-341): per-block partial of <a|b> per vector,
// a at a[i*ld_a + r], b at b[i*R + r]; finished by kg_reduce_partials (fixed order).
// ---------------------------------------------------------------------------------------
template <int R>
__global__ void __launch_bounds__(256) kg_dot_kernel(const c128 *__restrict__ a, int ld_a,
                                                      const c128 *__restrict__ b, int64_t n,
                                                      c128 *__restrict__ partial)
{
    __shared__ c128 red[32 * R];
    const int r = threadIdx.x & (R - 1);
    c128 sum = make_double2(0.0, 0.0);
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n * R;
         e += (int64_t)gridDim.x * blockDim.x) {
        const c128 L = ld_nc(a + (e / R) * ld_a + r), v = ld_nc(b + e);
        sum.x = fma(L.x, v.x, fma(L.y, v.y, sum.x));          // conj(a) * b
        sum.y = fma(L.x, v.y, fma(-L.y, v.x, sum.y));
    }
    c128 tot = block_reduce_per_r<R>(sum, red);
    if (threadIdx.x < R) partial[(int64_t)blockIdx.x * R + threadIdx.x] = tot;
}

// FTM reconstruction (eqs 22-24, Hanning window eq 28), per site and spin:
// f[row][j] = dtau/(2 pi hbar) sum_{n=-Nm}^{Nm} w_n Re[e^{i E_j n dtau/hbar} F[row][n+Nm]].
// The phase e^{i n x} is advanced by complex rotation and re-seeded from sincos every 32 terms.
__global__ void kg_ftm_reconstruct_kernel(const c128 *__restrict__ F, int64_t rows, int Nm, int window,
                                          double dtau_over_hbar, const double *__restrict__ energies,
                                          int ne, double *__restrict__ f)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t row = blockIdx.y;
    if (j >= ne || row >= rows) return;
    const double x = energies[j] * dtau_over_hbar;
    const c128 *Fr = F + row * (int64_t)(2 * Nm + 1) + Nm;
    double sx, cx;
    sincos(x, &sx, &cx);
    double sum = Fr[0].x, comp = 0.0;                          // n = 0, w_0 = 1
    double pr = 1.0, pi = 0.0;                                 // e^{i n x}
    for (int n = 1; n <= Nm; ++n) {
        if ((n & 31) == 0) sincos(n * x, &pi, &pr);
        else { const double t = pr * cx - pi * sx; pi = pr * sx + pi * cx; pr = t; }
        double w = 1.0;
        if (window) w = 0.5 * (1.0 + cospi((double)n / (Nm + 1.0)));
        // Re[e^{inx} F_n] + Re[e^{-inx} F_{-n}]
        const c128 fp = Fr[n], fm = Fr[-n];
        const double term = w * ((pr * fp.x - pi * fp.y) + (pr * fm.x + pi * fm.y)) - comp;
        const double ns = sum + term;
        comp = (ns - sum) - term;
        sum = ns;
    }
    f[row * (int64_t)ne + j] = sum * dtau_over_hbar / (2.0 * 3.14159265358979323846);
}

// ---------------------------------------------------------------------------------------
// create: hopping dictionary.  table[0..14] = bit patterns of the distinct non-zero values
// of H_ik/s found so far (EMPTY = all ones, a NaN pattern no finite hopping has).
// ---------------------------------------------------------------------------------------
#define SG_DICT_EMPTY 0xFFFFFFFFFFFFFFFFull

__global__ void kg_dict_collect(const double *__restrict__ hop, int64_t count,
                                unsigned long long *table, unsigned int *overflow)
{
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < count;
         e += (int64_t)gridDim.x * blockDim.x) {
        const double h = hop[e];
        if (h == 0.0) continue;
        const unsigned long long bits = (unsigned long long)__double_as_longlong(h);
        bool found = false;
        for (int sl = 0; sl < 15 && !found; ++sl) {
            unsigned long long c = *((volatile unsigned long long *)table + sl);
            if (c == SG_DICT_EMPTY) {
                const unsigned long long old = atomicCAS(table + sl, SG_DICT_EMPTY, bits);
                c = (old == SG_DICT_EMPTY) ? bits : old;
            }
            found = (c == bits);
        }
        if (!found) atomicOr(overflow, 1u);
    }
}

// idx[e] = (id << 28) | nl[e], id = position of hop[e] in the sorted dictionary (0 for 0.0)
__global__ void kg_dict_pack(const int32_t *__restrict__ nl, const double *__restrict__ hop,
                             int64_t count, const double *__restrict__ dict, int ndict,
                             int32_t *__restrict__ idx)
{
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < count;
         e += (int64_t)gridDim.x * blockDim.x) {
        const double h = hop[e];
        uint32_t id = 0;
        if (h != 0.0)
            for (int q = 1; q < ndict; ++q)
                if (dict[q] == h) id = (uint32_t)q;
        idx[e] = (int32_t)((id << 28) | (uint32_t)nl[e]);
    }
}
