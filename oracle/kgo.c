/*
 * kgo.c — CPU ORACLE for the Chebyshev hot path of arXiv 1307.0288
 * (Fan, Uppstu, Siro, Harju: linear-scaling Kubo-Greenwood on GPUs).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, the smoke check in
 * __graft_entry__.py and the cpu_baseline / --impl reference legs of bench.py may
 * call it.  It shares no code with paper_1307_0288_b200/ (the CUDA path) and
 * neither includes the other.
 *
 * Plain, slow, single-threaded C99: `double complex` state vectors, `long double`
 * accumulators for every inner product.  Every function follows the paper
 * ("P:n" = line n of PAPER.md) in the paper's order and notation; there is no
 * blocking, fusion or reordering.  Readings of silent/garbled passages are the
 * ones listed in DESIGN.md ("Readings", g1..g20 of SURVEY.md section 8c).
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): see DESIGN.md "Oracle pins".
 * No function in this file is "parity unpinned".
 *
 * Data structure (paper D1): neighbour list with per-site count NN_n and
 * indices NL_nk stored k-major: nl[k*n + i]; matrix elements hop[k*n + i] (real,
 * eq 13); entries with k >= nn[i] are ignored.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex kgo_c;

#define KGO_HBAR 0.6582119569 /* eV fs (CODATA 2018), DESIGN.md constants */

/* ------------------------------------------------------------------------- */
/* Counter-based PRNG.              */
/* bits = splitmix64-finaliser applied to a counter built from                */
/* (seed, stream, index); u = (bits >> 11) * 2^-53 in [0,1).                  */
/* The finaliser constants are those of the published SplitMix64 generator.   */
/* ------------------------------------------------------------------------- */
uint64_t kgo_mix64(uint64_t seed, uint64_t stream, uint64_t index)
{
    uint64_t z = (seed + 1u) * 0x9E3779B97F4A7C15ull;
    z ^= (stream + 1u) * 0xD1B54A32D192ED03ull;
    z += index * 0x9E3779B97F4A7C15ull;
    z ^= z >> 30;
    z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27;
    z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    return z;
}

double kgo_uniform(uint64_t seed, uint64_t stream, uint64_t index)
{
    return (double)(kgo_mix64(seed, stream, index) >> 11) * (1.0 / 9007199254740992.0);
}

/* ------------------------------------------------------------------------- */
/* Lattice generator (paper P:91-93 conventions; SURVEY App. A recipe).       */
/* Honeycomb sheet of ncx x ncy rectangular 4-atom cells; cell = sqrt(3)a     */
/* along x (zigzag) by 3a along y (armchair), a = 0.142 nm.            */
/* Site index i = 4*(cy*ncx + cx) + b.                                        */
/* x = (2cx + hx_b) * h, h = sqrt(3)*a/2 ; y = (6cy + hy_b) * (a/2).           */
/* Outputs: x[n], y[n], nn[n], nl[k*n+i] (k<3); unused slots hold i itself.   */
/* ------------------------------------------------------------------------- */
static const int HX[4] = {0, 0, 1, 1};
static const int HY[4] = {0, 2, 3, 5};
/* neighbour table: for basis b, three (dcx, dcy, b') entries, App. A order */
static const int NB[4][3][3] = {
    {{0, 0, 1}, {0, -1, 3}, {-1, -1, 3}},
    {{0, 0, 0}, {0, 0, 2}, {-1, 0, 2}},
    {{0, 0, 3}, {0, 0, 1}, {1, 0, 1}},
    {{0, 0, 2}, {0, 1, 0}, {1, 1, 0}},
};

void kgo_honeycomb(int64_t ncx, int64_t ncy, int periodic_x, int periodic_y, double a_nm,
                   double *x, double *y, int32_t *nn, int32_t *nl)
{
    const int64_t n = 4 * ncx * ncy;
    const double h = sqrt(3.0) * a_nm / 2.0;
    const double q = a_nm / 2.0;
    for (int64_t cy = 0; cy < ncy; ++cy)
        for (int64_t cx = 0; cx < ncx; ++cx)
            for (int b = 0; b < 4; ++b) {
                const int64_t i = 4 * (cy * ncx + cx) + b;
                x[i] = (double)(2 * cx + HX[b]) * h;
                y[i] = (double)(6 * cy + HY[b]) * q;
                int cnt = 0;
                for (int k = 0; k < 3; ++k) {
                    int64_t mx = cx + NB[b][k][0];
                    int64_t my = cy + NB[b][k][1];
                    if (mx < 0 || mx >= ncx) {
                        if (!periodic_x) continue;
                        mx = (mx + ncx) % ncx;
                    }
                    if (my < 0 || my >= ncy) {
                        if (!periodic_y) continue;
                        my = (my + ncy) % ncy;
                    }
                    nl[(int64_t)cnt * n + i] = (int32_t)(4 * (my * ncx + mx) + NB[b][k][2]);
                    ++cnt;
                }
                nn[i] = cnt;
                for (int k = cnt; k < 3; ++k) nl[(int64_t)k * n + i] = (int32_t)i;
            }
}

/* Honeycomb sheet with next-nearest-neighbour hopping ("more complicated tight-binding  */
/* models ... denser Hamiltonian"; the t' term of the standard graphene model): row width 9 — the */
/* three nearest neighbours of kgo_honeycomb in the same order with hopping t, then the six         */
/* second neighbours at distance sqrt(3) a (same sublattice) with hopping t2, in the order          */
/* (+2,0) (-2,0) (+1,+3) (-1,+3) (+1,-3) (-1,-3) of displacements in units (h, a/2).  Offsets wrap   */
/* on periodic axes, otherwise the neighbour is dropped and later ones shift down.  Outputs sized  */
/* for kmax = 9: nl[k*n+i], hop[k*n+i]; unused slots hold i and 0.                                  */
static const int NB2[4][6][3] = {   /* (dcx, dcy, b') for the six second neighbours of basis b */
    {{1, 0, 0}, {-1, 0, 0}, {0, 0, 2}, {-1, 0, 2}, {0, -1, 2}, {-1, -1, 2}},
    {{1, 0, 1}, {-1, 0, 1}, {0, 0, 3}, {-1, 0, 3}, {0, -1, 3}, {-1, -1, 3}},
    {{1, 0, 2}, {-1, 0, 2}, {1, 1, 0}, {0, 1, 0}, {1, 0, 0}, {0, 0, 0}},
    {{1, 0, 3}, {-1, 0, 3}, {1, 1, 1}, {0, 1, 1}, {1, 0, 1}, {0, 0, 1}},
};

void kgo_honeycomb_nnn(int64_t ncx, int64_t ncy, int periodic_x, int periodic_y, double a_nm, double t_eV,
                       double t2_eV, double *x, double *y, int32_t *nn, int32_t *nl, double *hop)
{
    const int64_t n = 4 * ncx * ncy;
    const double h = sqrt(3.0) * a_nm / 2.0;
    const double q = a_nm / 2.0;
    for (int64_t cy = 0; cy < ncy; ++cy)
        for (int64_t cx = 0; cx < ncx; ++cx)
            for (int b = 0; b < 4; ++b) {
                const int64_t i = 4 * (cy * ncx + cx) + b;
                x[i] = (double)(2 * cx + HX[b]) * h;
                y[i] = (double)(6 * cy + HY[b]) * q;
                int cnt = 0;
                for (int k = 0; k < 9; ++k) {
                    const int *e = k < 3 ? NB[b][k] : NB2[b][k - 3];
                    int64_t mx = cx + e[0], my = cy + e[1];
                    if (mx < 0 || mx >= ncx) {
                        if (!periodic_x) continue;
                        mx = (mx + ncx) % ncx;
                    }
                    if (my < 0 || my >= ncy) {
                        if (!periodic_y) continue;
                        my = (my + ncy) % ncy;
                    }
                    nl[(int64_t)cnt * n + i] = (int32_t)(4 * (my * ncx + mx) + e[2]);
                    hop[(int64_t)cnt * n + i] = k < 3 ? t_eV : t2_eV;
                    ++cnt;
                }
                nn[i] = cnt;
                for (int k = cnt; k < 9; ++k) { nl[(int64_t)k * n + i] = (int32_t)i; hop[(int64_t)k * n + i] = 0.0; }
            }
}

/* Vacancies ("removing carbon atoms randomly"; reading g15: delete and  */
/* compact).  The vacant set is the n_vac sites with the smallest (key, index) */
/* pairs, key_j = mix64(seed, stream 0, j).  vacant[j] = 1 if removed.         */
typedef struct { uint64_t key; int64_t idx; } kgo_keyidx;
static int kgo_cmp_keyidx(const void *pa, const void *pb)
{
    const kgo_keyidx *a = (const kgo_keyidx *)pa, *b = (const kgo_keyidx *)pb;
    if (a->key < b->key) return -1;
    if (a->key > b->key) return 1;
    if (a->idx < b->idx) return -1;
    if (a->idx > b->idx) return 1;
    return 0;
}

int kgo_vacancy_mask(int64_t n_full, int64_t n_vac, uint64_t seed, uint8_t *vacant)
{
    kgo_keyidx *ki = (kgo_keyidx *)malloc((size_t)n_full * sizeof(kgo_keyidx));
    if (!ki) return 1;
    for (int64_t j = 0; j < n_full; ++j) {
        ki[j].key = kgo_mix64(seed, 0, (uint64_t)j);
        ki[j].idx = j;
    }
    qsort(ki, (size_t)n_full, sizeof(kgo_keyidx), kgo_cmp_keyidx);
    memset(vacant, 0, (size_t)n_full);
    for (int64_t v = 0; v < n_vac; ++v) vacant[ki[v].idx] = 1;
    free(ki);
    return 0;
}

/* Delete vacant sites and compact: remaining sites keep their order and are   */
/* renumbered; neighbour lists drop vacant neighbours and shift down.          */
/* Returns the number of remaining sites.  Output arrays are sized for n_out   */
/* (= n_full - n_vac, known to the caller); nl_out is k-major with stride      */
/* n_out, unused slots hold the site's own new index.                          */
int64_t kgo_compact(int64_t n_full, const uint8_t *vacant, const double *x, const double *y,
                    const int32_t *nn, const int32_t *nl, int64_t n_out, double *x_out,
                    double *y_out, int32_t *nn_out, int32_t *nl_out)
{
    int64_t *newidx = (int64_t *)malloc((size_t)n_full * sizeof(int64_t));
    if (!newidx) return -1;
    int64_t c = 0;
    for (int64_t j = 0; j < n_full; ++j) newidx[j] = vacant[j] ? -1 : c++;
    if (c != n_out) { free(newidx); return -1; }
    for (int64_t j = 0; j < n_full; ++j) {
        if (vacant[j]) continue;
        const int64_t i = newidx[j];
        x_out[i] = x[j];
        y_out[i] = y[j];
        int cnt = 0;
        for (int k = 0; k < nn[j]; ++k) {
            const int64_t m = nl[(int64_t)k * n_full + j];
            if (vacant[m]) continue;
            nl_out[(int64_t)cnt * n_out + i] = (int32_t)newidx[m];
            ++cnt;
        }
        nn_out[i] = cnt;
        for (int k = cnt; k < 3; ++k) nl_out[(int64_t)k * n_out + i] = (int32_t)i;
    }
    free(newidx);
    return c;
}

/* Zigzag graphene nanoribbon (Fig. 4: "ZGNR 65536 x 16"): N_y zigzag chains   */
/* (P:91-93), periodic along x (the zigzag direction, the transport axis), zigzag edges.  Cut    */
/* from a sheet of ncx x (N_y/2 + 1) cells that is open along y: the sheet's open edges are      */
/* "bearded" (the b0 sites of the bottom cell row and the b3 sites of the top one hang on one    */
/* bond), a zigzag edge is obtained by removing the bottom row's b0 sites and the top row's      */
/* b1, b2, b3 sites — the cut then runs through the vertical bonds, every edge site keeps two    */
/* neighbours, and the N_y chains are {b1,b2} of cell rows 0..N_y/2-1 and {b3 of row c, b0 of    */
/* row c+1}, c = 0..N_y/2-1.  Writes vacant[4 ncx (N_y/2+1)] for kgo_compact; N_y must be even.  */
int kgo_zgnr_mask(int64_t ncx, int64_t n_chains, uint8_t *vacant)
{
    if (n_chains < 2 || (n_chains & 1)) return 1;
    const int64_t ncy = n_chains / 2 + 1;
    for (int64_t cy = 0; cy < ncy; ++cy)
        for (int64_t cx = 0; cx < ncx; ++cx)
            for (int b = 0; b < 4; ++b) {
                const int64_t i = 4 * (cy * ncx + cx) + b;
                vacant[i] = (uint8_t)((cy == 0 && b == 0) || (cy == ncy - 1 && b != 0));
            }
    return 0;
}

/* Anderson on-site energies (BASELINE config 4; reading g17):                 */
/* eps_j = W * (u(seed, stream 1, j) - 0.5).                                   */
void kgo_anderson(int64_t n, double w_eV, uint64_t seed, double *eps)
{
    for (int64_t j = 0; j < n; ++j) eps[j] = w_eV * (kgo_uniform(seed, 1, (uint64_t)j) - 0.5);
}

/* Uniform numbers of the random-phase vector r (stream 16+r); the harness     */
/* turns them into phi_j = exp(2 pi i u_j)/sqrt(N) ONCE and hands the same     */
/* bits to both sides (reading g19).                                           */
void kgo_phase_uniforms(int64_t n, uint64_t seed, int r, double *u)
{
    for (int64_t j = 0; j < n; ++j) u[j] = kgo_uniform(seed, 16 + (uint64_t)r, (uint64_t)j);
}

/* ------------------------------------------------------------------------- */
/* O1. bond displacement Delta_nk = X_m - X_n with minimum image (reading g2). */
/* ------------------------------------------------------------------------- */
static double kgo_bond_dx(double x_self, double x_nbr, double period)
{
    double d = x_nbr - x_self;
    if (period > 0.0) {
        if (d > 0.5 * period) d -= period;
        if (d < -0.5 * period) d += period;
    }
    return d;
}

/* ------------------------------------------------------------------------- */
/* O2. Operators.                                                              */
/* ------------------------------------------------------------------------- */
/* out = H~ in,  H~ = (H - E0)/s  (Alg. 8; scaling P:192).     */
void kgo_apply_h(int64_t n, int kmax, const int32_t *nn, const int32_t *nl, const double *hop,
                 const double *onsite, double e0, double s, const kgo_c *in, kgo_c *out)
{
    (void)kmax;
    for (int64_t i = 0; i < n; ++i) {
        kgo_c temp = ((onsite ? onsite[i] : 0.0) - e0) * in[i];
        for (int k = 0; k < nn[i]; ++k) {
            const int64_t m = nl[(int64_t)k * n + i];
            temp += hop[(int64_t)k * n + i] * in[m];
        }
        out[i] = temp / s;
    }
}

/* out = [X, H~] in:  ([X,H]phi)[n] = sum_m (X_n - X_m) H_nm phi[m]  (eq 41, */
/* eq 15), divided by s (reading g3).                                       */
void kgo_apply_xh(int64_t n, int kmax, const int32_t *nn, const int32_t *nl, const double *hop,
                  const double *x, double period, double s, const kgo_c *in, kgo_c *out)
{
    (void)kmax;
    for (int64_t i = 0; i < n; ++i) {
        kgo_c temp = 0.0;
        for (int k = 0; k < nn[i]; ++k) {
            const int64_t m = nl[(int64_t)k * n + i];
            const double xn_minus_xm = -kgo_bond_dx(x[i], x[m], period);
            temp += xn_minus_xm * hop[(int64_t)k * n + i] * in[m];
        }
        out[i] = temp / s;
    }
}

/* out = V in,  V = (i/hbar)[H, X]:  (V phi)[m] = (i/hbar) sum_n (X_n - X_m) H_mn phi[n] */
/* (eq 15), unscaled H, result in nm/fs.                                          */
void kgo_apply_v(int64_t n, int kmax, const int32_t *nn, const int32_t *nl, const double *hop,
                 const double *x, double period, const kgo_c *in, kgo_c *out)
{
    (void)kmax;
    for (int64_t i = 0; i < n; ++i) {
        kgo_c temp = 0.0;
        for (int k = 0; k < nn[i]; ++k) {
            const int64_t m = nl[(int64_t)k * n + i];
            temp += kgo_bond_dx(x[i], x[m], period) * hop[(int64_t)k * n + i] * in[m];
        }
        out[i] = (I / KGO_HBAR) * temp;
    }
}

/* <a|b> = sum conj(a_i) b_i, long double accumulation. */
static kgo_c kgo_dot(int64_t n, const kgo_c *a, const kgo_c *b)
{
    long double re = 0.0L, im = 0.0L;
    for (int64_t i = 0; i < n; ++i) {
        const long double ar = creal(a[i]), ai = cimag(a[i]);
        const long double br = creal(b[i]), bi = cimag(b[i]);
        re += ar * br + ai * bi;
        im += ar * bi - ai * br;
    }
    return (double)re + I * (double)im;
}

kgo_c kgo_inner(int64_t n, const kgo_c *a, const kgo_c *b) { return kgo_dot(n, a, b); }

/* ------------------------------------------------------------------------- */
/* O3. Chebyshev moments C_n = <phi_L|T_n(H~)|phi_R>, n = 0..M-1               */
/* (Alg. 5, eq 46; pointer rotation as in Alg. 6 l.7, g9).     */
/* ------------------------------------------------------------------------- */
int kgo_moments(int64_t n, int kmax, const int32_t *nn, const int32_t *nl, const double *hop,
                const double *onsite, double e0, double s, const kgo_c *phiL,
                const kgo_c *phiR, int M, kgo_c *mu)
{
    kgo_c *phi0 = (kgo_c *)malloc((size_t)n * sizeof(kgo_c));
    kgo_c *phi1 = (kgo_c *)malloc((size_t)n * sizeof(kgo_c));
    kgo_c *phi2 = (kgo_c *)malloc((size_t)n * sizeof(kgo_c));
    if (!phi0 || !phi1 || !phi2) { free(phi0); free(phi1); free(phi2); return 1; }
    memcpy(phi0, phiR, (size_t)n * sizeof(kgo_c));                 /* l.1 */
    if (M > 0) mu[0] = kgo_dot(n, phiL, phi0);                     /* l.2 */
    kgo_apply_h(n, kmax, nn, nl, hop, onsite, e0, s, phi0, phi1);  /* l.3 */
    if (M > 1) mu[1] = kgo_dot(n, phiL, phi1);                     /* l.4 */
    for (int m = 2; m < M; ++m) {                                  /* l.5 */
        kgo_apply_h(n, kmax, nn, nl, hop, onsite, e0, s, phi1, phi2);
        for (int64_t i = 0; i < n; ++i) phi2[i] = 2.0 * phi2[i] - phi0[i]; /* l.6 */
        mu[m] = kgo_dot(n, phiL, phi2);                            /* l.7 */
        kgo_c *t = phi0; phi0 = phi1; phi1 = phi2; phi2 = t;
    }
    free(phi0); free(phi1); free(phi2);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Bessel coefficients and truncation order (eq 36;        */
/* readings g6, g7): J_m from libm jn(); N_p = 1 + max{m : |J_m(x)| >= eps},   */
/* scanning from above.                                                        */
/* ------------------------------------------------------------------------- */
int kgo_bessel_np(double x, double eps)
{
    int mmax = (int)ceil(fabs(x)) + 200 + (int)ceil(30.0 * cbrt(fabs(x)));
    for (int m = mmax; m >= 0; --m)
        if (fabs(jn(m, x)) >= eps) return m + 1;
    return 1;
}

void kgo_bessel_j(double x, int np, double *j)
{
    for (int m = 0; m < np; ++m) j[m] = jn(m, x);
}

/* (-+ i)^m for U(+-dt): sign = +1 -> (-i)^m, sign = -1 -> (+i)^m. */
static kgo_c kgo_ipow(int sign, int m)
{
    static const kgo_c pm[4] = {1.0, -I, -1.0, I}; /* (-i)^m */
    static const kgo_c pp[4] = {1.0, I, -1.0, -I}; /* (+i)^m */
    return sign > 0 ? pm[m & 3] : pp[m & 3];
}

/* ------------------------------------------------------------------------- */
/* O4. out = U(+-dt) in, U(dt) = exp(-i H dt/hbar)                              */
/* (Alg. 6, eq 36), argument x = s|dt|/hbar,           */
/* global phase exp(-+ i E0 dt/hbar) when E0 != 0 (reading g4).                */
/* dt_fs > 0: U(dt); dt_fs < 0: U(-|dt|) = U^dagger(|dt|).                      */
/* ------------------------------------------------------------------------- */
int kgo_evolve(int64_t n, int kmax, const int32_t *nn, const int32_t *nl, const double *hop,
               const double *onsite, double e0, double s, const kgo_c *in, double dt_fs,
               double eps, kgo_c *out)
{
    const int sign = dt_fs >= 0.0 ? +1 : -1;
    const double xarg = s * fabs(dt_fs) / KGO_HBAR;
    const int np = kgo_bessel_np(xarg, eps);
    kgo_c *phi0 = (kgo_c *)malloc((size_t)n * sizeof(kgo_c));
    kgo_c *phi1 = (kgo_c *)malloc((size_t)n * sizeof(kgo_c));
    kgo_c *phi2 = (kgo_c *)malloc((size_t)n * sizeof(kgo_c));
    if (!phi0 || !phi1 || !phi2) { free(phi0); free(phi1); free(phi2); return 1; }
    memcpy(phi0, in, (size_t)n * sizeof(kgo_c));                          /* l.1 */
    kgo_apply_h(n, kmax, nn, nl, hop, onsite, e0, s, phi0, phi1);         /* l.2 */
    const kgo_c c0 = jn(0, xarg);
    const kgo_c c1 = np > 1 ? 2.0 * kgo_ipow(sign, 1) * jn(1, xarg) : 0.0;
    for (int64_t i = 0; i < n; ++i) out[i] = c0 * phi0[i] + c1 * phi1[i]; /* l.3 */
    for (int m = 2; m < np; ++m) {                                        /* l.4 */
        kgo_apply_h(n, kmax, nn, nl, hop, onsite, e0, s, phi1, phi2);
        for (int64_t i = 0; i < n; ++i) phi2[i] = 2.0 * phi2[i] - phi0[i]; /* l.5 */
        const kgo_c cm = 2.0 * kgo_ipow(sign, m) * jn(m, xarg);
        for (int64_t i = 0; i < n; ++i) out[i] += cm * phi2[i];           /* l.6 */
        kgo_c *t = phi0; phi0 = phi1; phi1 = phi2; phi2 = t;              /* l.7 */
    }
    if (e0 != 0.0) {
        const kgo_c ph = cexp(-I * e0 * dt_fs / KGO_HBAR);
        for (int64_t i = 0; i < n; ++i) out[i] *= ph;
    }
    free(phi0); free(phi1); free(phi2);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O5. out = [X, U(dt)] in, dt > 0 (Alg. 7; eqs 37, 39-41).          */
/* phi^x_0 = 0, phi^x_1 = [X,H~]phi,                                           */
/* phi^x_m = 2[X,H~]phi_{m-1} + 2H~phi^x_{m-1} - phi^x_{m-2}.                  */
/* ------------------------------------------------------------------------- */
int kgo_comm_evolve(int64_t n, int kmax, const int32_t *nn, const int32_t *nl,
                    const double *hop, const double *onsite, const double *x, double period,
                    double e0, double s, const kgo_c *in, double dt_fs, double eps, kgo_c *out)
{
    if (dt_fs <= 0.0) return 2;
    const double xarg = s * dt_fs / KGO_HBAR;
    const int np = kgo_bessel_np(xarg, eps);
    const size_t bytes = (size_t)n * sizeof(kgo_c);
    kgo_c *phi0 = (kgo_c *)malloc(bytes), *phi1 = (kgo_c *)malloc(bytes), *phi2 = (kgo_c *)malloc(bytes);
    kgo_c *px0 = (kgo_c *)malloc(bytes), *px1 = (kgo_c *)malloc(bytes), *px2 = (kgo_c *)malloc(bytes);
    kgo_c *tmp = (kgo_c *)malloc(bytes);
    if (!phi0 || !phi1 || !phi2 || !px0 || !px1 || !px2 || !tmp) {
        free(phi0); free(phi1); free(phi2); free(px0); free(px1); free(px2); free(tmp);
        return 1;
    }
    memcpy(phi0, in, bytes);                                               /* l.1 */
    memset(px0, 0, bytes);                                                 /* l.2 */
    kgo_apply_h(n, kmax, nn, nl, hop, onsite, e0, s, phi0, phi1);          /* l.3 */
    kgo_apply_xh(n, kmax, nn, nl, hop, x, period, s, in, px1);             /* l.4 */
    const kgo_c c1 = np > 1 ? 2.0 * kgo_ipow(+1, 1) * jn(1, xarg) : 0.0;
    for (int64_t i = 0; i < n; ++i) out[i] = c1 * px1[i];                  /* l.5 */
    for (int m = 2; m < np; ++m) {                                         /* l.6 */
        kgo_apply_h(n, kmax, nn, nl, hop, onsite, e0, s, phi1, phi2);
        for (int64_t i = 0; i < n; ++i) phi2[i] = 2.0 * phi2[i] - phi0[i]; /* l.7 */
        kgo_apply_xh(n, kmax, nn, nl, hop, x, period, s, phi1, px2);
        kgo_apply_h(n, kmax, nn, nl, hop, onsite, e0, s, px1, tmp);
        for (int64_t i = 0; i < n; ++i)
            px2[i] = 2.0 * px2[i] + 2.0 * tmp[i] - px0[i];                 /* l.8 */
        const kgo_c cm = 2.0 * kgo_ipow(+1, m) * jn(m, xarg);
        for (int64_t i = 0; i < n; ++i) out[i] += cm * px2[i];             /* l.9 */
        kgo_c *t = phi0; phi0 = phi1; phi1 = phi2; phi2 = t;               /* l.10 */
        t = px0; px0 = px1; px1 = px2; px2 = t;                            /* l.11 */
    }
    if (e0 != 0.0) {
        const kgo_c ph = cexp(-I * e0 * dt_fs / KGO_HBAR);
        for (int64_t i = 0; i < n; ++i) out[i] *= ph;
    }
    free(phi0); free(phi1); free(phi2); free(px0); free(px1); free(px2); free(tmp);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O6. DOS moments C_n^DOS = <phi|T_n(H~)|phi> (eq 32; Alg. 1 l.7).      */
/* ------------------------------------------------------------------------- */
int kgo_dos_moments(int64_t n, int kmax, const int32_t *nn, const int32_t *nl,
                    const double *hop, const double *onsite, double e0, double s,
                    const kgo_c *phi, int M, kgo_c *mu)
{
    return kgo_moments(n, kmax, nn, nl, hop, onsite, e0, s, phi, phi, M, mu);
}

/* ------------------------------------------------------------------------- */
/* O7. VAC moments (Alg. 2; eqs 33, 42-43; phi_L/phi_R P:313).       */
/* psi_0 = phi, chi_0 = V phi.  For k = 0..n_steps: mu[k][:] = moments with    */
/* phi_L = V psi_k, phi_R = chi_k; then psi_{k+1} = U(-dt) psi_k,              */
/* chi_{k+1} = U(-dt) chi_k  (time grid t_k = k dt, reading g8).               */
/* mu is [n_steps+1][M].                                                       */
/* ------------------------------------------------------------------------- */
/* Row k holds Mk[k] moments (Mk[k] = 0: no moments at t_k, the states are only advanced);  */
/* row stride ld.  Chebyshev moments do not depend on how many of them are asked for, so a   */
/* shorter row is a prefix of the longer one: tests/golden/make_goldens.py uses this to      */
/* tabulate all time steps of the large configs with a short prefix and full rows at the ends. */
int kgo_vac_sched(int64_t n, int kmax, const int32_t *nn, const int32_t *nl, const double *hop,
                  const double *onsite, const double *x, double period, double e0, double s,
                  const kgo_c *phi, int n_steps, const int *Mk, int ld, double dt_fs, double eps,
                  kgo_c *mu)
{
    const size_t bytes = (size_t)n * sizeof(kgo_c);
    kgo_c *psi = (kgo_c *)malloc(bytes), *chi = (kgo_c *)malloc(bytes);
    kgo_c *phiL = (kgo_c *)malloc(bytes), *nxt = (kgo_c *)malloc(bytes);
    int rc = 0;
    if (!psi || !chi || !phiL || !nxt) { rc = 1; goto done; }
    memcpy(psi, phi, bytes);
    kgo_apply_v(n, kmax, nn, nl, hop, x, period, phi, chi);
    for (int k = 0; k <= n_steps; ++k) {
        if (Mk[k] > 0) {
            kgo_apply_v(n, kmax, nn, nl, hop, x, period, psi, phiL);
            rc = kgo_moments(n, kmax, nn, nl, hop, onsite, e0, s, phiL, chi, Mk[k], mu + (size_t)k * ld);
            if (rc) goto done;
        }
        if (k == n_steps) break;
        rc = kgo_evolve(n, kmax, nn, nl, hop, onsite, e0, s, psi, -fabs(dt_fs), eps, nxt);
        if (rc) goto done;
        memcpy(psi, nxt, bytes);
        rc = kgo_evolve(n, kmax, nn, nl, hop, onsite, e0, s, chi, -fabs(dt_fs), eps, nxt);
        if (rc) goto done;
        memcpy(chi, nxt, bytes);
    }
done:
    free(psi); free(chi); free(phiL); free(nxt);
    return rc;
}

int kgo_vac(int64_t n, int kmax, const int32_t *nn, const int32_t *nl, const double *hop,
            const double *onsite, const double *x, double period, double e0, double s,
            const kgo_c *phi, int M, int n_steps, double dt_fs, double eps, kgo_c *mu)
{
    int *Mk = (int *)malloc((size_t)(n_steps + 1) * sizeof(int));
    if (!Mk) return 1;
    for (int k = 0; k <= n_steps; ++k) Mk[k] = M;
    const int rc = kgo_vac_sched(n, kmax, nn, nl, hop, onsite, x, period, e0, s, phi, n_steps, Mk, M,
                                 dt_fs, eps, mu);
    free(Mk);
    return rc;
}

/* ------------------------------------------------------------------------- */
/* O8. MSD moments (Alg. 3; eqs 34, 44).                             */
/* psi_0 = phi, psix_0 = 0.  For k = 0..n_steps: mu[k][:] = moments with       */
/* phi_L = phi_R = psix_k; then                                                */
/* psix_{k+1} = U(dt) psix_k + [X,U(dt)] psi_k  (eq 44),  psi_{k+1} = U(dt)psi_k. */
/* ------------------------------------------------------------------------- */
/* Per-row moment counts Mk[k] and row stride ld as in kgo_vac_sched. */
int kgo_msd_sched(int64_t n, int kmax, const int32_t *nn, const int32_t *nl, const double *hop,
                  const double *onsite, const double *x, double period, double e0, double s,
                  const kgo_c *phi, int n_steps, const int *Mk, int ld, double dt_fs, double eps,
                  kgo_c *mu)
{
    const size_t bytes = (size_t)n * sizeof(kgo_c);
    kgo_c *psi = (kgo_c *)malloc(bytes), *psix = (kgo_c *)malloc(bytes);
    kgo_c *a = (kgo_c *)malloc(bytes), *b = (kgo_c *)malloc(bytes);
    int rc = 0;
    if (!psi || !psix || !a || !b) { rc = 1; goto done; }
    memcpy(psi, phi, bytes);
    memset(psix, 0, bytes);
    for (int k = 0; k <= n_steps; ++k) {
        if (Mk[k] > 0) {
            rc = kgo_moments(n, kmax, nn, nl, hop, onsite, e0, s, psix, psix, Mk[k], mu + (size_t)k * ld);
            if (rc) goto done;
        }
        if (k == n_steps) break;
        rc = kgo_evolve(n, kmax, nn, nl, hop, onsite, e0, s, psix, fabs(dt_fs), eps, a);
        if (rc) goto done;
        rc = kgo_comm_evolve(n, kmax, nn, nl, hop, onsite, x, period, e0, s, psi, fabs(dt_fs), eps, b);
        if (rc) goto done;
        for (int64_t i = 0; i < n; ++i) psix[i] = a[i] + b[i];
        rc = kgo_evolve(n, kmax, nn, nl, hop, onsite, e0, s, psi, fabs(dt_fs), eps, a);
        if (rc) goto done;
        memcpy(psi, a, bytes);
    }
done:
    free(psi); free(psix); free(a); free(b);
    return rc;
}

int kgo_msd(int64_t n, int kmax, const int32_t *nn, const int32_t *nl, const double *hop,
            const double *onsite, const double *x, double period, double e0, double s,
            const kgo_c *phi, int M, int n_steps, double dt_fs, double eps, kgo_c *mu)
{
    int *Mk = (int *)malloc((size_t)(n_steps + 1) * sizeof(int));
    if (!Mk) return 1;
    for (int k = 0; k <= n_steps; ++k) Mk[k] = M;
    const int rc = kgo_msd_sched(n, kmax, nn, nl, hop, onsite, x, period, e0, s, phi, n_steps, Mk, M,
                                 dt_fs, eps, mu);
    free(Mk);
    return rc;
}

/* ------------------------------------------------------------------------- */
/* O9. KPM reconstruction (eqs 29-31 P:169-175 with Jackson damping eq 35      */
/* P:190-192), for a unit-norm phi and physical energies E (readings g1, g3):  */
/* f(E) = 1/(pi s sqrt(1-E~^2)) sum_n g_n (2-delta_n0) T_n(E~) Re mu_n,        */
/* E~ = (E-E0)/s, T_n(E~) = cos(n acos E~).                                    */
/* ------------------------------------------------------------------------- */
void kgo_jackson(int M, double *g)
{
    const double alpha = 1.0 / (M + 1.0);
    for (int nn_ = 0; nn_ < M; ++nn_)
        g[nn_] = (1.0 - nn_ * alpha) * cos(M_PI * nn_ * alpha) +
                 alpha * sin(M_PI * nn_ * alpha) / tan(M_PI * alpha);
}

void kgo_kpm_reconstruct(int M, const kgo_c *mu, int use_jackson, double e0, double s, int ne,
                         const double *energies, double *f)
{
    double *g = (double *)malloc((size_t)M * sizeof(double));
    if (use_jackson) kgo_jackson(M, g);
    else for (int m = 0; m < M; ++m) g[m] = 1.0;
    for (int j = 0; j < ne; ++j) {
        const double et = (energies[j] - e0) / s;
        const double th = acos(et);
        long double sum = 0.0L;
        for (int m = 0; m < M; ++m)
            sum += (long double)(g[m] * (m == 0 ? 1.0 : 2.0) * cos(m * th) * creal(mu[m]));
        f[j] = (double)sum / (M_PI * s * sqrt(1.0 - et * et));
    }
    free(g);
}

/* ------------------------------------------------------------------------- */
/* O10. Running conductivities and ballistic conductance from reconstructed   */
/* functions of (t_k, E_j), t_k = k dt, k = 0..nt (reading g8):               */
/*   rho[j]      = rho~(E_j)               (eq 29, per site and spin, 1/eV)   */
/*   fvac[k][j]  = rho~ C_vv(E_j, t_k)     (eq 30, nm^2/fs^2/eV)              */
/*   fmsd[k][j]  = rho~ DeltaX^2(E_j,t_k)  (eq 31, nm^2/eV)                   */
/* The paper's rho = dens * rho~ with dens = 2N/Omega (2 = spin, eq 8,   */
/* <phi|phi> = N P:128), so in units of e^2/h (h = 2 pi hbar):                */
/*   sigma_GK(E,t) = 2 pi hbar dens int_0^t rho~C_vv dt'      (eq 6  P:61)    */
/*   sigma_E1(E,t) = 2 pi hbar dens (1/2) d(rho~DX2)/dt       (eq 9  P:71)    */
/*   sigma_E2(E,t) = 2 pi hbar dens rho~DX2 / (2t), 0 at t=0  (eq 11)    */
/*   L(E,t)        = 2 sqrt(DX2) = 2 sqrt(fmsd/rho)           (eq 50)   */
/*   G(E,t)        = (W/L) sigma_E1, 0 where L = 0            (eq 51)   */
/* Discretisation (reading g14; the paper is silent): trapezoid rule for the  */
/* integral; central differences for the derivative, second-order one-sided   */
/* three-point formulas at k = 0 and k = nt (two-point when nt = 1).          */
/* Any output pointer may be NULL; fvac / fmsd may be NULL if unused.         */
/* ------------------------------------------------------------------------- */
static double kgo_ddt(const double *f, int k, int nt, int ne, int j, double dt)
{
    if (nt < 1) return 0.0;
    if (nt == 1) return (f[1 * ne + j] - f[0 * ne + j]) / dt;
    if (k == 0) return (-3.0 * f[0 * ne + j] + 4.0 * f[1 * ne + j] - f[2 * ne + j]) / (2.0 * dt);
    if (k == nt)
        return (3.0 * f[nt * ne + j] - 4.0 * f[(nt - 1) * ne + j] + f[(nt - 2) * ne + j]) / (2.0 * dt);
    return (f[(k + 1) * ne + j] - f[(k - 1) * ne + j]) / (2.0 * dt);
}

void kgo_transport(int nt, int ne, double dt_fs, double dens_per_nm2, double width_nm,
                   const double *rho, const double *fvac, const double *fmsd, double *sigma_gk,
                   double *sigma_e1, double *sigma_e2, double *length_nm, double *conductance)
{
    const double pref = 2.0 * M_PI * KGO_HBAR * dens_per_nm2;
    for (int j = 0; j < ne; ++j) {
        long double integral = 0.0L;
        for (int k = 0; k <= nt; ++k) {
            if (sigma_gk) {
                if (k > 0)
                    integral += 0.5L * ((long double)fvac[(k - 1) * ne + j] + fvac[k * ne + j]) * dt_fs;
                sigma_gk[k * ne + j] = pref * (double)integral;
            }
            if (!fmsd) continue;
            const double e1 = pref * 0.5 * kgo_ddt(fmsd, k, nt, ne, j, dt_fs);
            if (sigma_e1) sigma_e1[k * ne + j] = e1;
            if (sigma_e2) sigma_e2[k * ne + j] = k == 0 ? 0.0 : pref * fmsd[k * ne + j] / (2.0 * k * dt_fs);
            const double dx2 = fmsd[k * ne + j] / rho[j];
            const double len = 2.0 * sqrt(dx2 > 0.0 ? dx2 : 0.0);
            if (length_nm) length_nm[k * ne + j] = len;
            if (conductance) conductance[k * ne + j] = len > 0.0 ? width_nm / len * e1 : 0.0;
        }
    }
}

/* ------------------------------------------------------------------------- */
/* O11. Fourier moments (Alg. 4; eq 45; eqs 25-27):  */
/*   F_n = <phi_L| U(n dtau) |phi_R>,  n = -Nm..Nm,  stored at F[n + Nm].      */
/* l.1-6: phi' <- phi_R, F_0, then phi' <- U(dtau) phi' and F_n for n = 1..Nm; */
/* l.7-11: the same with U^dagger(dtau) for F_{-n}.  U by Alg. 6 (kgo_evolve). */
/* ------------------------------------------------------------------------- */
int kgo_fourier_moments(int64_t n, int kmax, const int32_t *nn, const int32_t *nl, const double *hop,
                        const double *onsite, double e0, double s, const kgo_c *phiL,
                        const kgo_c *phiR, int Nm, double dtau_fs, double eps, kgo_c *F)
{
    kgo_c *a = (kgo_c *)malloc((size_t)n * sizeof(kgo_c));
    kgo_c *b = (kgo_c *)malloc((size_t)n * sizeof(kgo_c));
    if (!a || !b) { free(a); free(b); return 1; }
    for (int dir = +1; dir >= -1; dir -= 2) {
        memcpy(a, phiR, (size_t)n * sizeof(kgo_c));                       /* l.1 / l.7 */
        if (dir > 0) F[Nm] = kgo_dot(n, phiL, a);                         /* l.2 */
        for (int m = 1; m <= Nm; ++m) {                                   /* l.3 / l.8 */
            if (kgo_evolve(n, kmax, nn, nl, hop, onsite, e0, s, a, dir * dtau_fs, eps, b)) {
                free(a); free(b); return 1;
            }
            kgo_c *t = a; a = b; b = t;                                   /* l.4 / l.9 */
            F[Nm + dir * m] = kgo_dot(n, phiL, a);                        /* l.5 / l.10 */
        }
    }
    free(a); free(b);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O12. FTM reconstruction (eqs 22-24) with the Hanning window       */
/* w_n = (1 + cos(pi n/(Nm+1)))/2 (eq 28), per site and spin for a   */
/* unit-norm phi (the paper's (2/Omega) Tr -> <phi|.|phi>, readings g1, g3):   */
/*   f(E) = dtau/(2 pi hbar) sum_{n=-Nm}^{Nm} w_n Re[ e^{i E n dtau/hbar} F_n ]  */
/* (delta(E-H) = (1/2 pi hbar) int dt e^{i(E-H)t/hbar}, discretised with dtau). */
/* ------------------------------------------------------------------------- */
void kgo_ftm_reconstruct(int Nm, const kgo_c *F, int use_window, double dtau_fs, int ne,
                         const double *energies, double *f)
{
    for (int j = 0; j < ne; ++j) {
        long double sum = 0.0L;
        for (int m = -Nm; m <= Nm; ++m) {
            const double w = use_window ? 0.5 * (1.0 + cos(M_PI * m / (Nm + 1.0))) : 1.0;
            sum += (long double)(w * creal(cexp(I * energies[j] * m * dtau_fs / KGO_HBAR) * F[m + Nm]));
        }
        f[j] = (double)sum * dtau_fs / (2.0 * M_PI * KGO_HBAR);
    }
}
