/*
 * kg.h — C ABI of libkg: the Chebyshev hot path of the linear-scaling real-space
 * Kubo-Greenwood method (arXiv 1307.0288), hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * "P:n" cites line n of PAPER.md (the paper's text).  Notation follows the paper:
 *   H      sparse real-symmetric tight-binding Hamiltonian given as a neighbour list
 *          NN_n / NL_nk with matrix elements H_{n,NL_nk}               (Alg. 8)
 *   X      diagonal position operator, X_m                                     (eq 14)
 *   V      velocity (i/hbar)[H, X]                                             (eq 15)
 *   H~     (H - E0)/s, spectrum inside [-1, 1]
 *   T_m    Chebyshev polynomials, T_m = 2 H~ T_{m-1} - T_{m-2}                 (eq 38)
 *   U(dt)  exp(-i H dt/hbar) = sum_m (2-d_m0)(-i)^m J_m(s dt/hbar) T_m(H~)     (eq 36)
 *
 * Units: eV, nm, fs; hbar = 0.6582119569 eV fs.
 *
 * POINTERS.  Every array argument may be a DEVICE pointer (cudaMalloc / torch CUDA tensor)
 * or a HOST pointer (pageable or pinned); the library detects which with
 * cudaPointerGetAttributes.  Host inputs are copied to library-owned device staging
 * buffers on `stream`; host outputs are written by an asynchronous device->host copy on
 * `stream` (for pageable memory CUDA makes that copy synchronous).  All arithmetic runs in
 * CUDA kernels; there is no CPU fallback.  All arrays are caller-owned and BORROWED IN STREAM
 * ORDER: device arrays and pinned host arrays are read / written by work that is still queued
 * on `stream` when the call returns, so they must stay alive and unmodified (inputs) / unread
 * (outputs) until that work has run — synchronise the stream, or order later work after it on
 * the same stream.  Pageable host arrays are consumed / filled before the call returns.
 * Inputs are never modified; `out` must not alias `in`.
 *
 * VECTORS are `[n][R]` complex128, site-major (the R values of one site are contiguous,
 * element (site i, vector r) at index i*R + r), R in {1, 2, 4, 8, 16}; kg_vac takes R <= 8
 * (it advances [psi | chi] as one batch of 2R columns).  kg_c128 is layout-compatible with
 * C99 `double complex`, std::complex<double> and torch.complex128.  The sites may be
 * re-numbered inside the library (KG_OPT_REORDER); every vector crosses this boundary in the
 * CALLER's site order.
 *
 * STREAMS.  `stream` is a cudaStream_t cast to void* (NULL = legacy default stream).  Calls
 * enqueue work on it and return without synchronising, except: kg_create_hamiltonian[_csr]
 * (validation result; also builds the two-step kernel's tile plans where KG_OPT_TWO_STEP's
 * default will use them), the first moments call after KG_OPT_TWO_STEP was forced on a handle
 * whose plan create did not build, calls that have to grow the workspace while a cached CUDA graph
 * refers to it, calls with KG_OPT_CHECK_INPUT set, and calls whose outputs are pageable host
 * memory.  Device outputs are valid once the stream has been synchronised.
 *
 * ERRORS.  Every call returns KG_OK or an error code; nothing throws or aborts across the
 * ABI (the bodies run inside a catch-all guard: a failed host allocation is KG_ENOMEM).
 * kg_last_error() returns a thread-local description of the last failure.
 *
 * A handle owns its device copy of the matrix and a lazily grown workspace (Chebyshev
 * vectors T_m, accumulators, per-block moment partials, cached CUDA graphs) that every call
 * on the handle re-uses: a handle is not thread-safe, and its calls must be issued on ONE
 * stream at a time (before switching streams, synchronise the old one or make the new one
 * wait on an event recorded in it) — two calls on different streams would race on the
 * workspace.  Different handles are independent.
 */
#ifndef KG_H
#define KG_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct kg_hamiltonian kg_hamiltonian; /* opaque, library-owned */
typedef struct { double re, im; } kg_c128;

enum {
    KG_OK = 0,
    KG_EINVAL = 1,       /* null pointer, bad size, index out of range, non-finite value, aliasing */
    KG_ENOMEM = 2,       /* device allocation failed */
    KG_ECUDA = 3,        /* CUDA runtime error (text in kg_last_error) */
    KG_ESPECTRUM = 4,    /* Gershgorin bound of (H - E0) exceeds s: recursion would diverge */
    KG_EUNSUPPORTED = 5  /* R not in the supported set, kmax too large */
};

/* Thread-local message of the last error returned on this thread ("" if none). */
const char *kg_last_error(void);

/*
 * kg_create_hamiltonian — build the scaled operator H~ = (H - E0)/s and the commutator
 * weights of [X, H~] from the paper's neighbour list (Alg. 8 "Require" lines
 * P:420-425; scaling P:192; [X,H] eq 15, eq 41).
 *
 *   n          number of sites (1 <= n < 2^31)
 *   kmax       row width of the list (1 <= kmax <= 32)
 *   nn[n]      NN_i, number of neighbours of site i (0 <= nn[i] <= kmax)
 *   nl[kmax*n] NL_ik at nl[k*n + i]  — k-major, "NL_00, NL_10, NL_20, ..., NL_01, ...";
 *              entries with k >= nn[i] are ignored
 *   hop_eV     H_{i,NL_ik} at hop_eV[k*n + i], real (eq 13), eV
 *   onsite_eV  H_ii, eV; NULL = 0
 *   x_nm[n]    X_i, the coordinate along the transport direction, nm
 *   period_x_nm  period of that coordinate; <= 0: open boundary.  Bond displacements
 *              X_m - X_i are reduced to the minimum image when periodic.
 *   e0_eV, scale_eV   H~ = (H - e0)/scale, scale > 0 (the half-width "Delta E" of
 *              BASELINE.json; NOT the paper's full bandwidth of eq 47-49)
 *
 * Validates (indices in range, counts <= kmax, finite values, H symmetric, Gershgorin bound
 * max_i(|H_ii - E0| + sum_k |H_ik|) <= s) on the device, synchronises `stream`, and returns
 * KG_EINVAL / KG_ESPECTRUM accordingly.  The caller may free its arrays after the call.
 */
int kg_create_hamiltonian(kg_hamiltonian **out, int64_t n, int32_t kmax, const int32_t *nn,
                          const int32_t *nl, const double *hop_eV, const double *onsite_eV,
                          const double *x_nm, double period_x_nm, double e0_eV, double scale_eV,
                          void *stream);

/* Same operator from CSR: rowptr[n+1] (int64), col[nnz] (int32), hop_eV[nnz]; the diagonal is
 * given separately in onsite_eV (diagonal entries inside the CSR arrays are rejected).
 * kmax becomes the longest row.  Converted to the k-major list on the device. */
int kg_create_hamiltonian_csr(kg_hamiltonian **out, int64_t n, const int64_t *rowptr,
                              const int32_t *col, const double *hop_eV, const double *onsite_eV,
                              const double *x_nm, double period_x_nm, double e0_eV,
                              double scale_eV, void *stream);

/* Frees the device matrix and workspace.  NULL is accepted. */
int kg_destroy_hamiltonian(kg_hamiltonian *h);

/* Bytes of device memory currently owned by the handle (matrix + workspace). */
size_t kg_workspace_bytes(const kg_hamiltonian *h);

/* Number of sites n and row width kmax of a handle (0 on NULL). */
int64_t kg_num_sites(const kg_hamiltonian *h);

/*
 * kg_moments — Chebyshev moments C_m = <phi_L| T_m(H~) |phi_R>, m = 0..M-1, per vector
 * (Alg. 5, eq 46).  <a|b> = sum_i conj(a_i) b_i.
 *   phiL, phiR  [n][R]; may be the same pointer
 *   mu          [R][M] complex128 (vector r at mu[r*M + m]), M >= 2
 * One fused kernel per Chebyshev step (recursion eq 38 + inner product) — or per two steps,
 * KG_OPT_TWO_STEP — and a final fixed-order reduction: results are bitwise reproducible run to
 * run for a given handle and option set.
 */
int kg_moments(kg_hamiltonian *h, const kg_c128 *phiL, const kg_c128 *phiR, int R, int M,
               kg_c128 *mu, void *stream);

/* kg_dos_moments — C_m^DOS = <phi| T_m(H~) |phi> (eq 32; Alg. 1 l.7): kg_moments with
 * phi_L = phi_R = phi.  For a unit-norm phi, mu_0 = 1. */
int kg_dos_moments(kg_hamiltonian *h, const kg_c128 *phi, int R, int M, kg_c128 *mu,
                   void *stream);

/*
 * kg_evolve — out = U(dt) in for dt_fs > 0, out = U(-|dt|) in = U^dagger(|dt|) in for dt_fs < 0
 * (Alg. 6, eq 36), Bessel argument x = s |dt|/hbar, global phase
 * exp(-i E0 dt/hbar).  The series keeps N_p = 1 + max{m : |J_m(x)| >= bessel_eps} terms
 * (bessel_eps <= 0 selects 1e-15).  in, out: [n][R], out must not alias in.
 * dt_fs = 0 is KG_EINVAL.
 */
int kg_evolve(kg_hamiltonian *h, const kg_c128 *in, kg_c128 *out, int R, double dt_fs,
              double bessel_eps, void *stream);

/* kg_apply_velocity — out = V in, V = (i/hbar)[H, X] with the unscaled H (eq 15):
 * out[i] = (i/hbar) sum_k (X_{NL_ik} - X_i) H_{i,NL_ik} in[NL_ik], nm/fs. */
int kg_apply_velocity(kg_hamiltonian *h, const kg_c128 *in, kg_c128 *out, int R, void *stream);

/*
 * kg_evolve_x — one step of eq 44, in place on caller-owned device or host arrays:
 *   psix <- U(dt) psix + [X, U(dt)] psi,      psi <- U(dt) psi          (dt_fs > 0)
 * with [X, U(dt)] from eq 37 and the recursions eqs 39-41 (Alg. 7).
 * psix = 0 gives psix <- [X, U(dt)] psi.  psi, psix: [n][R].
 */
int kg_evolve_x(kg_hamiltonian *h, kg_c128 *psi, kg_c128 *psix, int R, double dt_fs,
                double bessel_eps, void *stream);

/*
 * kg_vac — velocity auto-correlation moments (Alg. 2; eqs 33, 42-43):
 *   C_m^VAC(t_k) = <phi| U(t_k) V T_m(H~) U^dagger(t_k) V |phi>,   t_k = k dt, k = 0..n_steps
 * computed as <V psi_k| T_m(H~) |chi_k> with psi_0 = phi, chi_0 = V phi and
 * psi_{k+1} = U(-dt) psi_k, chi_{k+1} = U(-dt) chi_k.
 *   phi [n][R] unit-norm random vectors;  mu [R][n_steps+1][M]  (r, k, m) at
 *   mu[(r*(n_steps+1) + k)*M + m].  dt_fs > 0, n_steps >= 0, M >= 2.
 */
int kg_vac(kg_hamiltonian *h, const kg_c128 *phi, int R, int M, int n_steps, double dt_fs,
           double bessel_eps, kg_c128 *mu, void *stream);

/*
 * kg_msd — mean-square-displacement moments (Alg. 3; eqs 34, 44):
 *   C_m^MSD(t_k) = <phi| [X,U(t_k)]^dagger T_m(H~) [X,U(t_k)] |phi>
 * with psix_k = [X, U(t_k)] phi advanced by eq 44; row k = 0 is exactly 0.
 * Same argument and output layout as kg_vac.
 */
int kg_msd(kg_hamiltonian *h, const kg_c128 *phi, int R, int M, int n_steps, double dt_fs,
           double bessel_eps, kg_c128 *mu, void *stream);

/*
 * kg_bessel_terms — host helper exposing the series coefficients the library uses (eq 36
 * P:200): writes N_p to *np_out and, if j != NULL, J_m(x) for m < min(N_p, cap) to
 * the HOST array j.  Pure host arithmetic (no GPU needed).
 */
int kg_bessel_terms(double x, double bessel_eps, int *np_out, double *j, int cap);

/*
 * kg_kpm_reconstruct — kernel-polynomial reconstruction of a function of energy from Chebyshev
 * moments (eqs 29-31) with Jackson damping (eq 35), for unit-norm phi:
 *   f[row][j] = 1/(pi s sqrt(1 - x_j^2)) * sum_{m<M} g_m (2 - delta_m0) T_m(x_j) Re mu[row][m],
 *   x_j = (E_j - E0)/s,  g_m = (1 - m a) cos(pi m a) + a sin(pi m a) cot(pi a),  a = 1/(M+1).
 * Applied to kg_dos_moments it gives rho(E) per site and spin (1/eV, integrates to 1); to a row
 * of kg_vac / kg_msd it gives rho(E) C_vv(E,t) (nm^2/fs^2/eV) / rho(E) DeltaX^2(E,t) (nm^2/eV).
 *   mu        [rows][M] complex128 (any leading shape flattened to rows), host or device
 *   jackson   1: g_m as above; 0: g_m = 1 (Dirichlet)
 *   energies_eV [n_energies], host or device; every |x_j| must be < 1: a host grid is checked
 *             (KG_EINVAL), a device grid is not read back — such entries of f are NaN
 *   f         [rows][n_energies] fp64, host or device
 * Runs as CUDA kernels on `stream`; temporaries are stream-ordered allocations from a memory pool
 * that the library creates per device at the first post-processing call there (kg_kpm_reconstruct,
 * kg_transport, kg_ftm_reconstruct) and keeps, with whatever it has grown to, until the process
 * exits; the application's default pool is not touched.  Once the pool is warm the call neither
 * allocates with cudaMalloc nor synchronises.
 */
int kg_kpm_reconstruct(const kg_c128 *mu, int64_t rows, int M, int jackson, double e0_eV,
                       double scale_eV, const double *energies_eV, int n_energies, double *f,
                       void *stream);

/*
 * kg_kpm_reconstruct_noalloc — the same reconstruction (eqs 29-31, Jackson damping eq 35
 * P:190-192; same formula, same kernels, same results as kg_kpm_reconstruct) for callers that are
 * not in a position to allocate device memory: a program that has already given all of the GPU's
 * memory to an arena of its own (a framework's caching allocator; a run whose Chebyshev vectors
 * were sized to fill the card), where one more cudaMalloc or a growing memory pool fails, and a
 * program that post-processes moments inside a loop with a latency budget that a fresh allocation
 * (which can stall the whole device) would break.  This call allocates nothing — no cudaMalloc,
 * cudaMallocAsync, cudaFree or allocating library routine, on the host or on the device.  The
 * damped weights (2 - delta_m0) g_m, the one temporary the reconstruction needs, are written to
 * a fixed array inside the library image instead:
 *
 *   LIMIT    M <= KG_KPM_NOALLOC_MAX_M (16384 weights = 128 KiB of device memory, occupied on
 *            every GPU that loads libkg until the process exits).  A longer series is KG_EINVAL
 *            with the limit in kg_last_error(); use kg_kpm_reconstruct for it.
 *   POINTERS mu [rows][M], energies_eV [n_energies] and f [rows][n_energies] must all be DEVICE
 *            memory (a host array would have to be staged, which takes an allocation): a host
 *            pointer is KG_EINVAL.  The energy grid is therefore never checked on the host;
 *            entries with |(E_j - E0)/s| >= 1 give NaN in f, as for a device grid in
 *            kg_kpm_reconstruct.
 *   SHARING  there is ONE weight array per GPU, used by every call from every thread and stream.
 *            A call rewrites entries 0..M-1 before it reads them and reads no others, so what an
 *            earlier call left behind does no harm; but two calls whose kernels can overlap on
 *            the GPU (issued on different streams without an ordering between them) race on the
 *            array and give wrong results.  Issue them on one stream, or order them with events.
 *   FIRST CALL  the first call on each device looks the array's device address up
 *            (cudaGetSymbolAddress, with the calling thread's current device) and keeps it; make
 *            that first call outside any stream capture.  Later calls only enqueue two kernels
 *            on `stream`.  Device ordinals >= 64 are KG_EUNSUPPORTED.
 * Does not synchronise.  Other arguments as kg_kpm_reconstruct.
 */
#define KG_KPM_NOALLOC_MAX_M 16384
int kg_kpm_reconstruct_noalloc(const kg_c128 *mu, int64_t rows, int M, int jackson, double e0_eV,
                               double scale_eV, const double *energies_eV, int n_energies,
                               double *f, void *stream);

/*
 * kg_transport — running conductivities and ballistic length / conductance on a (t_k, E_j) grid,
 * t_k = k dt, k = 0..n_steps, from reconstructed functions (kg_kpm_reconstruct):
 *   rho[j] = rho~(E_j);  fvac[k][j] = rho~ C_vv(E_j,t_k);  fmsd[k][j] = rho~ DeltaX^2(E_j,t_k).
 * With the paper's rho = dens * rho~, dens = 2N/Omega (nm^-2 for a 2-D sample; eq 8),
 * in units of e^2/h:
 *   sigma_gk = 2 pi hbar dens * int_0^t rho~C_vv dt'         (eq 6; trapezoid rule)
 *   sigma_e1 = 2 pi hbar dens * (1/2) d(rho~DX2)/dt          (eq 9; central differences,
 *                                                             second-order one-sided at both ends)
 *   sigma_e2 = 2 pi hbar dens * rho~DX2 / (2 t), 0 at t = 0  (eq 11)
 *   length_nm = 2 sqrt(fmsd / rho)                           (eq 50)
 *   conductance = (width_nm / length_nm) * sigma_e1, 0 where the length is 0  (eq 51)
 * All arrays fp64, host or device; tables are [n_steps+1][n_energies].  Every output pointer may
 * be NULL; fvac (fmsd, rho) may be NULL when no requested output needs it.  Does not synchronise.
 * The stochastic trace average over random vectors (eq 21) is the caller's: average the
 * reconstructed rows over vectors before this call (the functions are linear in the moments).
 */
int kg_transport(int n_steps, int n_energies, double dt_fs, double dens_per_nm2, double width_nm,
                 const double *rho, const double *fvac, const double *fmsd, double *sigma_gk,
                 double *sigma_e1, double *sigma_e2, double *length_nm, double *conductance,
                 void *stream);

/*
 * kg_fourier_moments — Fourier moments F_n = <phi_L| U(n dtau) |phi_R>, n = -Nm..Nm (Alg. 4
 * P:320-344, eq 45; eqs 25-27): phi' <- phi_R, then Nm applications of U(dtau) (Alg. 6, as
 * kg_evolve) with an inner product after each, and the same with U^dagger(dtau) for n < 0.
 *   phiL, phiR [n][R] (may be the same pointer);  F [R][2*Nm+1] complex128, F_n of vector r at
 *   F[r*(2*Nm+1) + n + Nm];  dtau_fs > 0 (the paper's choice: pi hbar / s);  Nm >= 0.
 * Inner products use per-block partials and a fixed-order final sum (bitwise reproducible).
 */
int kg_fourier_moments(kg_hamiltonian *h, const kg_c128 *phiL, const kg_c128 *phiR, int R, int Nm,
                       double dtau_fs, double bessel_eps, kg_c128 *F, void *stream);

/*
 * kg_ftm_reconstruct — Fourier-transform-method reconstruction (eqs 22-24) with the
 * Hanning window w_n = (1 + cos(pi n/(Nm+1)))/2 (eq 28; window = 0: w_n = 1), per site
 * and spin for unit-norm phi:
 *   f[row][j] = dtau/(2 pi hbar) * sum_{n=-Nm}^{Nm} w_n Re[ exp(i E_j n dtau/hbar) F[row][n+Nm] ].
 *   F [rows][2*Nm+1], energies_eV [n_energies], f [rows][n_energies]; host or device pointers.
 * Does not synchronise.
 */
int kg_ftm_reconstruct(const kg_c128 *F, int64_t rows, int Nm, int window, double dtau_fs,
                       const double *energies_eV, int n_energies, double *f, void *stream);

/* Tuning / introspection (not part of the paper's problem statement). */
enum {
    KG_OPT_USE_GRAPHS = 1,   /* replay the one-step moment loop as a cached CUDA graph: 1 always, 0 never, -1 (default)
                                when n * R <= 2^21 (launch-bound sizes); never on the legacy default stream, which
                                cannot be captured */
    KG_OPT_BLOCKS_PER_SM = 2, /* persistent grid = SMs * this (default chosen per kernel) */
    KG_OPT_THREADS = 3,      /* threads per block (default 256) */
    KG_OPT_STAGED = 4,       /* 1 (default): moment steps run the TMA-staged kernel when eligible */
    KG_OPT_STAGES = 5,       /* shared-memory ring depth of the staged kernel (0 = auto) */
    KG_OPT_STAGED_CTAS = 6,  /* CTAs per SM of the staged kernel (0 = auto) */
    KG_OPT_ALTERNATE = 7,    /* 1 (default): alternate the sweep direction step to step (L2 reuse) */
    KG_OPT_DICT = 8,         /* 0: drop the hopping dictionary, stream fp64 hoppings (general path) */
    KG_OPT_DOUBLING = 9,     /* 1 (default): two moments per Chebyshev sweep via 2 T_a T_b = T_{a+b} +
                                T_{|a-b|} — when phi_L and phi_R are the same array (kg_dos_moments,
                                kg_msd) and, advancing [phi_L | phi_R] as one batch, in kg_vac;
                                0: literal Alg. 5 */
    KG_OPT_CLENSHAW = 10,    /* 1 (default): U(dt) phi and the pair of eq 44 summed by Clenshaw's backward
                                recurrence (no accumulator streams); 0: forward recursion + accumulation
                                as in Alg. 6 / Alg. 7 */
    KG_OPT_REORDER = 12,     /* process-wide, read at create (kg_set_default_option): re-number the sites
                                internally so that consecutive sites form compact patches of the lattice
                                (recursive breadth-first bisection of the neighbour list, on groups of 8 consecutive
                                caller sites so that a site keeps its caller index modulo 8; moments do not
                                depend on the site order, vectors are permuted at the boundary of every call):
                                1 always, 0 never, -1 (default) when n >= 65536.
                                COST: only the moment loops (kg_moments, kg_dos_moments, kg_vac, kg_msd) gain from the
                                new order.  On a re-ordered handle every call that takes or returns a vector pays one
                                extra pass over it per vector argument (a gather into internal order on the way in, a
                                scatter on the way out) and keeps staging buffers of n * R * 16 bytes each in the
                                workspace: kg_apply_velocity is 3 sweeps instead of 1, each kg_evolve of a caller-driven
                                loop 2 extra sweeps, kg_evolve_x 4.  A handle used mainly for kg_evolve /
                                kg_apply_velocity is better created with the option at 0.  Moments are bitwise
                                reproducible for a given setting, not across settings (the summation order follows
                                the site order) */
    KG_OPT_TWO_STEP = 13,    /* doubling moment loops run two Chebyshev steps per pass with the tile + two halo
                                rings in shared memory (temporal blocking), on <= 2 contiguous columns at a time
                                (wider batches as column-pair planes side by side in one launch, when the batch exceeds the L2):
                                1 whenever the plan fits, 0 never, -1 (default) when the sites are re-ordered
                                and there are at least four 1024-element tiles per SM */
    KG_OPT_CHECK_INPUT = 14, /* 1: every input vector is scanned for NaN / Inf (one extra pass and a stream
                                synchronisation per call) and the call returns KG_EINVAL; 0 (default): not checked —
                                non-finite input gives non-finite output.  (The matrix is always checked at create.) */
    KG_OPT_ONE_LAUNCH = 15,  /* launch-bound sizes (all 512-element tiles of a batch fit the shared memory of one
                                8-CTA cluster: n * R <= 16 K elements for the paper's model; 9-16 tiles use a 16-CTA cluster when the device takes it): the moment loop after
                                its first step runs as ONE kernel, one cluster barrier per Chebyshev step, vectors
                                and matrix rows in distributed shared memory; bitwise equal to the per-step
                                launches.  -1 (default) / 1: on when eligible, 0: off */
    KG_OPT_PDL = 11          /* consecutive sweeps chained by programmatic dependent launch (the next sweep's
                                CTAs are scheduled while this one drains): 1 on, 0 off, -1 (default) on for
                                launch-bound sizes, n * R <= 2^18 */
};
int kg_set_option(kg_hamiltonian *h, int option, int64_t value);

/* Options that act at create time (KG_OPT_REORDER): process-wide default for handles created
 * afterwards.  Not thread-safe against concurrent kg_create_hamiltonian calls. */
int kg_set_default_option(int option, int64_t value);

/* Number of kernel launches (graph nodes included) the handle has enqueued since creation. */
int64_t kg_launch_count(const kg_hamiltonian *h);

#ifdef __cplusplus
}
#endif
#endif /* KG_H */
