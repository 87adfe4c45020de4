/*
 * cool.h — C ABI of the B200-native per-cell two-temperature radiative cooling step of
 * arXiv 2505.08855.  The library is libcool_b200.so; every compute step runs in
 * hand-written sm_100a CUDA kernels.  There is no CPU fallback: every entry point that
 * touches a device returns COOL_ECUDA when no usable CUDA device exists.
 *
 * What the step computes (per cell: "The cooling function utilizes the
 * values of H_th, B, n_e and T_e obtained from the simulation to find the appropriate
 * interpolated cooling rate from a precomputed table"; L185: the explicit limiter;
 * L197: the temperature floor; L140-L147: Coulomb exchange):
 *
 *   repeat nsub times with h = dt/nsub:
 *     x_k   = log10(primitive of table axis k)            (L122-L124: log-spaced axes)
 *     t_k   = clamp((x_k - lo_k)/Delta_k, 0, n_k - 1)      (edge clamp, texture-clamp semantics)
 *     y     = multilinear interpolation of the stored log10 values;  rate = 10^y
 *     nproc = 1: Lambda = rate.   nproc = 3: Q_thin = Q_brem + eta Q_syn (eq 10) and
 *             Lambda = Q_total of eqs 11-12 (L110-L116) with the cell's H_th (eqs 13-14)
 *     floor : Lambda = 0 when p_gas/rho < (pi/2)(h_floor Omega_K r)^2      (eq 19)
 *     Q_cc  : eq 15 (L142-L144), from a coefficient table or analytically
 *     dE    = min(Lambda h, f_limit u_e)                                   (L185)
 *     x     = sign(Q_cc) min(|Q_cc| h, f_limit u_donor, equalising transfer)
 *     u_e  += x - dE ;  u_i -= x ;  Theta_s = u_s (gamma_s - 1)(m_p/m_e)/rho
 *   luminosity diagnostic  L = sum dE vol / dt                             (eq 22)
 *
 * Conventions: Theta_s = k_B T_s/(m_e c^2) for BOTH species (L63, L147); rho in units of
 * units.rho_scale_cgs; bsq = b^2 with (4 pi)^-1/2 absorbed (L173); times in r_g/c of
 * units.mbh_msun; u_s = rho Theta_s (m_e/m_p)/(gamma_s - 1).  dt is fluid-frame time.
 *
 * All functions return cool_status (0 = COOL_OK), never abort and never print.  After a
 * failure cool_last_error() holds a thread-local message.
 */
#ifndef COOL_H
#define COOL_H

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { COOL_OK = 0, COOL_EINVAL = 1, COOL_ENOMEM = 2, COOL_ECUDA = 3, COOL_EUNSUPPORTED = 4 } cool_status;
typedef enum { COOL_F32 = 0, COOL_F64 = 1 } cool_dtype;
typedef enum { COOL_AX_LOG_RHO = 0, COOL_AX_LOG_THETA_E = 1, COOL_AX_LOG_BSQ = 2, COOL_AX_LOG_THETA_I = 3,
               /* the paper's own table parameters, cgs units: disk thermal scale height [cm], magnetic
                * field strength [G], electron density [cm^-3], electron temperature [K] */
               COOL_AX_LOG_HTH = 4, COOL_AX_LOG_B = 5, COOL_AX_LOG_NE = 6, COOL_AX_LOG_TE = 7 } cool_axis;

/* Kernel variants (north_star (c)).  All give the same result within the fp tolerance except
 * COOL_V_TEX_HWFILTER, whose hardware filter uses 8-bit fixed-point weights (reported, not
 * gated), and COOL_V_ANALYTIC, which ignores the table values and evaluates eqs 1-12. */
typedef enum {
    COOL_V_AUTO = 0,         /* library picks: SMEM if the table fits, else GLOBAL          */
    COOL_V_TEX_POINT = 1,    /* cudaTextureObject point fetches + software weights          */
    COOL_V_TEX_HWFILTER = 2, /* hardware-filtered texture (linear filter mode)              */
    COOL_V_SMEM = 3,         /* table staged in shared memory (<= ~200 KB)                  */
    COOL_V_GLOBAL = 4,       /* L2-resident global-memory gathers through the read-only path */
    COOL_V_ANALYTIC = 5      /* eqs 1-12 evaluated per cell, no table                       */
} cool_variant;

typedef enum { COOL_COULOMB_AUTO = 0, /* coefficient table if the cool_table has one, else analytic */
               COOL_COULOMB_OFF = 1, COOL_COULOMB_TABLE = 2, COOL_COULOMB_ANALYTIC = 3 } cool_coulomb_mode;

/* Time integration of the radiative sink: (i) explicit with the 30 % limiter, or (ii) implicit.
 * The paper gives no equations for (ii); the implicit scheme here is backward Euler per sub-step (reading
 * C-18): Theta_e' solves  th - Theta_e + h th Lambda(th_c)/u_e(th_c) - q (Theta_i - th) = 0  with th_c = th clamped to
 * the table's Theta_e range, q = a/(1 + a g), a = h K C(Theta_e, Theta_i) (Coulomb coefficient at the start state,
 * driving difference at the end state), Theta_i' = Theta_i - g q (Theta_i - Theta_e').  No limiter (f_limit is
 * ignored); always positive.  fp64 cells are solved in fp64; fp32 cells by an fp32 search on the library's log2 tables, with
 * the rate's exponent summed in fp64 inside the bracketing interval where the cell radiates more than 3 % of its energy
 * (which is what holds 1e-5).  Variants: GLOBAL, SMEM, TEX_POINT (AUTO picks);
 * TEX_HWFILTER and ANALYTIC return COOL_EUNSUPPORTED. */
typedef enum { COOL_SCHEME_EXPLICIT = 0, COOL_SCHEME_IMPLICIT = 1 } cool_scheme;

/* Unit system and fixed parameters of the physics (Table I). */
typedef struct {
    double rho_scale_cgs;        /* g cm^-3 per code density unit (Table I)                      */
    double mbh_msun;             /* black-hole mass in solar masses (L220: 10)                   */
    double gamma_e, gamma_i;     /* adiabatic indices (L207: 5/3)                                */
    double ln_lambda;            /* Coulomb logarithm (L147: 20)                                 */
    double ion_theta_mass_ratio; /* theta_i used inside eq 15 = Theta_i / this; 1 = as printed   */
    double hth_cm;               /* H_th [cm] for tables without a Theta_i axis                  */
    double r_ref_rg, spin;       /* radius [r_g] and spin for H_th = c_s/Omega_K (eqs 13-14)     */
} cool_units;

/* A cooling table as data.  Two shapes are supported:
 *   ndim = 3, nproc = 1 : axes are a permutation of {LOG_RHO, LOG_THETA_E, LOG_BSQ};
 *                         host_data[0] = log10 Lambda_code (total rate at H_th = units.hth_cm)
 *   ndim = 4, nproc = 3 : axes are a permutation of all four; host_data[0..2] =
 *                         log10 Q_brem_code, log10 Q_syn_code, log10 eta_compton; H_th from
 *                         eqs 13-14 at r_ref with the cell's Theta_e + Theta_i
 *   ndim = 4, nproc = 1 : THE PAPER'S TABLE (L122-L124, L155-L159): axis[] = {LOG_HTH, LOG_B, LOG_NE, LOG_TE} in this
 *                         order (T_e fastest, as the paper flattens it); host_data[0] = log10 Q_total[erg cm^-3 s^-1].  The
 *                         step forms the four parameters of every cell itself (L181): H_th = c_s/Omega_K from eqs 13-14
 *                         with the cell's own radius cool_cells.r (r_ref_rg when r is NULL), B = sqrt(4 pi bsq rho_scale c^2),
 *                         n_e = rho rho_scale/m_p, T_e = Theta_e m_e c^2/k_B, and converts the tabulated rate to code units.
 *                         Optional Coulomb table host_coulomb3 = log10 [Q_cc/(T_i - T_e)] over (log10 n_e, log10 T_i[K],
 *                         log10 T_e[K]), T_e fastest (L147; per kelvin, so that it is smooth through T_i = T_e).  Variants:
 *                         GLOBAL, TEX_POINT, TEX_HWFILTER (the paper's scheme: hardware bilinear on (H_th, B), manual
 *                         interpolation on the flattened (n_e, T_e) axis), ANALYTIC; explicit scheme only.
 * nproc = 0 (no data) is allowed: only COOL_V_ANALYTIC can then be applied.
 * Arrays are row-major with axis[ndim-1] fastest, n[0]*...*n[ndim-1] floats each, node k of
 * axis a at log10-coordinate lo[a] + k (hi[a]-lo[a])/(n[a]-1); n[a] >= 2, hi[a] > lo[a].
 * host_coulomb (optional, may be NULL) = log10 C(Theta_i, Theta_e), nc[0] x nc[1] floats,
 * Theta_e fastest, where Q_cc = pref rho^2 (Theta_i - Theta_e) C (eq 15). */
typedef struct {
    int ndim;
    int axis[4];                 /* cool_axis values */
    int n[4];
    double lo[4], hi[4];
    int nproc;
    const float *host_data[3];   /* HOST pointers; copied by cool_table_create */
    const float *host_coulomb;   /* HOST pointer or NULL */
    int nc[2];
    double clo[2], chi[2];
    cool_units units;
    /* the paper's Coulomb table (ndim = 4, nproc = 1 tables only; HOST pointer or NULL): nc3[0] x nc3[1] x nc3[2] floats */
    const float *host_coulomb3;
    int nc3[3];
    double c3lo[3], c3hi[3];
} cool_table_desc;

/* One batch of cells, structure of arrays, ncell contiguous elements of `dtype` each.
 * cool_apply: DEVICE pointers.  cool_apply_host: HOST pointers (pinned memory makes the
 * copies asynchronous).  theta_*_out may alias theta_*_in.  The caller owns all of them;
 * the library never frees or keeps them.  16-byte alignment enables 128-bit accesses;
 * other alignments are accepted and take a scalar path. */
typedef struct {
    long long ncell;
    cool_dtype dtype;
    const void *rho, *bsq;                     /* read-only */
    const void *theta_e_in, *theta_i_in;       /* read-only unless aliased by the outputs */
    void *theta_e_out, *theta_i_out;
    const void *r;                             /* optional radius [r_g] per cell; NULL: no floor */
    const void *vol;                           /* optional sqrt(-g) dV weights; NULL: 1 */
    /* Optional radial luminosity profile (numerator of eq 25): cells are grouped into consecutive shells of
     * shell_cells cells (all (theta, phi) cells of one radial index when phi is fastest); lum_shell receives
     * 4 doubles per shell, [shell][total, brems, synch, compton] = sum over the shell of dE vol/dt (overwritten).
     * lum_shell is a DEVICE array for cool_apply and a HOST array for cool_apply_host, of 4 ceil(ncell/shell_cells)
     * doubles; NULL: no profile.  shell_cells must be a positive multiple of 128 and the call must also ask for the
     * diagnostics (d_diag / h_diag != NULL).  The shell sums are accumulated with fp64 atomics (order dependent in the
     * last bits); their total equals cool_diag.lum_* to rounding. */
    long long shell_cells;
    double *lum_shell;
    /* Optional per-cell event flags, one byte per cell (overwritten): bit 0 = the 30 % limiter capped the radiative loss in
     * some sub-step (L185), bit 1 = the temperature floor switched cooling off (eq 19), bit 2 = a table coordinate was
     * clamped (C-7), bit 3 = the cell was recomputed by the precise pass (fp32 cells whose Theta_e visits a table interval
     * too steep for fp32 coordinates, e.g. the K2 -> 2 theta^2 switch of L87).  Bits 0-2 are the per-cell
     * terms of cool_diag.n_limited / n_floored / n_clamped.  DEVICE array for cool_apply, HOST array for cool_apply_host;
     * NULL: not wanted.  Needs the diagnostics (d_diag / h_diag != NULL); 4-byte alignment enables 32-bit stores. */
    unsigned char *flags;
} cool_cells;

typedef struct {
    double dt;                   /* fluid-frame time step [r_g/c], > 0 */
    int nsub;                    /* >= 1 equal sub-steps */
    double f_limit;              /* 0 < f_limit < 0.5; the paper uses 0.3 (L185) */
    double h_floor;              /* (H/R)_floor of eq 19; 0 = off; needs cells.r */
    cool_variant variant;
    cool_coulomb_mode coulomb;
    cool_scheme scheme;          /* COOL_SCHEME_EXPLICIT (0) or COOL_SCHEME_IMPLICIT */
} cool_params;

/* Diagnostics of one call (sums over the cells of the call; overwritten, not accumulated).
 * lum_* = sum dE vol/dt, split by the shares of Q_thin (brems, synch, Compton-added) when
 * nproc = 3, zero otherwise.  n_* count cells in which the event happened in any sub-step. */
typedef struct {
    double lum_total, lum_brems, lum_synch, lum_compton;
    long long n_limited, n_floored, n_clamped;
} cool_diag;

typedef struct cool_table cool_table;      /* opaque */

/* Host table builder (north_star (a)): tabulates eqs 1-12 (and eq 15's coefficient C when
 * out_coulomb != NULL) on the grid that `shape` describes (its host_data / host_coulomb
 * pointers are ignored).  out[p] must hold prod(n) floats for p < nproc; out_coulomb
 * nc[0]*nc[1] floats — for the paper's table (axes LOG_HTH, LOG_B, LOG_NE, LOG_TE) nc3[0]*nc3[1]*nc3[2] floats of
 * log10 [Q_cc/(T_i - T_e)].  Runs on `nthreads` host threads (<= 0: all available).  Host only;
 * needs no GPU.  Errors: COOL_EINVAL for a malformed shape. */
cool_status cool_table_build_host(const cool_table_desc *shape, float *const out[3], float *out_coulomb, int nthreads);

/* The same tabulation on a CUDA device, for the paper's table only (axes LOG_HTH, LOG_B, LOG_NE, LOG_TE; nproc = 1):
 * 100^4 nodes (L124) take the host builder minutes and the device a second.  host_out: HOST array of prod(n) floats
 * (log10 Q_total[erg cm^-3 s^-1]).  Synchronous.  Errors: COOL_EINVAL, COOL_EUNSUPPORTED (another shape), COOL_ENOMEM,
 * COOL_ECUDA (no usable device). */
cool_status cool_table_build_device(const cool_table_desc *shape, int device, float *host_out);

/* Uploads a table to `device` and prepares every device representation (linear arrays,
 * cudaArray + texture objects, the shared-memory image).  Host arrays are copied; the
 * caller may free them on return.  *out is owned by the library until cool_table_destroy.
 * Errors: COOL_EINVAL (shape, NULL, non-finite values), COOL_ENOMEM, COOL_ECUDA. */
cool_status cool_table_create(const cool_table_desc *desc, int device, cool_table **out);

/* One cooling + Coulomb update of all cells, asynchronous on `cuda_stream` (a cudaStream_t;
 * NULL = the default stream).  Does not synchronise.  Safe to call concurrently on different
 * streams with the same table.  d_diag: DEVICE pointer to one cool_diag, or NULL.
 * Per-cell numerical trouble is not an error: non-positive bsq/Theta clamp to the lower
 * table edge, rho <= 0 leaves the cell unchanged, NaN inputs give NaN outputs for that
 * cell only.  Errors: COOL_EINVAL (NULL/negative sizes/params out of range),
 * COOL_EUNSUPPORTED (variant impossible for this table, e.g. SMEM with a table that does not
 * fit; COOL_V_AUTO never fails this way), COOL_ECUDA.
 * Launches: one kernel; two for fp32 cells in a sub-stepped or 4-D step on a table with a steep Theta_e interval (the K2 -> 2 theta^2
 * switch of PAPER.md L87): the fp32 kernel passes the few cells that visit it through and a small second kernel recomputes them
 * in fp64, which is what holds 1e-5 on every cell; one more when cells->lum_shell is set.  The library keeps a small per-stream
 * workspace for this (allocated on the first call on a stream; cool_apply_noalloc below never allocates). */
cool_status cool_apply(const cool_table *table, const cool_cells *cells, const cool_params *params,
                       cool_diag *d_diag, void *cuda_stream);

/* Same update for HOST arrays: the library stages chunks through device memory it owns,
 * overlapping host->device copies, kernels and device->host copies on internal streams, and
 * returns after the outputs (and *h_diag, if not NULL) are complete in host memory. */
cool_status cool_apply_host(const cool_table *table, const cool_cells *host_cells, const cool_params *params,
                            cool_diag *h_diag);

/* cool_apply for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
 * Same arguments, same kernels, same results as cool_apply (DEVICE arrays, asynchronous on `cuda_stream`), but the scratch
 * memory the step needs — the per-block partial sums and the ticket of the luminosity diagnostic (eq 22), and the work lists
 * of the precise pass — lives in ONE file-scope device array of COOL_NOALLOC_SCRATCH_BYTES that every GPU which loads the
 * library holds until the process exits.  The call runs no cudaMalloc, cudaFree or allocating library routine.
 * Limits: cells->ncell <= COOL_NOALLOC_MAX_CELLS and no radial profile (cells->lum_shell must be NULL); beyond them the call
 * returns COOL_EINVAL / COOL_EUNSUPPORTED with a message in cool_last_error() and launches nothing.
 * Sharing: every call on a device uses the same array, whatever the table or the stream, and the array keeps the last call's
 * contents (the call clears what must start at zero, on `cuda_stream`).  Calls that overlap on the GPU — different streams
 * without an ordering between them — RACE on it: order them (one stream, or events), or use cool_apply.
 * The first call on a device resolves the array's device address (cudaGetSymbolAddress); make that call — ncell = 0 will
 * do — before starting a graph capture. */
#define COOL_NOALLOC_MAX_CELLS (1ll << 24)
#define COOL_NOALLOC_SCRATCH_BYTES (4u << 20)
cool_status cool_apply_noalloc(const cool_table *table, const cool_cells *cells, const cool_params *params,
                               cool_diag *d_diag, void *cuda_stream);

/* Which variant COOL_V_AUTO resolves to for this table (always a concrete variant). */
cool_variant cool_table_auto_variant(const cool_table *table);

/* Number of kernel launches the last cool_apply / cool_apply_host on this thread issued. */
int cool_last_launch_count(void);

/* Name of the step kernel instantiation the last cool_apply / cool_apply_host on this thread launched (the dispatcher's own
 * choice of lookup policy, Coulomb staging, thread count), e.g. "cool_f32_kernel<MODE=3,F32GlobalQ,DIAG=0,CM=1,NSUB1=1,768x2>".
 * Thread-local, never NULL ("" before the first launch). */
const char *cool_last_kernel_name(void);

cool_status cool_table_destroy(cool_table *table);

/* Radiation-pressure temperature correction (eq 29; post-processing of the high-accretion-rate
 * runs, Figs 9(b) and 10).  Eq 29, P = a T_e^4 + N k_B (T_e + T_i), with P the simulated gas pressure
 * N k_B (T_e + T_i) and only T_e recalculated (L345: T_i cancels), is  a T^4 + N k_B (T - T_e) = 0; its one root in
 * (0, T_e] replaces Theta_e in every cell whose in-cell scattering depth tau_sca = n_e sigma_T H (L353) exceeds
 * tau_crit (the paper uses 1 for Fig. 9(b) and 4.6 for Fig. 10).  a = 7.5646e-15 erg cm^-3 K^-4 as printed (L345),
 * N = n_e = rho rho_scale_cgs/m_p.  Other cells, and cells with rho <= 0, Theta_e <= 0 or NaN, are copied unchanged.
 * Only units->rho_scale_cgs and units->mbh_msun are used; no table is needed.
 * d_rho, d_theta_e, d_hscale (scale height H of the cell's radius, in r_g), d_theta_e_out: DEVICE arrays of ncell
 * elements of `dtype` on the CURRENT device, owned by the caller; d_theta_e_out may alias d_theta_e; 16-byte
 * alignment of all four enables 128-bit accesses, other alignments take a scalar path.  d_ncorrected: DEVICE pointer
 * to one long long that receives the number of corrected cells (overwritten), or NULL.  Asynchronous on
 * `cuda_stream`; does not synchronise.  One kernel launch.  Errors: COOL_EINVAL (NULL arrays with ncell > 0, ncell < 0,
 * tau_crit < 0 or not finite, non-positive units), COOL_ECUDA. */
cool_status cool_radpress_correct(const cool_units *units, long long ncell, cool_dtype dtype, const void *d_rho,
                                  const void *d_theta_e, const void *d_hscale, double tau_crit, void *d_theta_e_out,
                                  long long *d_ncorrected, void *cuda_stream);

const char *cool_last_error(void);         /* thread-local, never NULL */
const char *cool_version(void);

#ifdef __cplusplus
}
#endif
#endif /* COOL_H */
