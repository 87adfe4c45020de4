/*
 * cool_oracle.c — ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, fp64 CPU statement of the per-cell two-temperature cooling step of
 * arXiv 2505.08855 (reference text: PAPER.md).  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code,
 * header, table or constant generator with paper_2505_08855_b200/ (the CUDA product).
 *
 * Part A  analytic physics, §II eqs 1-15 (L57-L147)
 * Part B  the table-interpolated, limited, sub-stepped update (PAPER.md L122-L124,
 *         L181, L185, L197; readings C-1..C-17 of SURVEY.md §8(c) / DESIGN.md)
 * Part B' the implicit scheme (L185 (ii), L369; reading C-18)
 * Part C  the radiation-pressure temperature correction (eq 29; reading C-20)
 * Part D  the paper's own table (L122-L124): Q(H_th, B, n_e, T_e) in cgs units with H_th per cell from
 *         eqs 13-14 and the cell's radius (L128-L136), Coulomb table Q_cc(n_e, T_i, T_e) (readings C-22, C-23);
 *         it is Part B with four more axis kinds, so the same orc_step_cell runs it
 *
 * Pins (tests/test_oracle_*.py): closed-form brems scaling, incomplete-gamma closed
 * form of the synchrotron integral, scipy.special.kve for the Bessel functions,
 * residual of eq 5, limits of eqs 7 and 11, node-exact / linear-exact interpolation,
 * conservation / positivity / no-crossing of the update, brute force on tiny tables;
 * Part C: manufactured roots of eq 29, mpmath roots of the unreduced quartic, both limits.
 * Nothing here is "parity unpinned".
 *
 * Everything is double precision; no blocking, fusion or reordering beyond what the
 * equations state.
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- CODATA-2018 constants, cgs ------------------------------------------------ */
#define ORC_C      2.99792458e10      /* cm/s  */
#define ORC_KB     1.380649e-16       /* erg/K */
#define ORC_ME     9.1093837015e-28   /* g     */
#define ORC_MP     1.67262192369e-24  /* g     */
#define ORC_QE     4.80320471257e-10  /* esu   */
#define ORC_HPL    6.62607015e-27     /* erg s */
#define ORC_SIGT   6.6524587321e-25   /* cm^2  */
#define ORC_SIGSB  5.670374419e-5     /* erg cm^-2 s^-1 K^-4 */
#define ORC_GMSUN  1.32712440018e26   /* cm^3/s^2 */
#define ORC_PI     3.14159265358979323846

/* Unit system of the caller (SURVEY §8 conventions; PAPER.md L220 M = 10 Msun,
 * Table I L287-L296 rho_scale, L207 gamma = 5/3, a = 0.9375). */
typedef struct {
    double rho_scale_cgs;        /* g cm^-3 per code density unit              */
    double mbh_msun;             /* black-hole mass                            */
    double gamma_e, gamma_i;     /* adiabatic indices                          */
    double ln_lambda;            /* Coulomb logarithm, C-4: 20                 */
    double ion_theta_mass_ratio; /* C-3: theta_i(eq 15) = Theta_i / this       */
    double hth_cm;               /* C-6: fixed H_th for 3-D tables             */
    double r_ref_rg, spin;       /* C-6: radius/spin for H_th in 4-D tables    */
} orc_units;

static double orc_rg(const orc_units *u) { return ORC_GMSUN * u->mbh_msun / (ORC_C * ORC_C); }
static double orc_tg(const orc_units *u) { return orc_rg(u) / ORC_C; }
/* erg cm^-3 s^-1  ->  code energy density per code time */
static double orc_rate_conv(const orc_units *u) { return orc_tg(u) / (u->rho_scale_cgs * ORC_C * ORC_C); }

double orc_ne_cgs(const orc_units *u, double rho) { return rho * u->rho_scale_cgs / ORC_MP; }   /* C-14 */
double orc_bfield_gauss(const orc_units *u, double bsq)                                         /* L173 */
{
    return sqrt(4.0 * ORC_PI * bsq * u->rho_scale_cgs * ORC_C * ORC_C);
}

/* ================================================================================
 * Part A.1  Bremsstrahlung, eqs 1-2.
 * ============================================================================== */
double orc_brems_cgs(double ne, double th)
{
    double fee, fei;
    if (th < 1.0) {
        fee = pow(th, 1.5) * (1.0 + 1.1 * th + th * th - 1.25 * pow(th, 2.5));
        fei = 4.0 * sqrt(2.0 * th / (ORC_PI * ORC_PI * ORC_PI)) * (1.0 + 1.781 * pow(th, 1.34));
    } else {
        fee = 1.34 * th * (log(1.123 * th) + 1.28);
        fei = 9.0 * th / (2.0 * ORC_PI) * (log(1.123 * th + 0.48) + 1.5);
    }
    return 2.56e-22 * ne * ne * fee + 1.48e-22 * ne * ne * fei;
}

/* ================================================================================
 * Modified Bessel functions of the second kind, exponentially scaled:
 *   Khat_nu(x) = e^x K_nu(x) = int_0^inf exp(-x (cosh t - 1)) cosh(nu t) dt
 * (textbook integral representation).  Trapezoid rule, which
 * converges geometrically for this analytic, doubly-exponentially decaying
 * integrand.  The upper limit is where the exponent reaches -80.
 * ============================================================================== */
double orc_bessel_k_scaled(double nu, double x)
{
    /* cosh t - 1 = 2 sinh^2(t/2) is used so that large x (tiny t) keeps full precision */
    const int N = 256;
    const double tmax = 2.0 * asinh(sqrt(40.0 / x));   /* x (cosh tmax - 1) = 80 */
    const double h = tmax / N;
    double s = 0.5; /* f(0)/2 = 1/2 */
    for (int k = 1; k <= N; ++k) {
        double t = k * h;
        double sh = sinh(0.5 * t);
        s += exp(-2.0 * x * sh * sh) * cosh(nu * t);
    }
    return s * h;
}
/* K2 from the recurrence K_{n+1} = K_{n-1} + (2n/x) K_n (holds for the scaled form). */
double orc_bessel_k2_scaled(double x)
{
    return orc_bessel_k_scaled(0.0, x) + (2.0 / x) * orc_bessel_k_scaled(1.0, x);
}

/* ================================================================================
 * Part A.2  Synchrotron, eqs 3-6.
 * ============================================================================== */
/* ln I'(x) at x = e^u, eq 4 (L76). */
static double orc_ln_iprime(double u)
{
    return log(4.0505) - u / 6.0 + log(1.0 + 0.4 * exp(-0.25 * u) + 0.5316 * exp(-0.5 * u))
           - 1.8899 * exp(u / 3.0);
}
double orc_iprime(double x) { return exp(orc_ln_iprime(log(x))); }

/* K2(1/theta_e), with the paper's low-temperature substitution 2 theta_e^2 for
 * T_e <= 1e8 K (L87, reading C-12: literal threshold). */
double orc_k2_tilde(double th)
{
    double te = th * ORC_ME * ORC_C * ORC_C / ORC_KB;
    if (te > 1.0e8) {
        double x = 1.0 / th;
        return orc_bessel_k2_scaled(x) * exp(-x);
    }
    return 2.0 * th * th;
}

/* nu = s * x_M  (inverse of x_M = 4 pi m_e c nu / (3 e B theta_e^2), L74). */
static double orc_synch_s(double B, double th)
{
    return 3.0 * ORC_QE * B * th * th / (4.0 * ORC_PI * ORC_ME * ORC_C);
}

/* x_c = x_M(nu_c): root of eq 5 (L80), H eps_s(nu_c) = 2 pi nu_c^2 k_B T_e / c^2,
 * i.e. I'(x)/x = s theta_e m_e K2tilde / (2*4.43e-30 H n_e).  Bisection in u = ln x
 * (reading C-11: "numerical integration" = numerical root finding).  The left side
 * decreases monotonically from +inf to 0, so the root is unique. */
double orc_synch_xc(double H, double B, double ne, double th)
{
    double s = orc_synch_s(B, th);
    double lnR = log(s) + log(th) + log(ORC_ME) + log(orc_k2_tilde(th)) - log(2.0 * 4.43e-30 * H * ne);
    double a = -1200.0, b = 90.0; /* ln x bracket */
    for (int it = 0; it < 200; ++it) {
        double m = 0.5 * (a + b);
        double g = orc_ln_iprime(m) - m - lnR;
        if (g > 0.0) a = m; else b = m;
    }
    return exp(0.5 * (a + b));
}

/* 16-point Gauss-Legendre nodes by Newton iteration on P_16 (textbook). */
static void orc_gauss_legendre16(double *xn, double *wn)
{
    const int n = 16;
    for (int i = 0; i < n; ++i) {
        double z = cos(ORC_PI * (i + 0.75) / (n + 0.5)), pp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 1; j <= n; ++j) {
                double p3 = p2; p2 = p1;
                p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j;
            }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            double dz = p1 / pp;
            z -= dz;
            if (fabs(dz) < 1e-16) break;
        }
        xn[i] = z;
        wn[i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

/* J(x_c) = int_{x_c}^inf x I'(x) dx, composite Gauss-Legendre in u = ln x
 * (integrand x^2 I'(x) du).  Upper limit where exp(-1.8899 x^{1/3}) has fallen by
 * e^-80 from its value at x_c. */
double orc_synch_J(double xc)
{
    double xn[16], wn[16];
    orc_gauss_legendre16(xn, wn);
    double uc = log(xc);
    double tc = 1.8899 * cbrt(xc);
    double umax = 3.0 * log((tc + 80.0) / 1.8899);
    if (umax <= uc) return 0.0;
    int npanel = (int)ceil((umax - uc) / 0.5);
    double hw = (umax - uc) / npanel;
    double sum = 0.0;
    for (int p = 0; p < npanel; ++p) {
        double c = uc + (p + 0.5) * hw;
        for (int i = 0; i < 16; ++i) {
            double u = c + 0.5 * hw * xn[i];
            sum += wn[i] * exp(2.0 * u + orc_ln_iprime(u));
        }
    }
    return sum * 0.5 * hw;
}

/* Q_syn of eq 6 (L84): Rayleigh-Jeans part below nu_c (prefactor 2piR^2/(2H piR^2) = 1/H)
 * plus optically thin part above nu_c.  Returns erg cm^-3 s^-1; *nu_c_out = nu_c [Hz]. */
double orc_synch_cgs(double H, double B, double ne, double th, double *nu_c_out)
{
    double s = orc_synch_s(B, th);
    double xc = orc_synch_xc(H, B, ne, th);
    double nuc = s * xc;
    double te = th * ORC_ME * ORC_C * ORC_C / ORC_KB;
    double rj = 2.0 * ORC_PI * ORC_KB * te * nuc * nuc * nuc / (3.0 * ORC_C * ORC_C * H);
    double thin = 4.43e-30 * 4.0 * ORC_PI * ne * s * s * orc_synch_J(xc) / orc_k2_tilde(th);
    if (nu_c_out) *nu_c_out = nuc;
    return rj + thin;
}

/* ================================================================================
 * Part A.3  Inverse-Compton enhancement, eqs 7-9.
 * Reading C-1: exponent -1 - ln P / ln A (series sum); the printed "1 - lnP/lnA"
 * is available with printed_exponent != 0 for comparison only.
 * ============================================================================== */
double orc_compton_eta_ex(double nu_c, double ne, double H, double th, int printed_exponent)
{
    double x = ORC_HPL * nu_c / (ORC_ME * ORC_C * ORC_C);    /* E_init / m_e c^2 */
    if (!(x < 3.0 * th)) return 1.0;                         /* L99: soft photons only */
    double tau = 2.0 * ne * ORC_SIGT * H;
    double P = -expm1(-tau);
    if (!(P > 0.0)) return 1.0;
    double Am1 = 4.0 * th + 16.0 * th * th;
    double A = 1.0 + Am1;
    double lnA = log1p(Am1);
    double PA = P * A;
    if (fabs(1.0 - PA) < 1e-8)
        return 1.0 + P * Am1 * log(3.0 * th / x) / lnA;
    double expo = (printed_exponent ? 1.0 : -1.0) - log(P) / lnA;
    return 1.0 + P * Am1 / (1.0 - PA) * (1.0 - pow(x / (3.0 * th), expo));
}
double orc_compton_eta(double nu_c, double ne, double H, double th)
{
    return orc_compton_eta_ex(nu_c, ne, H, th, 0);
}

/* ================================================================================
 * Part A.4  Totals, eqs 10-12 (reading C-2: sigma = Stefan-
 * Boltzmann, tau_obs = tau_abs).
 * ============================================================================== */
double orc_bridge_cgs(double H, double ne, double th, double qthin)
{
    double te = th * ORC_ME * ORC_C * ORC_C / ORC_KB;
    double bb = 4.0 * ORC_SIGSB * te * te * te * te;
    double tau_sca = 2.0 * ne * ORC_SIGT * H;
    double tau_abs = H * qthin / bb;
    return (bb / H) / (1.5 * (tau_abs + tau_sca) + sqrt(3.0) + 1.0 / tau_abs);
}
/* out[0]=Q_brem, out[1]=Q_syn, out[2]=eta, out[3]=Q_thin, out[4]=Q_total, out[5]=nu_c */
void orc_cooling_cgs(double H, double B, double ne, double th, double *out)
{
    double nuc;
    double qbr = orc_brems_cgs(ne, th);
    double qsy = orc_synch_cgs(H, B, ne, th, &nuc);
    double eta = orc_compton_eta(nuc, ne, H, th);
    double qthin = qbr + eta * qsy;
    out[0] = qbr; out[1] = qsy; out[2] = eta; out[3] = qthin;
    out[4] = orc_bridge_cgs(H, ne, th, qthin);
    out[5] = nuc;
}

/* ================================================================================
 * Part A.5  Scale height, eqs 13-14 (code units c = 1, lengths
 * r_g).  P_s = rho Theta_s m_e/m_p (Theta_i defined with m_e, L147 / C-3),
 * u_s = P_s/(gamma_s - 1); rho h = rho + u + P; gamma P -> gamma_e P_e + gamma_i P_i
 * (equal to eq 14 when gamma_e = gamma_i).  rho cancels.
 * ============================================================================== */
double orc_omega_k(double r_rg, double spin) { return 1.0 / (pow(r_rg, 1.5) + spin); }
double orc_hth_cm(const orc_units *u, double th_e, double th_i, double r_rg)
{
    double mr = ORC_ME / ORC_MP;
    double pe = th_e * mr, pi = th_i * mr;
    double cs2 = (u->gamma_e * pe + u->gamma_i * pi) /
                 (1.0 + pe / (u->gamma_e - 1.0) + pi / (u->gamma_i - 1.0) + pe + pi);
    return orc_rg(u) * sqrt(cs2) / orc_omega_k(r_rg, u->spin);
}

/* ================================================================================
 * Part A.6  Coulomb exchange, eq 15.  With scaled Bessel
 * functions the exponentials cancel identically because 1/theta_m = 1/theta_e +
 * 1/theta_i.  C(theta_e, theta_i) is the Bessel bracket / [K2 K2].
 * ============================================================================== */
double orc_coulomb_C(double th_e, double th_i)
{
    double xe = 1.0 / th_e, xi = 1.0 / th_i, xm = xe + xi;
    double s = th_e + th_i;
    double num = (2.0 * s * s + 1.0) / s * orc_bessel_k_scaled(1.0, xm) + 2.0 * orc_bessel_k_scaled(0.0, xm);
    return num / (orc_bessel_k2_scaled(xe) * orc_bessel_k2_scaled(xi));
}
/* erg cm^-3 s^-1 per unit rho_code^2 (Theta_i - Theta_e) C :
 * (3/2)(m_e/m_p) lnLambda c sigma_T m_e c^2 (rho_scale/m_p)^2 ; k_B(T_i-T_e) = m_e c^2 (Theta_i-Theta_e). */
double orc_coulomb_pref_cgs(const orc_units *u)
{
    double n1 = u->rho_scale_cgs / ORC_MP;
    return 1.5 * (ORC_ME / ORC_MP) * u->ln_lambda * ORC_C * ORC_SIGT * ORC_ME * ORC_C * ORC_C * n1 * n1;
}
/* Q_cc in code units; > 0 heats the electrons. */
double orc_coulomb_code(const orc_units *u, double rho, double th_e, double th_i)
{
    double C = orc_coulomb_C(th_e, th_i / u->ion_theta_mass_ratio);
    return orc_coulomb_pref_cgs(u) * orc_rate_conv(u) * rho * rho * (th_i - th_e) * C;
}

/* ================================================================================
 * Table nodes (what a cooling table stores; reading C-5: log10 of the code-unit
 * rate, eta stored as log10 eta).
 * ============================================================================== */
/* 3-D table (log rho, log Theta_e, log bsq) at fixed H = hth_cm: log10 Lambda_code. */
double orc_node_total_log10(const orc_units *u, double rho, double th_e, double bsq)
{
    double out[6];
    orc_cooling_cgs(u->hth_cm, orc_bfield_gauss(u, bsq), orc_ne_cgs(u, rho), th_e, out);
    return log10(out[4] * orc_rate_conv(u));
}
/* 4-D process tables (log rho, log Theta_e, log bsq, log Theta_i), H from eqs 13-14
 * at r_ref: out = {log10 Qbrem_code, log10 Qsyn_code, log10 eta}. */
void orc_node_proc_log10(const orc_units *u, double rho, double th_e, double bsq, double th_i, double *out3)
{
    double out[6];
    double H = orc_hth_cm(u, th_e, th_i, u->r_ref_rg);
    orc_cooling_cgs(H, orc_bfield_gauss(u, bsq), orc_ne_cgs(u, rho), th_e, out);
    out3[0] = log10(out[0] * orc_rate_conv(u));
    out3[1] = log10(out[1] * orc_rate_conv(u));
    out3[2] = log10(out[2]);
}

/* Combine per-process code-unit rates into Q_total (code units), eqs 10-12, with the
 * cell's own H (eqs 13-14 at r_ref).  frac3 (optional) = shares of Q_thin:
 * brems, synchrotron, Compton-added. */
double orc_combine_code(const orc_units *u, double rho, double th_e, double th_i,
                        double qbr, double qsy, double eta, double *frac3)
{
    double conv = orc_rate_conv(u);
    double H = orc_hth_cm(u, th_e, th_i, u->r_ref_rg);
    double qthin = qbr + eta * qsy;
    if (frac3) { frac3[0] = qbr / qthin; frac3[1] = qsy / qthin; frac3[2] = (eta - 1.0) * qsy / qthin; }
    return orc_bridge_cgs(H, orc_ne_cgs(u, rho), th_e, qthin / conv) * conv;
}

/* ================================================================================
 * Part B  the step.
 * ============================================================================== */
enum { ORC_AX_LOG_RHO = 0, ORC_AX_LOG_THETA_E = 1, ORC_AX_LOG_BSQ = 2, ORC_AX_LOG_THETA_I = 3,
       /* Part D, the paper's parameters in cgs units (L122-L124): */
       ORC_AX_LOG_HTH = 4, ORC_AX_LOG_B = 5, ORC_AX_LOG_NE = 6, ORC_AX_LOG_TE = 7,
       ORC_AX_LOG_TI = 8 /* Coulomb table only (L147) */ };

typedef struct {
    int ndim;               /* 3 or 4 (any 1..4 works)                              */
    int axis[4];            /* which primitive each table axis is the log10 of      */
    int n[4];               /* nodes per axis                                       */
    double lo[4], hi[4];    /* log10 bounds, node-centred                           */
    int nproc;              /* 1: total Lambda; 3: brems, synch, eta                */
    const float *data[3];   /* row-major, axis[ndim-1] fastest, log10 values        */
    const float *coul;      /* optional log10 C over (log Theta_i, log Theta_e)     */
    int nc[2];
    double clo[2], chi[2];
    /* Part D: */
    int cgs;                /* 1: data[0] holds log10 Q_total in erg cm^-3 s^-1 (the paper's table) */
    const float *coul3;     /* optional log10 [Q_cc / (T_i - T_e)] in erg cm^-3 s^-1 K^-1 over (log n_e, log T_i[K], log T_e[K]), T_e fastest (L147, C-23) */
    int nc3[3];
    double c3lo[3], c3hi[3];
} orc_table;

/* B1: coordinate -> (i, w) with edge clamping (C-7).  Returns 1 if clamped. */
static int orc_locate(double x, double lo, double hi, int n, int *i, double *w)
{
    double delta = (hi - lo) / (n - 1);
    double t = (x - lo) / delta;
    int clamped = 0;
    if (t < 0.0) { t = 0.0; clamped = 1; }
    if (t > (double)(n - 1)) { t = (double)(n - 1); clamped = 1; }
    int ii = (int)floor(t);
    if (ii > n - 2) ii = n - 2;
    *i = ii; *w = t - ii;
    return clamped;
}

/* B2: multilinear interpolation, y = sum over the 2^ndim corners of prod(w) * T. */
double orc_interp(int ndim, const int *n, const double *lo, const double *hi,
                  const float *T, const double *x, int *clamped)
{
    int i[4]; double w[4]; int cl = 0;
    for (int k = 0; k < ndim; ++k) {
        if (isnan(x[k])) { if (clamped) *clamped = 0; return NAN; }
        cl |= orc_locate(x[k], lo[k], hi[k], n[k], &i[k], &w[k]);
    }
    if (clamped) *clamped = cl;
    double y = 0.0;
    for (int c = 0; c < (1 << ndim); ++c) {
        double pw = 1.0; size_t off = 0;
        for (int k = 0; k < ndim; ++k) {
            int bit = (c >> k) & 1;
            pw *= bit ? w[k] : (1.0 - w[k]);
            off = off * (size_t)n[k] + (size_t)(i[k] + bit);
        }
        y += pw * (double)T[off];
    }
    return y;
}

/* One cell, nsub sub-steps (reading C-10).  rate_mode 0: table, 1: analytic Part A.
 * coulomb_mode 0: off, 1: coefficient table, 2: analytic eq 15.
 * diag7: lum_total, lum_brems, lum_synch, lum_compton, limited, floored, clamped. */
static void orc_step_cell(const orc_table *tab, const orc_units *un,
                          double rho, double bsq, double *the_io, double *thi_io,
                          double r, double vol, double dt, int nsub, double f_limit, double h_floor,
                          int rate_mode, int coulomb_mode,
                          double *lam0, double *qcc0, double *diag7)
{
    const double mr = ORC_ME / ORC_MP;
    const double ge1 = un->gamma_e - 1.0, gi1 = un->gamma_i - 1.0;
    const double h = dt / nsub;
    double the = *the_io, thi = *thi_io;
    double de_sum[4] = {0, 0, 0, 0};
    int limited = 0, floored = 0, clamped = 0;

    for (int s = 0; s < nsub; ++s) {
        /* B1/B2: rate lookup */
        double prim[9];
        prim[ORC_AX_LOG_RHO] = rho; prim[ORC_AX_LOG_THETA_E] = the;
        prim[ORC_AX_LOG_BSQ] = bsq; prim[ORC_AX_LOG_THETA_I] = thi;
        /* Part D: the paper's parameters of this cell, this sub-step (L181: "the values of H_th, B, n_e and T_e obtained
         * from the simulation"); H_th = c_s/Omega_K with the cell's own radius (eqs 13-14; r <= 0: r_ref) */
        prim[ORC_AX_LOG_HTH] = orc_hth_cm(un, the, thi, r > 0.0 ? r : un->r_ref_rg);
        prim[ORC_AX_LOG_B] = orc_bfield_gauss(un, bsq > 0.0 ? bsq : 0.0);
        prim[ORC_AX_LOG_NE] = orc_ne_cgs(un, rho);
        prim[ORC_AX_LOG_TE] = the * ORC_ME * ORC_C * ORC_C / ORC_KB;
        prim[ORC_AX_LOG_TI] = thi * ORC_ME * ORC_C * ORC_C / ORC_KB;
        double lam, frac[3] = {0, 0, 0};
        if (rate_mode == 0) {
            double x[4]; int cl = 0;
            for (int k = 0; k < tab->ndim; ++k) {       /* C-7: non-positive -> lower edge */
                double q = prim[tab->axis[k]];
                x[k] = (q > 0.0) ? log10(q) : -INFINITY;
            }
            if (tab->nproc == 1) {
                lam = pow(10.0, orc_interp(tab->ndim, tab->n, tab->lo, tab->hi, tab->data[0], x, &cl));
                if (tab->cgs) lam *= orc_rate_conv(un);         /* the paper's table is in erg cm^-3 s^-1 */
            } else {
                double q[3];
                for (int p = 0; p < 3; ++p)
                    q[p] = pow(10.0, orc_interp(tab->ndim, tab->n, tab->lo, tab->hi, tab->data[p], x, &cl));
                lam = orc_combine_code(un, rho, the, thi, q[0], q[1], q[2], frac);
            }
            clamped |= cl;
        } else {
            double out[6];
            double H = (tab->ndim == 4) ? orc_hth_cm(un, the, thi, un->r_ref_rg) : un->hth_cm;
            if (tab->cgs) H = prim[ORC_AX_LOG_HTH];
            orc_cooling_cgs(H, orc_bfield_gauss(un, bsq), orc_ne_cgs(un, rho), the, out);
            lam = out[4] * orc_rate_conv(un);
            frac[0] = out[0] / out[3]; frac[1] = out[1] / out[3]; frac[2] = (out[2] - 1.0) * out[1] / out[3];
        }
        /* B3: temperature floor, eq 19 (L195), reading C-13 */
        if (h_floor > 0.0 && r > 0.0) {
            double tfloor = 0.5 * ORC_PI * pow(h_floor * orc_omega_k(r, un->spin) * r, 2.0);
            if ((the + thi) * mr < tfloor) { lam = 0.0; floored = 1; }
        }
        /* B4: Coulomb */
        double qcc = 0.0;
        if (coulomb_mode == 1) {
            double xc[2] = { thi > 0.0 ? log10(thi) : -INFINITY, the > 0.0 ? log10(the) : -INFINITY };
            double C = pow(10.0, orc_interp(2, tab->nc, tab->clo, tab->chi, tab->coul, xc, NULL));
            qcc = orc_coulomb_pref_cgs(un) * orc_rate_conv(un) * rho * rho * (thi - the) * C;
        } else if (coulomb_mode == 2) {
            qcc = (thi == the) ? 0.0 : orc_coulomb_code(un, rho, the, thi);
        } else if (coulomb_mode == 3) {     /* Part D: the paper's Q_cc(n_e, T_i, T_e) table (L147), stored per kelvin of T_i - T_e (C-23) */
            double q3[3] = { prim[ORC_AX_LOG_NE], prim[ORC_AX_LOG_TI], prim[ORC_AX_LOG_TE] }, x3[3];
            for (int k = 0; k < 3; ++k) x3[k] = (q3[k] > 0.0) ? log10(q3[k]) : -INFINITY;
            double kq = pow(10.0, orc_interp(3, tab->nc3, tab->c3lo, tab->c3hi, tab->coul3, x3, NULL));
            qcc = kq * (prim[ORC_AX_LOG_TI] - prim[ORC_AX_LOG_TE]) * orc_rate_conv(un);
        }
        if (s == 0) { if (lam0) *lam0 = lam; if (qcc0) *qcc0 = qcc; }
        /* B5: limited explicit update (L185; readings C-8, C-9) */
        double ue = rho * the * mr / ge1, ui = rho * thi * mr / gi1;
        double de = lam * h;
        if (de > f_limit * ue) { de = f_limit * ue; limited = 1; }
        double xeq = (ui * gi1 - ue * ge1) / (ge1 + gi1);   /* transfer that equalises Theta */
        double x = fabs(qcc) * h;
        double udonor = (qcc > 0.0) ? ui : ue;
        if (x > f_limit * udonor) x = f_limit * udonor;
        if (x > fabs(xeq)) x = fabs(xeq);
        if (qcc < 0.0) x = -x;
        if (qcc == 0.0) x = 0.0;
        ue = ue - de + x;
        ui = ui - x;
        the = ue * ge1 / (mr * rho);
        thi = ui * gi1 / (mr * rho);
        de_sum[0] += de;
        de_sum[1] += de * frac[0]; de_sum[2] += de * frac[1]; de_sum[3] += de * frac[2];
    }
    *the_io = the; *thi_io = thi;
    /* B6: luminosity diagnostic, eq 22 (L222) restricted to the applied loss */
    for (int k = 0; k < 4; ++k) diag7[k] = de_sum[k] * vol / dt;
    diag7[4] = limited; diag7[5] = floored; diag7[6] = clamped;
}

/* Whole field.  r, vol, lam0, qcc0, cell_lum may be NULL.  diag7 is the sum over cells; cell_lum[c][0..3] is cell c's
 * own term of the luminosity sums (eq 22), from which radial profiles (eq 25) are plain partial sums. */
void orc_step(const orc_table *tab, const orc_units *un, long long ncell,
              const double *rho, const double *bsq, const double *the_in, const double *thi_in,
              const double *r, const double *vol,
              double dt, int nsub, double f_limit, double h_floor, int rate_mode, int coulomb_mode,
              double *the_out, double *thi_out, double *lam0, double *qcc0, double *cell_lum, double *diag7, int nthreads,
              unsigned char *cell_flags)   /* optional, per cell: bit 0 limited, bit 1 floored, bit 2 clamped (diag7[4..6] of the cell) */
{
    double acc[7] = {0, 0, 0, 0, 0, 0, 0};
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel num_threads(nthreads)
    {
        double loc[7] = {0, 0, 0, 0, 0, 0, 0};
#pragma omp for schedule(static)
        for (long long c = 0; c < ncell; ++c) {
            double the = the_in[c], thi = thi_in[c], d7[7];
            if (cell_lum) for (int k = 0; k < 4; ++k) cell_lum[4 * c + k] = 0.0;
            if (cell_flags) cell_flags[c] = 0;
            if (isnan(rho[c]) || isnan(bsq[c]) || isnan(the) || isnan(thi)) {
                the_out[c] = NAN; thi_out[c] = NAN;
                if (lam0) lam0[c] = NAN;
                if (qcc0) qcc0[c] = NAN;
                continue;
            }
            if (!(rho[c] > 0.0)) {          /* no matter to cool: pass through */
                the_out[c] = the; thi_out[c] = thi;
                if (lam0) lam0[c] = 0.0;
                if (qcc0) qcc0[c] = 0.0;
                continue;
            }
            orc_step_cell(tab, un, rho[c], bsq[c], &the, &thi, r ? r[c] : 0.0, vol ? vol[c] : 1.0,
                          dt, nsub, f_limit, h_floor, rate_mode, coulomb_mode,
                          lam0 ? &lam0[c] : NULL, qcc0 ? &qcc0[c] : NULL, d7);
            the_out[c] = the; thi_out[c] = thi;
            if (cell_lum) for (int k = 0; k < 4; ++k) cell_lum[4 * c + k] = d7[k];
            if (cell_flags) cell_flags[c] = (unsigned char)((d7[4] != 0.0) | ((d7[5] != 0.0) << 1) | ((d7[6] != 0.0) << 2));
            for (int k = 0; k < 7; ++k) loc[k] += d7[k];
        }
#pragma omp critical
        for (int k = 0; k < 7; ++k) acc[k] += loc[k];
    }
    if (diag7) memcpy(diag7, acc, sizeof acc);
}

/* ================================================================================
 * Part B'  the implicit scheme (PAPER.md L185 (ii): "an implicit solver for the cooling
 * step ... adapted [from] the implicit-explicit (IMEX) solver ... used in the M1
 * radiation scheme"; L369: ~1.8x the cost).  The paper gives no equations; this is
 * reading C-18 of DESIGN.md, step by step:
 *
 *   per sub-step h = dt/nsub, from the start state (Theta_e, Theta_i):
 *     a   = h K C(Theta_e, Theta_i),  K C (Theta_i - Theta_e) = dTheta_e/dt of eq 15;
 *           the coefficient C is taken at the start state (the explicit half of IMEX),
 *           the driving difference at the end state (linearly implicit):
 *             x = a (Theta_i' - theta),  Theta_i' = Theta_i - g x,  g = (gamma_i-1)/(gamma_e-1)
 *           =>  x = a (Theta_i - theta) / (1 + a g)
 *     rhat(theta) = Lambda(rho, theta_c, bsq, Theta_i) (gamma_e-1) / (m_e/m_p rho theta_c),
 *           theta_c = theta clamped to the table's Theta_e range: outside the range the
 *           cooling TIME u_e/Lambda is held at its edge value (this is what makes the
 *           root positive); Theta_i inside Lambda (4-D tables, through H) is the start
 *           value; the floor test (eq 19) is taken at the start state
 *     backward Euler for the radiative sink:  theta is the root of
 *       F(theta) = theta - Theta_e + h theta rhat(theta) - a (Theta_i - theta)/(1 + a g)
 *     in (0, Theta_e + a Theta_i/(1 + a g)]  (F(0) < 0 <= F(upper end)), found by bisection
 *     Theta_e' = theta,  Theta_i' = Theta_i - g x(theta);  no limiter.
 *   diagnostic: dE = h Lambda at the end state (= h theta rhat(theta) in Theta units).
 *
 * Pins (tests/test_oracle_implicit.py): residual of the root, dt -> 0 agrees with the
 * unlimited explicit step, closed form for a constant cooling time (theta' = theta/(1+h/t_c)),
 * Coulomb-only closed form (linear 2x2 backward Euler), positivity for h Lambda >> u_e,
 * energy balance, no temperature crossing, zero exchange at equality.
 * ============================================================================== */
typedef struct {
    const orc_table *tab; const orc_units *un;
    double rho, bsq, the0, thi0, h, a, g, floored;
} orc_imp_ctx;

/* rhat(theta) * h * theta: the radiative loss of Theta_e over h at trial state theta;
 * lam_out/frac/cl (optional) return Lambda (code units), process shares, clamp flag. */
static double orc_imp_loss(const orc_imp_ctx *c, double theta, double *lam_out, double *frac, int *cl_out)
{
    const orc_table *tab = c->tab;
    const double mr = ORC_ME / ORC_MP, ge1 = c->un->gamma_e - 1.0;
    if (lam_out) *lam_out = 0.0;
    if (frac) { frac[0] = frac[1] = frac[2] = 0.0; }
    if (cl_out) *cl_out = 0;
    if (c->floored != 0.0 || !(theta > 0.0)) return 0.0;
    /* Theta_e range of the table */
    double tlo = 0.0, thi_edge = INFINITY;
    for (int k = 0; k < tab->ndim; ++k)
        if (tab->axis[k] == ORC_AX_LOG_THETA_E) { tlo = pow(10.0, tab->lo[k]); thi_edge = pow(10.0, tab->hi[k]); }
    double thc = theta < tlo ? tlo : (theta > thi_edge ? thi_edge : theta);
    double prim[4], x[4]; int cl = 0;
    prim[ORC_AX_LOG_RHO] = c->rho; prim[ORC_AX_LOG_THETA_E] = thc;
    prim[ORC_AX_LOG_BSQ] = c->bsq; prim[ORC_AX_LOG_THETA_I] = c->thi0;
    for (int k = 0; k < tab->ndim; ++k) {
        double q = prim[tab->axis[k]];
        x[k] = (q > 0.0) ? log10(q) : -INFINITY;
    }
    double lam;
    if (tab->nproc == 1) {
        lam = pow(10.0, orc_interp(tab->ndim, tab->n, tab->lo, tab->hi, tab->data[0], x, &cl));
    } else {
        double q[3];
        for (int p = 0; p < 3; ++p)
            q[p] = pow(10.0, orc_interp(tab->ndim, tab->n, tab->lo, tab->hi, tab->data[p], x, &cl));
        lam = orc_combine_code(c->un, c->rho, thc, c->thi0, q[0], q[1], q[2], frac);
    }
    if (theta != thc) cl = 1;
    if (cl_out) *cl_out = cl;
    double rhat = lam * ge1 / (mr * c->rho * thc);
    if (lam_out) *lam_out = rhat * theta * mr * c->rho / ge1;      /* Lambda at the trial state */
    return c->h * theta * rhat;
}
static double orc_imp_F(const orc_imp_ctx *c, double theta)
{
    return theta - c->the0 + orc_imp_loss(c, theta, NULL, NULL, NULL) - c->a * (c->thi0 - theta) / (1.0 + c->a * c->g);
}

static void orc_imp_setup(orc_imp_ctx *c, const orc_table *tab, const orc_units *un, double rho, double bsq,
                          double the, double thi, double r, double h, double h_floor, int coulomb_mode)
{
    const double mr = ORC_ME / ORC_MP, ge1 = un->gamma_e - 1.0, gi1 = un->gamma_i - 1.0;
    c->tab = tab; c->un = un; c->rho = rho; c->bsq = bsq; c->the0 = the; c->thi0 = thi; c->h = h; c->g = gi1 / ge1;
    c->floored = 0.0;
    if (h_floor > 0.0 && r > 0.0) {
        double tfloor = 0.5 * ORC_PI * pow(h_floor * orc_omega_k(r, un->spin) * r, 2.0);
        if ((the + thi) * mr < tfloor) c->floored = 1.0;
    }
    double C = 0.0;
    if (coulomb_mode == 1) {
        double xc[2] = { thi > 0.0 ? log10(thi) : -INFINITY, the > 0.0 ? log10(the) : -INFINITY };
        C = pow(10.0, orc_interp(2, tab->nc, tab->clo, tab->chi, tab->coul, xc, NULL));
    } else if (coulomb_mode == 2) {
        C = orc_coulomb_C(the, thi / un->ion_theta_mass_ratio);
    }
    /* dTheta_e/dt = K C (Theta_i - Theta_e),  K = pref conv rho (gamma_e-1)/(m_e/m_p) */
    c->a = h * orc_coulomb_pref_cgs(un) * orc_rate_conv(un) * rho * C * ge1 / mr;
}

/* F(theta) of the FIRST sub-step for one cell: lets a test check that a result which differs from the
 * oracle's root is still a root (several roots can exist where Lambda is not monotone in Theta_e). */
double orc_implicit_residual(const orc_table *tab, const orc_units *un, double rho, double bsq, double the, double thi,
                             double r, double dt, int nsub, double h_floor, int coulomb_mode, double theta_trial)
{
    orc_imp_ctx c;
    orc_imp_setup(&c, tab, un, rho, bsq, the, thi, r, dt / nsub, h_floor, coulomb_mode);
    return orc_imp_F(&c, theta_trial);
}

static void orc_step_cell_implicit(const orc_table *tab, const orc_units *un,
                                   double rho, double bsq, double *the_io, double *thi_io,
                                   double r, double vol, double dt, int nsub, double h_floor, int coulomb_mode, double *diag7)
{
    const double mr = ORC_ME / ORC_MP, ge1 = un->gamma_e - 1.0;
    const double h = dt / nsub;
    double the = *the_io, thi = *thi_io;
    double de_sum[4] = {0, 0, 0, 0};
    int floored = 0, clamped = 0;
    for (int s = 0; s < nsub; ++s) {
        orc_imp_ctx c;
        orc_imp_setup(&c, tab, un, rho, bsq, the, thi, r, h, h_floor, coulomb_mode);
        if (c.floored != 0.0) floored = 1;
        double lo = 0.0, hi = the + c.a * thi / (1.0 + c.a * c.g);
        if (!(hi > 0.0)) {              /* Theta_e = 0 and nothing to gain: nothing to do */
            continue;
        }
        for (int it = 0; it < 200; ++it) {
            double m = 0.5 * (lo + hi);
            if (m == lo || m == hi) break;
            if (orc_imp_F(&c, m) < 0.0) lo = m; else hi = m;
        }
        double theta = hi;                                  /* F(hi) >= 0: the first representable point at or past the root */
        double lam, frac[3]; int cl;
        double loss = orc_imp_loss(&c, theta, &lam, frac, &cl);
        (void)loss;
        clamped |= cl;
        double x = c.a * (thi - theta) / (1.0 + c.a * c.g);
        double de = lam * h;                                /* energy radiated, code units */
        de_sum[0] += de; de_sum[1] += de * frac[0]; de_sum[2] += de * frac[1]; de_sum[3] += de * frac[2];
        the = theta;
        thi = thi - c.g * x;
    }
    (void)mr; (void)ge1;
    *the_io = the; *thi_io = thi;
    for (int k = 0; k < 4; ++k) diag7[k] = de_sum[k] * vol / dt;
    diag7[4] = 0.0; diag7[5] = floored; diag7[6] = clamped;
}

/* Whole field, implicit scheme.  r, vol may be NULL.  diag7 is the sum over cells. */
void orc_step_implicit(const orc_table *tab, const orc_units *un, long long ncell,
                       const double *rho, const double *bsq, const double *the_in, const double *thi_in,
                       const double *r, const double *vol, double dt, int nsub, double h_floor, int coulomb_mode,
                       double *the_out, double *thi_out, double *cell_lum, double *diag7, int nthreads)
{
    double acc[7] = {0, 0, 0, 0, 0, 0, 0};
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel num_threads(nthreads)
    {
        double loc[7] = {0, 0, 0, 0, 0, 0, 0};
#pragma omp for schedule(dynamic, 256)
        for (long long c = 0; c < ncell; ++c) {
            double the = the_in[c], thi = thi_in[c], d7[7];
            if (cell_lum) for (int k = 0; k < 4; ++k) cell_lum[4 * c + k] = 0.0;
            if (isnan(rho[c]) || isnan(bsq[c]) || isnan(the) || isnan(thi)) { the_out[c] = NAN; thi_out[c] = NAN; continue; }
            if (!(rho[c] > 0.0)) { the_out[c] = the; thi_out[c] = thi; continue; }
            orc_step_cell_implicit(tab, un, rho[c], bsq[c], &the, &thi, r ? r[c] : 0.0, vol ? vol[c] : 1.0,
                                   dt, nsub, h_floor, coulomb_mode, d7);
            the_out[c] = the; thi_out[c] = thi;
            if (cell_lum) for (int k = 0; k < 4; ++k) cell_lum[4 * c + k] = d7[k];
            for (int k = 0; k < 7; ++k) loc[k] += d7[k];
        }
#pragma omp critical
        for (int k = 0; k < 7; ++k) acc[k] += loc[k];
    }
    if (diag7) memcpy(diag7, acc, sizeof acc);
}

/* Fill tables node by node from Part A (used by tests to check the product's builder
 * and to build tiny brute-force tables).  Node coordinate = lo + i*(hi-lo)/(n-1). */
void orc_fill_total3(const orc_units *un, const int *n, const double *lo, const double *hi, float *out, int nthreads)
{
    long long tot = (long long)n[0] * n[1] * n[2];
#pragma omp parallel for schedule(dynamic, 64) num_threads(nthreads > 0 ? nthreads : 1)
    for (long long t = 0; t < tot; ++t) {
        int k = (int)(t % n[2]), j = (int)((t / n[2]) % n[1]), i = (int)(t / ((long long)n[1] * n[2]));
        double rho = pow(10.0, lo[0] + i * (hi[0] - lo[0]) / (n[0] - 1));
        double the = pow(10.0, lo[1] + j * (hi[1] - lo[1]) / (n[1] - 1));
        double bsq = pow(10.0, lo[2] + k * (hi[2] - lo[2]) / (n[2] - 1));
        out[t] = (float)orc_node_total_log10(un, rho, the, bsq);
    }
}
/* 4-D process tables over (log rho, log Theta_e, log bsq, log Theta_i), Theta_i fastest: log10 Q_brem, log10 Q_syn (code
 * units) and log10 eta at every node, from orc_node_proc_log10 (used where a run must not load the product's builder). */
void orc_fill_proc4(const orc_units *un, const int *n, const double *lo, const double *hi, float *out0, float *out1, float *out2, int nthreads)
{
    long long tot = (long long)n[0] * n[1] * n[2] * n[3];
#pragma omp parallel for schedule(dynamic, 64) num_threads(nthreads > 0 ? nthreads : 1)
    for (long long t = 0; t < tot; ++t) {
        long long rem = t;
        double x[4], o3[3];
        for (int k = 3; k >= 0; --k) { x[k] = pow(10.0, lo[k] + (double)(rem % n[k]) * (hi[k] - lo[k]) / (n[k] - 1)); rem /= n[k]; }
        orc_node_proc_log10(un, x[0], x[1], x[2], x[3], o3);
        out0[t] = (float)o3[0]; out1[t] = (float)o3[1]; out2[t] = (float)o3[2];
    }
}
void orc_fill_coulomb2(const orc_units *un, const int *nc, const double *clo, const double *chi, float *out)
{
    for (int a = 0; a < nc[0]; ++a)
        for (int b = 0; b < nc[1]; ++b) {
            double thi = pow(10.0, clo[0] + a * (chi[0] - clo[0]) / (nc[0] - 1));
            double the = pow(10.0, clo[1] + b * (chi[1] - clo[1]) / (nc[1] - 1));
            out[(size_t)a * nc[1] + b] = (float)log10(orc_coulomb_C(the, thi / un->ion_theta_mass_ratio));
        }
}
/* Part D fillers: the paper's table (L124), node by node from Part A.  n, lo, hi over (log10 H_th[cm], log10 B[G],
 * log10 n_e[cm^-3], log10 T_e[K]), T_e fastest; values log10 Q_total[erg cm^-3 s^-1]. */
void orc_fill_total4_cgs(const int *n, const double *lo, const double *hi, float *out, int nthreads)
{
    long long tot = (long long)n[0] * n[1] * n[2] * n[3];
#pragma omp parallel for schedule(dynamic, 64) num_threads(nthreads > 0 ? nthreads : 1)
    for (long long t = 0; t < tot; ++t) {
        long long rem = t;
        double x[4];
        for (int k = 3; k >= 0; --k) { x[k] = lo[k] + (double)(rem % n[k]) * (hi[k] - lo[k]) / (n[k] - 1); rem /= n[k]; }
        double o6[6];
        orc_cooling_cgs(pow(10.0, x[0]), pow(10.0, x[1]), pow(10.0, x[2]), pow(10.0, x[3]) * ORC_KB / (ORC_ME * ORC_C * ORC_C), o6);
        out[t] = (float)log10(o6[4]);
    }
}
/* Coulomb table of L147 over (log10 n_e, log10 T_i[K], log10 T_e[K]), T_e fastest.  Eq 15 with rho/m_p = n_i = n_e (C-14)
 * is Q_cc = (3/2)(m_e/m_p) n_e^2 lnLambda c k_B sigma_T (T_i - T_e) C(theta_e, theta_i); the table stores
 * log10 [Q_cc/(T_i - T_e)], which is positive and smooth through T_i = T_e where Q_cc itself changes sign (C-23). */
void orc_fill_coulomb3_cgs(const orc_units *un, const int *n, const double *lo, const double *hi, float *out)
{
    const double k2t = ORC_KB / (ORC_ME * ORC_C * ORC_C);
    for (int a = 0; a < n[0]; ++a)
        for (int b = 0; b < n[1]; ++b)
            for (int c = 0; c < n[2]; ++c) {
                double ne = pow(10.0, lo[0] + a * (hi[0] - lo[0]) / (n[0] - 1));
                double ti = pow(10.0, lo[1] + b * (hi[1] - lo[1]) / (n[1] - 1));
                double te = pow(10.0, lo[2] + c * (hi[2] - lo[2]) / (n[2] - 1));
                double C = orc_coulomb_C(te * k2t, ti * k2t / un->ion_theta_mass_ratio);
                double k = 1.5 * (ORC_ME / ORC_MP) * ne * ne * un->ln_lambda * ORC_C * ORC_KB * ORC_SIGT * C;
                out[((size_t)a * n[1] + b) * n[2] + c] = (float)log10(k);
            }
}
int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ======================================================================================
 * Part C — radiation-pressure temperature correction (eq 29;
 * DESIGN.md reading C-20).  Post-processing, cell by cell.
 *
 *   P = P_rad + P_gas = a T_e^4 + N k_B T_gas,   T_gas = T_e + T_i          (eq 29)
 *
 * P is the pressure the simulation holds for the cell, which has no radiation term (L332:
 * "our simulations do not take radiation pressure into account"): P = N k_B (T_e + T_i)
 * with the simulated temperatures.  The paper recalculates T_e only (L345), so T_i is the
 * simulated one on both sides and N k_B T_i cancels:
 *
 *   a T^4 + N k_B (T - T_e) = 0,     0 < T <= T_e                             (one root)
 *
 * solved where the in-cell scattering depth tau_sca = n_e sigma_T H(r) (L353) exceeds a
 * threshold (1 for Fig. 9(b); 4.6 for Fig. 10); other cells keep T_e.
 * a = 7.5646e-15 erg cm^-3 K^-4 is the value the paper prints (L345), not 4 sigma_SB/c.
 * N = n_e (C-14: fully ionised hydrogen).  The root is found by bisection on [0, T_e].
 * ====================================================================================== */
#define ORC_ARAD 7.5646e-15           /* erg cm^-3 K^-4, as printed (L345) */

double orc_tau_sca_cell(const orc_units *u, double rho, double hscale_rg)     /* L353 */
{
    return orc_ne_cgs(u, rho) * ORC_SIGT * (hscale_rg * orc_rg(u));
}

/* Returns the corrected Theta_e; *corrected = 1 if the quartic was solved for this cell. */
double orc_radpress_cell(const orc_units *u, double rho, double the, double hscale_rg, double tau_crit, int *corrected)
{
    *corrected = 0;
    if (!(rho > 0.0) || !(the > 0.0) || !(orc_tau_sca_cell(u, rho, hscale_rg) > tau_crit)) return the;
    double N = orc_ne_cgs(u, rho);
    double Te = the * ORC_ME * ORC_C * ORC_C / ORC_KB;          /* K */
    double lo = 0.0, hi = Te;                                   /* f(0) = -N k T_e < 0 <= a T_e^4 = f(T_e) */
    for (int it = 0; it < 200; ++it) {
        double T = 0.5 * (lo + hi);
        double f = ORC_ARAD * T * T * T * T + N * ORC_KB * (T - Te);
        if (f > 0.0) hi = T; else lo = T;
    }
    *corrected = 1;
    return 0.5 * (lo + hi) * ORC_KB / (ORC_ME * ORC_C * ORC_C);
}

void orc_radpress(const orc_units *u, long long ncell, const double *rho, const double *the, const double *hscale_rg,
                  double tau_crit, double *the_out, long long *ncorrected)
{
    long long cnt = 0;
    for (long long k = 0; k < ncell; ++k) {
        int c;
        the_out[k] = orc_radpress_cell(u, rho[k], the[k], hscale_rg[k], tau_crit, &c);
        cnt += c;
    }
    *ncorrected = cnt;
}
