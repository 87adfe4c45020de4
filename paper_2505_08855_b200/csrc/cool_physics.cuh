// cool_physics.cuh — analytic emissivities of arXiv 2505.08855 §II in fp64,
// callable from host (table builder, cool_builder.cu) and device (COOL_V_ANALYTIC kernel).
// Product code: shares nothing with oracle/.  Algorithms differ from the oracle's on purpose
// (safeguarded Newton instead of bisection for nu_c, closed-form incomplete gamma functions
// instead of quadrature for the frequency integral).
#pragma once
#include <math.h>

#if defined(__CUDACC__)
#define CP_HD __host__ __device__ __forceinline__
#define CP_HD_NOINLINE inline __host__ __device__ __noinline__
#else
#define CP_HD inline
#define CP_HD_NOINLINE inline
#endif

namespace coolphys {

// CODATA-2018, cgs
constexpr double kC = 2.99792458e10, kKB = 1.380649e-16, kME = 9.1093837015e-28, kMP = 1.67262192369e-24;
constexpr double kQE = 4.80320471257e-10, kHPL = 6.62607015e-27, kSIGT = 6.6524587321e-25, kSIGSB = 5.670374419e-5;
constexpr double kGMSUN = 1.32712440018e26, kPI = 3.14159265358979323846;
constexpr double kMEC2 = kME * kC * kC;          // erg
constexpr double kTHETA_TO_K = kMEC2 / kKB;      // T_e = Theta_e * this
constexpr double kMR = kME / kMP;

struct Units {                                    // mirrors cool_units
    double rho_scale_cgs, mbh_msun, gamma_e, gamma_i, ln_lambda, ion_theta_mass_ratio, hth_cm, r_ref_rg, spin;
};
struct Derived {                                  // everything the kernels need, precomputed once
    double rg_cm, tg_s, rate_conv;                // rate_conv: erg cm^-3 s^-1 -> code
    double ne_per_rho;                            // n_e = ne_per_rho * rho              (C-14)
    double b2_per_bsq;                            // B^2[G^2] = b2_per_bsq * bsq         (L173)
    double coul_pref_code;                        // Q_cc = this * rho^2 (Th_i - Th_e) C (eq 15)
    double h_per_cs;                              // H_th[cm] = h_per_cs * c_s  at r_ref (eq 13)
};
CP_HD Derived derive(const Units& u)
{
    Derived d;
    d.rg_cm = kGMSUN * u.mbh_msun / (kC * kC);
    d.tg_s = d.rg_cm / kC;
    d.rate_conv = d.tg_s / (u.rho_scale_cgs * kC * kC);
    d.ne_per_rho = u.rho_scale_cgs / kMP;
    d.b2_per_bsq = 4.0 * kPI * u.rho_scale_cgs * kC * kC;
    d.coul_pref_code = 1.5 * kMR * u.ln_lambda * kC * kSIGT * kMEC2 * d.ne_per_rho * d.ne_per_rho * d.rate_conv;
    d.h_per_cs = d.rg_cm * (pow(u.r_ref_rg, 1.5) + u.spin);
    return d;
}

// ---- eqs 1-2 (L59-L63): bremsstrahlung, erg cm^-3 s^-1 per n_e^2 ------------------------
CP_HD double brems_per_ne2(double th)
{
    double fee, fei;
    if (th < 1.0) {
        double rt = sqrt(th);
        fee = th * rt * (1.0 + th * (1.1 + th) - 1.25 * th * th * rt);
        fei = 4.0 * sqrt(2.0 / (kPI * kPI * kPI)) * rt * (1.0 + 1.781 * pow(th, 1.34));
    } else {
        fee = 1.34 * th * (log(1.123 * th) + 1.28);
        fei = (4.5 / kPI) * th * (log(1.123 * th + 0.48) + 1.5);
    }
    return 2.56e-22 * fee + 1.48e-22 * fei;
}

// ---- exponentially scaled modified Bessel functions e^x K_nu(x), nu = 0, 1 -------------
// Trapezoid rule on e^x K_nu(x) = int_0^inf exp(-2x sinh^2(t/2)) cosh(nu t) dt; 64 points reach
// fp64 round-off because the integrand is analytic and decays doubly exponentially.
CP_HD void bessel_k01_scaled(double x, double& k0, double& k1)
{
    const int N = 64;
    const double tmax = 2.0 * asinh(sqrt(22.0 / x));      // exponent -44 at the cut
    const double h = tmax / N;
    double s0 = 0.5, s1 = 0.5;
    for (int k = 1; k <= N; ++k) {
        double t = k * h;
        double sh = sinh(0.5 * t);
        double e = exp(-2.0 * x * sh * sh);
        s0 += e;
        s1 += e * (1.0 + 2.0 * sh * sh);                  // cosh t = 1 + 2 sinh^2(t/2)
    }
    k0 = s0 * h; k1 = s1 * h;
}
CP_HD double bessel_k2_scaled(double x)
{
    double k0, k1;
    bessel_k01_scaled(x, k0, k1);
    return k0 + (2.0 / x) * k1;
}

// K2(1/theta_e) with the paper's low-temperature replacement 2 theta_e^2 (L87, literal 1e8 K)
CP_HD double k2_tilde(double th)
{
    if (th * kTHETA_TO_K > 1.0e8) {
        double x = 1.0 / th;
        return bessel_k2_scaled(x) * exp(-x);
    }
    return 2.0 * th * th;
}

// ---- eq 4 (L76): ln I'(x) and its u-derivative at x = e^u --------------------------------
CP_HD void ln_iprime(double u, double& f, double& dfdu)
{
    double a = 0.4 * exp(-0.25 * u), b = 0.5316 * exp(-0.5 * u), c = 1.8899 * exp(u / 3.0);
    double s = 1.0 + a + b;
    f = 1.398840330288409 /* ln 4.0505 */ - u / 6.0 + log(s) - c;
    dfdu = -1.0 / 6.0 - (0.25 * a + 0.5 * b) / s - c / 3.0;
}

// upper incomplete gamma function Gamma(a, t), a > 0, returned as Gamma(a,t) * e^{+t} * t^{-a}
// is avoided: we return the plain value (underflows to 0 for t > ~740, as it should).
CP_HD double gamma_upper(double a, double t, double gamma_a)
{
    if (t <= 0.0) return gamma_a;
    if (t < a + 1.0) {                               // series for the lower function
        double term = 1.0 / a, sum = term, ap = a;
        for (int n = 0; n < 500; ++n) {
            ap += 1.0;
            term *= t / ap;
            sum += term;
            if (fabs(term) < fabs(sum) * 1e-17) break;
        }
        return gamma_a - sum * exp(-t + a * log(t));
    }
    // modified Lentz evaluation of the continued fraction
    const double tiny = 1e-300;
    double b = t + 1.0 - a, c = 1.0 / tiny, d = 1.0 / b, hcf = d;
    for (int i = 1; i < 500; ++i) {
        double an = -i * (i - a);
        b += 2.0;
        d = an * d + b; if (fabs(d) < tiny) d = tiny;
        c = b + an / c; if (fabs(c) < tiny) c = tiny;
        d = 1.0 / d;
        double del = d * c;
        hcf *= del;
        if (fabs(del - 1.0) < 1e-16) break;
    }
    return exp(-t + a * log(t)) * hcf;
}

// J(x_c) = int_{x_c}^inf x I'(x) dx.  With t = 1.8899 x^{1/3} the integrand is a sum of
// t^{s-1} e^{-t} terms, s = 5.5, 4.75, 4  (eq 4 inserted in eq 6).
CP_HD double synch_J(double xc)
{
    const double a = 1.8899;
    const double g55 = 52.34277778455352, g475 = 16.586206539225937;             // Gamma(5.5), Gamma(4.75)
    double tc = a * cbrt(xc);
    double i55 = gamma_upper(5.5, tc, g55), i475 = gamma_upper(4.75, tc, g475);
    double i4 = exp(-tc) * (6.0 + tc * (6.0 + tc * (3.0 + tc)));
    const double a4 = a * a * a * a;
    return 3.0 * 4.0505 * (i55 / (a4 * a * sqrt(a)) + 0.4 * i475 / (a4 * pow(a, 0.75)) + 0.5316 * i4 / a4);
}

struct Cooling { double brems, synch, eta, thin, total, nu_c; };   // cgs

// eqs 3-6: x_c from eq 5 by safeguarded Newton in u = ln x, then eq 6.
CP_HD_NOINLINE double synch_cgs(double H, double B, double ne, double th, double* nu_c)
{
    const double s = 3.0 * kQE * B * th * th / (4.0 * kPI * kME * kC);      // nu = s x_M
    const double k2 = k2_tilde(th);
    const double lnR = log(s * th * kME * k2 / (8.86e-30 * H * ne));
    // F(u) = ln I'(e^u) - u - lnR, strictly decreasing
    double lo = -1200.0, hi = 90.0;
    double u = (lnR > 0.5) ? (0.7667 - lnR) * 0.6 : 0.0;
    if (u < lo) u = 0.5 * (lo + hi);
    for (int it = 0; it < 200; ++it) {
        double f, df;
        ln_iprime(u, f, df);
        f -= u + lnR; df -= 1.0;
        if (f > 0.0) lo = u; else hi = u;
        double un = u - f / df;
        if (!(un > lo && un < hi)) un = 0.5 * (lo + hi);
        if (fabs(un - u) <= 1e-15 * fmax(1.0, fabs(u))) { u = un; break; }
        u = un;
    }
    const double xc = exp(u);
    const double nuc = s * xc;
    const double te = th * kTHETA_TO_K;
    const double rj = 2.0 * kPI * kKB * te * nuc * nuc * nuc / (3.0 * kC * kC * H);
    const double thin = 4.43e-30 * 4.0 * kPI * ne * s * s * synch_J(xc) / k2;
    *nu_c = nuc;
    return rj + thin;
}

// eqs 7-9 with the series-sum exponent -1 - lnP/lnA (reading C-1)
CP_HD double compton_eta(double nu_c, double ne, double H, double th)
{
    double x = kHPL * nu_c / kMEC2;
    if (!(x < 3.0 * th)) return 1.0;
    double P = -expm1(-2.0 * ne * kSIGT * H);
    if (!(P > 0.0)) return 1.0;
    double am1 = 4.0 * th * (1.0 + 4.0 * th);
    double lnA = log1p(am1);
    double onemPA = 1.0 - P * (1.0 + am1);
    double lr = log(3.0 * th / x);                       // > 0
    if (fabs(onemPA) < 1e-8) return 1.0 + P * am1 * lr / lnA;
    // (x/3theta)^(-1 - lnP/lnA) = exp(lr (1 + lnP/lnA))
    return 1.0 + P * am1 / onemPA * (1.0 - exp(lr * (1.0 + log(P) / lnA)));
}

// eqs 11-12 (sigma = Stefan-Boltzmann, tau_obs = tau_abs; reading C-2)
CP_HD double bridge_cgs(double H, double ne, double th, double qthin)
{
    double te = th * kTHETA_TO_K, te2 = te * te;
    double bb_over_h = 4.0 * kSIGSB * te2 * te2 / H;
    double tau_abs = qthin / bb_over_h;
    double tau_sca = 2.0 * ne * kSIGT * H;
    // (bb/H)/(1.5 tau + sqrt3 + 1/tau_abs) = qthin / (1 + tau_abs (sqrt3 + 1.5 (tau_abs + tau_sca)))
    return qthin / (1.0 + tau_abs * (1.7320508075688772 + 1.5 * (tau_abs + tau_sca)));
}

CP_HD_NOINLINE Cooling cooling_cgs(double H, double B, double ne, double th)
{
    Cooling c;
    c.brems = brems_per_ne2(th) * ne * ne;
    c.synch = synch_cgs(H, B, ne, th, &c.nu_c);
    c.eta = compton_eta(c.nu_c, ne, H, th);
    c.thin = c.brems + c.eta * c.synch;
    c.total = bridge_cgs(H, ne, th, c.thin);
    return c;
}

// eqs 13-14 in code units (c = 1): c_s^2 = (gamma_e P_e + gamma_i P_i)/(rho + u + P), rho cancels
CP_HD double sound_speed2(const Units& u, double th_e, double th_i)
{
    double pe = th_e * kMR, pi = th_i * kMR;
    return (u.gamma_e * pe + u.gamma_i * pi) / (1.0 + pe * u.gamma_e / (u.gamma_e - 1.0) + pi * u.gamma_i / (u.gamma_i - 1.0));
}

// eq 15: C(theta_e, theta_i) = [ (2s^2+1)/s K1(1/th_m) + 2 K0(1/th_m) ] / [K2(1/th_e) K2(1/th_i)]
// with scaled Bessel functions (the exponentials cancel since 1/th_m = 1/th_e + 1/th_i).
CP_HD_NOINLINE double coulomb_C(double th_e, double th_i)
{
    double xe = 1.0 / th_e, xi = 1.0 / th_i;
    double s = th_e + th_i;
    double k0, k1;
    bessel_k01_scaled(xe + xi, k0, k1);
    return ((2.0 * s * s + 1.0) / s * k1 + 2.0 * k0) / (bessel_k2_scaled(xe) * bessel_k2_scaled(xi));
}

}  // namespace coolphys
