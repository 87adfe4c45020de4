// cool_builder.cu — host table builder (north_star subsystem (a)): tabulates PAPER.md eqs 1-12
// (and the Coulomb coefficient of eq 15) on a log-spaced grid (L122-L124, L147).  Host threads only.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <thread>
#include <vector>

#include "cool_internal.h"

namespace cool {

bool desc_is_cgs(const cool_table_desc *d)
{
    return d && d->ndim == 4 && d->axis[0] == COOL_AX_LOG_HTH && d->axis[1] == COOL_AX_LOG_B && d->axis[2] == COOL_AX_LOG_NE && d->axis[3] == COOL_AX_LOG_TE;
}

static bool units_valid(const cool_units &u, std::string *why)
{
    if (!(u.rho_scale_cgs > 0 && u.mbh_msun > 0 && u.gamma_e > 1 && u.gamma_i > 1 && u.ln_lambda > 0 &&
          u.ion_theta_mass_ratio > 0 && u.hth_cm > 0 && u.r_ref_rg > 0 && std::isfinite(u.spin))) {
        *why = "units: need rho_scale, mbh, ln_lambda, ion_theta_mass_ratio, hth_cm, r_ref > 0 and gamma_e, gamma_i > 1";
        return false;
    }
    return true;
}

static bool axes_valid(const cool_table_desc *d, std::string *why)
{
    if (d->ndim == 4 && d->axis[0] >= COOL_AX_LOG_HTH) {          // the paper's table (L122-L124)
        if (!desc_is_cgs(d) || !(d->nproc == 1 || d->nproc == 0)) { *why = "the paper's table has axes {LOG_HTH, LOG_B, LOG_NE, LOG_TE} in this order and nproc = 1"; return false; }
        for (int k = 0; k < 4; ++k) {
            if (d->n[k] < 2 || d->n[k] > 4096) { *why = "n[k] must be in [2, 4096]"; return false; }
            if (!(d->hi[k] > d->lo[k]) || !std::isfinite(d->lo[k]) || !std::isfinite(d->hi[k])) { *why = "need finite hi[k] > lo[k]"; return false; }
        }
        return units_valid(d->units, why);
    }
    if (!((d->ndim == 3 && (d->nproc == 1 || d->nproc == 0)) || (d->ndim == 4 && (d->nproc == 3 || d->nproc == 0)))) {
        *why = "supported shapes: ndim=3 with nproc=1, ndim=4 with nproc=3 (nproc=0: analytic only)";
        return false;
    }
    int seen[4] = {0, 0, 0, 0};
    for (int k = 0; k < d->ndim; ++k) {
        int a = d->axis[k];
        if (a < 0 || a > 3 || seen[a]) { *why = "axis[] must be distinct cool_axis values"; return false; }
        if (d->ndim == 3 && a == COOL_AX_LOG_THETA_I) { *why = "a 3-D table has axes log rho, log Theta_e, log bsq"; return false; }
        seen[a] = 1;
        if (d->n[k] < 2 || d->n[k] > 4096) { *why = "n[k] must be in [2, 4096]"; return false; }
        if (!(d->hi[k] > d->lo[k]) || !std::isfinite(d->lo[k]) || !std::isfinite(d->hi[k])) { *why = "need finite hi[k] > lo[k]"; return false; }
    }
    return units_valid(d->units, why);
}
bool desc_valid(const cool_table_desc *d, bool need_coulomb_shape, std::string *why)
{
    if (!d) { *why = "NULL descriptor"; return false; }
    if (!axes_valid(d, why)) return false;
    if (need_coulomb_shape && desc_is_cgs(d)) {
        for (int k = 0; k < 3; ++k)
            if (d->nc3[k] < 2 || d->nc3[k] > 4096 || !(d->c3hi[k] > d->c3lo[k])) { *why = "Coulomb table: nc3[k] in [2,4096], c3hi[k] > c3lo[k]"; return false; }
        return true;
    }
    if (need_coulomb_shape) {
        for (int k = 0; k < 2; ++k)
            if (d->nc[k] < 2 || d->nc[k] > 4096 || !(d->chi[k] > d->clo[k])) { *why = "Coulomb table: nc[k] in [2,4096], chi[k] > clo[k]"; return false; }
    }
    return true;
}

coolphys::Units to_units(const cool_units &u)
{
    coolphys::Units p;
    p.rho_scale_cgs = u.rho_scale_cgs; p.mbh_msun = u.mbh_msun; p.gamma_e = u.gamma_e; p.gamma_i = u.gamma_i;
    p.ln_lambda = u.ln_lambda; p.ion_theta_mass_ratio = u.ion_theta_mass_ratio; p.hth_cm = u.hth_cm;
    p.r_ref_rg = u.r_ref_rg; p.spin = u.spin;
    return p;
}

template <class F>
static void parallel_for(long long n, int nthreads, F f)
{
    if (nthreads <= 0) nthreads = (int)std::max(1u, std::thread::hardware_concurrency());
    nthreads = (int)std::min<long long>(nthreads, std::max<long long>(1, n / 64));
    std::atomic<long long> next{0};
    const long long chunk = 256;
    auto work = [&]() {
        for (;;) {
            long long b = next.fetch_add(chunk);
            if (b >= n) break;
            long long e = std::min(n, b + chunk);
            for (long long i = b; i < e; ++i) f(i);
        }
    };
    std::vector<std::thread> th;
    for (int t = 1; t < nthreads; ++t) th.emplace_back(work);
    work();
    for (auto &t : th) t.join();
}

}  // namespace cool

extern "C" cool_status cool_table_build_host(const cool_table_desc *shape, float *const out[3], float *out_coulomb, int nthreads)
{
    using namespace cool;
    std::string why;
    if (!desc_valid(shape, out_coulomb != nullptr, &why)) { set_error("cool_table_build_host: %s", why.c_str()); return COOL_EINVAL; }
    if (shape->nproc > 0 && !out) { set_error("cool_table_build_host: out is NULL"); return COOL_EINVAL; }
    for (int p = 0; p < shape->nproc; ++p)
        if (!out[p]) { set_error("cool_table_build_host: out[%d] is NULL", p); return COOL_EINVAL; }

    const coolphys::Units un = to_units(shape->units);
    const coolphys::Derived der = coolphys::derive(un);
    const int nd = shape->ndim, np = shape->nproc;
    long long total = 1;
    for (int k = 0; k < nd; ++k) total *= shape->n[k];

    if (desc_is_cgs(shape)) {
        // the paper's table: log10 Q_total[erg cm^-3 s^-1] at (H_th[cm], B[G], n_e[cm^-3], T_e[K]) nodes, T_e fastest (L124, L157)
        if (np > 0) {
            parallel_for(total, nthreads, [&](long long flat) {
                double x[4];
                long long rem = flat;
                for (int k = 3; k >= 0; --k) {
                    x[k] = pow(10.0, shape->lo[k] + (double)(rem % shape->n[k]) * (shape->hi[k] - shape->lo[k]) / (shape->n[k] - 1));
                    rem /= shape->n[k];
                }
                out[0][flat] = (float)log10(coolphys::cooling_cgs(x[0], x[1], x[2], x[3] / coolphys::kTHETA_TO_K).total);
            });
        }
        if (out_coulomb) {
            // Q_cc(n_e, T_i, T_e) of L147 per kelvin of T_i - T_e: (3/2)(m_e/m_p) n_e^2 lnLambda c k_B sigma_T C(theta_e, theta_i)
            const int n0 = shape->nc3[0], n1 = shape->nc3[1], n2 = shape->nc3[2];
            parallel_for((long long)n0 * n1 * n2, nthreads, [&](long long flat) {
                const int c = (int)(flat % n2), b = (int)((flat / n2) % n1), a = (int)(flat / ((long long)n1 * n2));
                const double ne = pow(10.0, shape->c3lo[0] + a * (shape->c3hi[0] - shape->c3lo[0]) / (n0 - 1));
                const double ti = pow(10.0, shape->c3lo[1] + b * (shape->c3hi[1] - shape->c3lo[1]) / (n1 - 1));
                const double te = pow(10.0, shape->c3lo[2] + c * (shape->c3hi[2] - shape->c3lo[2]) / (n2 - 1));
                const double C = coolphys::coulomb_C(te / coolphys::kTHETA_TO_K, ti / coolphys::kTHETA_TO_K / un.ion_theta_mass_ratio);
                out_coulomb[flat] = (float)log10(1.5 * coolphys::kMR * ne * ne * un.ln_lambda * coolphys::kC * coolphys::kKB * coolphys::kSIGT * C);
            });
        }
        return COOL_OK;
    }
    if (np > 0) {
        parallel_for(total, nthreads, [&](long long flat) {
            double prim[4] = {0, 0, 0, 0};           // indexed by cool_axis: rho, theta_e, bsq, theta_i
            long long rem = flat;
            for (int k = nd - 1; k >= 0; --k) {
                int i = (int)(rem % shape->n[k]);
                rem /= shape->n[k];
                double x = shape->lo[k] + i * (shape->hi[k] - shape->lo[k]) / (shape->n[k] - 1);
                prim[shape->axis[k]] = pow(10.0, x);
            }
            const double rho = prim[COOL_AX_LOG_RHO], the = prim[COOL_AX_LOG_THETA_E];
            const double ne = der.ne_per_rho * rho;
            const double B = sqrt(der.b2_per_bsq * prim[COOL_AX_LOG_BSQ]);
            double H = un.hth_cm;
            if (nd == 4) H = der.h_per_cs * sqrt(coolphys::sound_speed2(un, the, prim[COOL_AX_LOG_THETA_I]));
            coolphys::Cooling c = coolphys::cooling_cgs(H, B, ne, the);
            if (np == 1) {
                out[0][flat] = (float)log10(c.total * der.rate_conv);
            } else {
                out[0][flat] = (float)log10(c.brems * der.rate_conv);
                out[1][flat] = (float)log10(c.synch * der.rate_conv);
                out[2][flat] = (float)log10(c.eta);
            }
        });
    }
    if (out_coulomb) {
        const int n0 = shape->nc[0], n1 = shape->nc[1];
        parallel_for((long long)n0 * n1, nthreads, [&](long long flat) {
            int a = (int)(flat / n1), b = (int)(flat % n1);
            double thi = pow(10.0, shape->clo[0] + a * (shape->chi[0] - shape->clo[0]) / (n0 - 1));
            double the = pow(10.0, shape->clo[1] + b * (shape->chi[1] - shape->clo[1]) / (n1 - 1));
            out_coulomb[flat] = (float)log10(coolphys::coulomb_C(the, thi / un.ion_theta_mass_ratio));
        });
    }
    return COOL_OK;
}
