// cool_builder.cu — host table builder (north_star subsystem (a)): tabulates PAPER.md eqs 1-12
// (and the Coulomb coefficient of eq 15) on a log-spaced grid (L122-L124, L147).  Host threads only.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <thread>
#include <vector>

#include "cool_internal.h"

namespace cool {

static bool axes_valid(const cool_table_desc *d, std::string *why)
{
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
    const cool_units &u = d->units;
    if (!(u.rho_scale_cgs > 0 && u.mbh_msun > 0 && u.gamma_e > 1 && u.gamma_i > 1 && u.ln_lambda > 0 &&
          u.ion_theta_mass_ratio > 0 && u.hth_cm > 0 && u.r_ref_rg > 0 && std::isfinite(u.spin))) {
        *why = "units: need rho_scale, mbh, ln_lambda, ion_theta_mass_ratio, hth_cm, r_ref > 0 and gamma_e, gamma_i > 1";
        return false;
    }
    return true;
}
bool desc_valid(const cool_table_desc *d, bool need_coulomb_shape, std::string *why)
{
    if (!d) { *why = "NULL descriptor"; return false; }
    if (!axes_valid(d, why)) return false;
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
