// cool_implicit.cuh — the implicit cooling scheme (COOL_SCHEME_IMPLICIT; PAPER.md L185 (ii), L369; reading C-18 of
// DESIGN.md), first correct CUDA path: fp64 arithmetic for either cell dtype, one thread per cell (vector) of the SoA
// stream, the table read through the same lookup policies as the fp64 explicit path.
//
// Per sub-step h, from the start state (Theta_e, Theta_i):
//   q        = a/(1 + a g),  a = h K C(Theta_e, Theta_i),  g = (gamma_i - 1)/(gamma_e - 1)      (Coulomb: coefficient at
//              the start state, driving difference at the end state  =>  transfer x = q (Theta_i - theta))
//   loss(th) = h th Lambda(rho, th_c, bsq, Theta_i) (gamma_e - 1)/(m_e/m_p rho th_c),  th_c = th clamped to the table's
//              Theta_e range (the cooling time is held outside the range, which keeps the root positive)
//   theta    = root of  F(th) = th - Theta_e + loss(th) - q (Theta_i - th)  in (0, Theta_e + q Theta_i]
//   Theta_e' = theta,  Theta_i' = Theta_i - g q (Theta_i - theta);  no limiter.
// The root is bracketed from the start (F(0) < 0 <= F(upper end)) and refined by Illinois-type false position with a
// bisection safeguard until the bracket is two ulps wide; F' >= 1 wherever the loss does not decrease with Theta_e, so
// the answer is then within rounding of the root.
#pragma once
#include "cool_kernels.cuh"

namespace cool {

struct ImpCell {            // what F needs, fixed over one sub-step
    double rho, the0, thi0, q, tmin, tmax;
    Loc64 lr, lb, li;
    bool floored;
};

// loss(th) in Theta units; optionally the process shares of Q_thin and the clamp flag of the Theta_e coordinate
template <int MODE, class Fetch>
__device__ __forceinline__ double imp_loss(const DevTable &T, const StepConst &S, const Fetch &F, const ImpCell &c, double th,
                                           double *frac, int *clamped)
{
    if (frac) { frac[0] = frac[1] = frac[2] = 0.0; }
    if (clamped) *clamped = 0;
    if (c.floored || !(th > 0.0)) return 0.0;
    const double thc = fmin(fmax(th, c.tmin), c.tmax);
    Loc64 le = locate64(T.ax[CAX_THE], thc);
    if (clamped) *clamped = le.clamped | (thc != th);
    double lam;
    if constexpr (MODE == 3) {
        lam = exp10(interp3_f64(F, c.lr, le, c.lb));
    } else {
        double y[3];
        interp4_f64(F, c.lr, le, c.li, c.lb, y);
        const double qbr = exp10(y[0]), qsy = exp10(y[1]), eta = exp10(y[2]);
        const double qthin = qbr + eta * qsy;                                               // eq 10
        const double cs2 = (S.ae * thc + S.ai * c.thi0) / (1.0 + S.be * thc + S.bi * c.thi0);   // eq 14
        const double H = S.h_per_cs * sqrt(cs2);                                            // eq 13
        const double th2 = thc * thc;
        const double tau_abs = qthin * H / (S.bb_k * th2 * th2);                            // eq 12
        const double tau_sca = S.tausca_k * c.rho * H;
        lam = qthin / (1.0 + tau_abs * (1.7320508075688772 + 1.5 * (tau_abs + tau_sca)));   // eq 11
        if (frac) { frac[0] = qbr / qthin; frac[1] = qsy / qthin; frac[2] = (eta - 1.0) * qsy / qthin; }
    }
    return S.h * th * (lam * S.ge1 / (c.rho * S.mr * thc));
}

template <int MODE, class Fetch>
__device__ __forceinline__ double imp_F(const DevTable &T, const StepConst &S, const Fetch &F, const ImpCell &c, double th)
{
    return (th - c.the0) + imp_loss<MODE>(T, S, F, c, th, nullptr, nullptr) - c.q * (c.thi0 - th);
}

template <int MODE, class Fetch>
__device__ void implicit_cell(const DevTable &T, const DevConst &K, const StepConst &S, const Fetch &F,
                              double rho, double bsq, double &the, double &thi, double r, double vol, DiagAcc &acc)
{
    if (isnan(rho) || isnan(bsq) || isnan(the) || isnan(thi)) { the = thi = __longlong_as_double(0x7ff8000000000000LL); return; }
    if (!(rho > 0.0)) return;
    ImpCell c;
    c.rho = rho;
    c.lr = locate64(T.ax[CAX_RHO], rho); c.lb = locate64(T.ax[CAX_BSQ], bsq);
    c.tmin = exp10(T.ax[CAX_THE].lo10); c.tmax = exp10(T.ax[CAX_THE].lo10 + (T.ax[CAX_THE].n - 1) / T.ax[CAX_THE].inv10);
    const double g = S.gi1 / S.ge1;
    int floored = 0, clamped = c.lr.clamped | c.lb.clamped;
    double de_sum[4] = {0, 0, 0, 0};
    for (int s = 0; s < S.nsub; ++s) {
        c.the0 = the; c.thi0 = thi;
        c.floored = false;
        if (S.hfloor2 > 0.0 && r > 0.0) {
            const double ok = r / (r * sqrt(r) + S.spin);            // Omega_K r
            if ((the + thi) * S.mr < S.hfloor2 * ok * ok) { c.floored = true; floored = 1; }
        }
        if constexpr (MODE == 4) { c.li = locate64(T.ax[CAX_THI], thi); clamped |= c.li.clamped; }
        double C = 0.0;
        if (S.coulomb == 1) C = coulomb_C_table64(T, the, thi);
        else if (S.coulomb == 2) C = coolphys::coulomb_C(the, thi / K.units.ion_theta_mass_ratio);
        const double a = S.coul_kh * rho * C;
        c.q = a / (1.0 + a * g);

        double lo = 0.0, hi = the + c.q * thi;
        if (!(hi > 0.0)) continue;
        double flo = -hi, fhi = imp_F<MODE>(T, S, F, c, hi);         // F(0) = -Theta_e - q Theta_i
        int side = 0;
        for (int it = 0; it < 200 && fhi != 0.0; ++it) {
            const double width = hi - lo;
            if (!(width > 4.4408920985006262e-16 * hi)) break;       // two ulps
            double m = hi - fhi * (width / (fhi - flo));
            if (!(m > lo && m < hi) || (it % 3) == 2) m = lo + 0.5 * width;
            if (m == lo || m == hi) break;
            const double fm = imp_F<MODE>(T, S, F, c, m);
            if (fm < 0.0) { lo = m; flo = fm; if (side == -1) fhi *= 0.5; side = -1; }
            else { hi = m; fhi = fm; if (side == 1) flo *= 0.5; side = 1; }
        }
        // polish the last two ulps by bisection so that hi is the first representable point with F >= 0
        for (int it = 0; it < 4; ++it) {
            const double m = lo + 0.5 * (hi - lo);
            if (m == lo || m == hi) break;
            if (imp_F<MODE>(T, S, F, c, m) < 0.0) lo = m; else hi = m;
        }
        const double theta = hi;
        double frac[3]; int cl;
        const double de = imp_loss<MODE>(T, S, F, c, theta, frac, &cl);
        clamped |= cl;
        de_sum[0] += de; de_sum[1] += de * frac[0]; de_sum[2] += de * frac[1]; de_sum[3] += de * frac[2];
        thi = thi - g * (c.q * (thi - theta));
        the = theta;
    }
    const double wgt = rho * vol;
#pragma unroll
    for (int k = 0; k < 4; ++k) acc.lum[k] += de_sum[k] * wgt;
    acc.flo += floored; acc.cla += clamped;
}

template <class Real, int MODE, class Fetch, int THREADS>
__global__ void __launch_bounds__(THREADS)
cool_implicit_kernel(const DevTable T, const DevConst K, const StepConst S, const CellPtrs C, double *partials, unsigned *ticket, cool_diag *d_diag)
{
    extern __shared__ __align__(16) unsigned char smem_imp[];
    const Fetch F(T, smem_imp);
    if (Fetch::kSmem) __syncthreads();
    DiagAcc acc;
    const long long stride = (long long)gridDim.x * THREADS;
    for (long long c = (long long)blockIdx.x * THREADS + threadIdx.x; c < C.ncell; c += stride) {
        double the = (double)((const Real *)C.the_in)[c], thi = (double)((const Real *)C.thi_in)[c];
        const double rho = (double)((const Real *)C.rho)[c], bsq = (double)((const Real *)C.bsq)[c];
        const double rr = S.has_r ? (double)((const Real *)C.r)[c] : 0.0, vv = S.has_vol ? (double)((const Real *)C.vol)[c] : 1.0;
        implicit_cell<MODE, Fetch>(T, K, S, F, rho, bsq, the, thi, rr, vv, acc);
        ((Real *)C.the_out)[c] = (Real)the;
        ((Real *)C.thi_out)[c] = (Real)thi;
    }
    if (d_diag) reduce_diag(acc, S.lum_k, partials, ticket, d_diag);
}

template <class Real, int MODE, class Fetch>
static cudaError_t launch_implicit_one(const LaunchCtx &L, size_t smem)
{
    constexpr int THREADS = 256;
    auto kern = cool_implicit_kernel<Real, MODE, Fetch, THREADS>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    int occ = 0;
    cudaError_t eo = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, THREADS, smem);
    if (eo != cudaSuccess) return eo;
    if (occ < 1) occ = 1;
    const LaunchArgs &a = *L.a;
    // cells differ widely in iteration count: several waves of small blocks balance better than one persistent wave
    long long need = (a.ncell + THREADS - 1) / THREADS;
    const long long cap = (long long)L.t->sm_count * (occ * 8 < 32 ? occ * 8 : 32);     // <= the diagnostics workspace (32 blocks per SM)
    const int grid = (int)(need < 1 ? 1 : (need < cap ? need : cap));
    CellPtrs C{a.rho, a.bsq, a.the_in, a.thi_in, a.r, a.vol, a.the_out, a.thi_out, a.ncell};
    kern<<<grid, THREADS, smem, L.st>>>(L.t->dev, L.t->cst, *L.S, C, a.partials, a.ticket, a.d_diag);
    return cudaGetLastError();
}

cudaError_t launch_implicit(const LaunchCtx &L, int mode, cool_variant v, cool_dtype dt);

}  // namespace cool
