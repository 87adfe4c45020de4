// cool_implicit.cuh — the implicit cooling scheme (COOL_SCHEME_IMPLICIT; PAPER.md L185 (ii), L369; reading C-18 of
// DESIGN.md): one thread per cell of the SoA stream, the table read through the lookup policies of the fp64 explicit
// path; fp64 arithmetic for fp64 cells (first part of this file), fp32 arithmetic on the T' tables for fp32 cells (second part).
//
// Per sub-step h, from the start state (Theta_e, Theta_i):
//   q        = a/(1 + a g),  a = h K C(Theta_e, Theta_i),  g = (gamma_i - 1)/(gamma_e - 1)      (Coulomb: coefficient at
//              the start state, driving difference at the end state  =>  transfer x = q (Theta_i - theta))
//   loss(th) = h th Lambda(rho, th_c, bsq, Theta_i) (gamma_e - 1)/(m_e/m_p rho th_c),  th_c = th clamped to the table's
//              Theta_e range (the cooling time is held outside the range, which keeps the root positive)
//   theta    = root of  F(th) = th - Theta_e + loss(th) - q (Theta_i - th)  in (0, Theta_e + q Theta_i]
//   Theta_e' = theta,  Theta_i' = Theta_i - g q (Theta_i - theta);  no limiter.
// F(0) < 0 <= F(Theta_e + q Theta_i) always.  Inside one Theta_e interval of the table every channel is linear in the
// interval coordinate once (rho, bsq[, Theta_i]) are contracted, so the solve is: (1) a galloping, then binary, search over the table's
// Theta_e NODES for the interval that brackets the root (one contraction per probed node), (2) inside that interval,
// Illinois-type false position with a bisection safeguard on values that need no further table access, until the bracket
// is two ulps wide (outside the table range F is linear: closed form).  F' >= 1 wherever the loss does not decrease
// with Theta_e, so the answer is within rounding of the root; where Lambda is not monotone several roots can exist
// and any of them is a solution of the scheme.
#pragma once
#include "cool_f32.cuh"

namespace cool {

// The (rho, bsq[, Theta_i]) contraction of the table at Theta_e node i: within one Theta_e interval every channel is
// linear in the interval coordinate w, so a root solve needs the table only at the two nodes of the interval.
template <int MODE, class Fetch>
__device__ __forceinline__ void imp_node(const Fetch &F, const Loc64 &r, const Loc64 &b, const Loc64 &ii, int i, double (&y)[3])
{
    y[0] = y[1] = y[2] = 0.0;
    if constexpr (MODE == 3) {
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int cr = c >> 1, cb = c & 1;
            y[0] += (cr ? r.w : 1.0 - r.w) * (cb ? b.w : 1.0 - b.w) * (double)F.at1(r.i + cr, i, b.i + cb);
        }
    } else {
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const int cr = c >> 2, ci = (c >> 1) & 1, cb = c & 1;
            const double pw = (cr ? r.w : 1.0 - r.w) * (ci ? ii.w : 1.0 - ii.w) * (cb ? b.w : 1.0 - b.w);
            const float4 v = F.at4(r.i + cr, i, ii.i + ci, b.i + cb);
            y[0] += pw * v.x; y[1] += pw * v.y; y[2] += pw * v.z;
        }
    }
}

struct ImpStep { double rho, thi0, q, R; };      // fixed over one sub-step: R = Theta_e + q Theta_i

// Radiative loss of Theta_e over h at trial state th, from the channel logs y at th_c (th clamped to the table range)
template <int MODE>
__device__ __forceinline__ double imp_loss_y(const StepConst &S, const ImpStep &c, double th, double thc, const double (&y)[3], double *frac)
{
    double lam;
    if constexpr (MODE == 3) {
        lam = exp10(y[0]);
    } else {
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
__device__ void implicit_cell(const DevTable &T, const DevConst &K, const StepConst &S, const Fetch &F,
                              double rho, double bsq, double &the, double &thi, double r, double vol, DiagAcc &acc, long long cell,
                              unsigned char *flags)
{
    if (flags) flags[cell] = 0;
    if (isnan(rho) || isnan(bsq) || isnan(the) || isnan(thi)) { the = thi = __longlong_as_double(0x7ff8000000000000LL); return; }
    if (!(rho > 0.0)) return;
    const AxisCoef &ax = T.ax[CAX_THE];
    const int n = ax.n;
    const Loc64 lr = locate64(T.ax[CAX_RHO], rho), lb = locate64(T.ax[CAX_BSQ], bsq);
    Loc64 li{0, 0.0, 0};
    const double g = S.gi1 / S.ge1;
    int floored = 0, clamped = lr.clamped | lb.clamped;
    double de_sum[4] = {0, 0, 0, 0};
    auto node_theta = [&](int i) { return exp10(ax.lo10 + (double)i / ax.inv10); };
    for (int s = 0; s < S.nsub; ++s) {
        bool flo = false;
        if (S.hfloor2 > 0.0 && r > 0.0) {
            const double ok = r / (r * sqrt(r) + S.spin);            // Omega_K r
            if ((the + thi) * S.mr < S.hfloor2 * ok * ok) { flo = true; floored = 1; }
        }
        if constexpr (MODE == 4) { li = locate64(T.ax[CAX_THI], thi); clamped |= li.clamped; }
        double C = 0.0;
        if (S.coulomb == 1) C = coulomb_C_table64(T, the, thi);
        else if (S.coulomb == 2) C = coolphys::coulomb_C(the, thi / K.units.ion_theta_mass_ratio);
        const double a = S.coul_kh * rho * C;
        ImpStep c{rho, thi, a / (1.0 + a * g), 0.0};
        c.R = the + c.q * thi;
        if (!(c.R > 0.0)) continue;
        const double opq = 1.0 + c.q;

        double theta, de = 0.0, frac[3] = {0.0, 0.0, 0.0};
        if (flo) {
            theta = c.R / opq;                                       // no radiative sink this sub-step
        } else {
            // 1. the Theta_e interval that brackets the root: binary search over the nodes below R
            //    (F(0) < 0 and F(th >= R) >= 0 always; index -1 stands for theta = 0, imax + 1 for min(node, R))
            int imax = -1;
            if (c.R > exp10(ax.lo10)) {
                const double tR = (log10(c.R) - ax.lo10) * ax.inv10;
                imax = tR >= (double)(n - 1) ? n - 1 : (int)tR;
            }
            int ilo = -1, ihi = imax + 1;
            double ya[3] = {0, 0, 0}, yb[3] = {0, 0, 0};
            bool have_b = false;
            auto probe = [&](int m) {                        // F at node m; narrows [ilo, ihi]; true when F < 0 there
                double ym[3];
                imp_node<MODE>(F, lr, lb, li, m, ym);
                const double tm = node_theta(m);
                const double fm = tm * opq - c.R + imp_loss_y<MODE>(S, c, tm, tm, ym, nullptr);
                if (fm < 0.0) { ilo = m; ya[0] = ym[0]; ya[1] = ym[1]; ya[2] = ym[2]; return true; }
                ihi = m; yb[0] = ym[0]; yb[1] = ym[1]; yb[2] = ym[2]; have_b = true;
                return false;
            };
            // gallop down from the node just below R (weak cooling leaves the root in the interval that holds R: one probe),
            // then bisect what is left
            for (int m = imax, step = 1; m >= 0; m -= step, step <<= 1)
                if (probe(m)) break;
            while (ihi - ilo > 1) probe((ilo + ihi) >> 1);
            if (ilo == -1 || ilo == n - 1) {
                // 2a. outside the table range the cooling time is held: F is linear, closed form
                const int e = ilo == -1 ? 0 : n - 1;
                double ye[3];
                if (ilo == -1 && have_b && ihi == 0) { ye[0] = yb[0]; ye[1] = yb[1]; ye[2] = yb[2]; }
                else if (ilo == n - 1) { ye[0] = ya[0]; ye[1] = ya[1]; ye[2] = ya[2]; }
                else imp_node<MODE>(F, lr, lb, li, e, ye);
                const double te = node_theta(e);
                const double hr = imp_loss_y<MODE>(S, c, te, te, ye, frac) / te;      // h rhat at the edge
                theta = c.R / (opq + hr);
                de = theta * hr;
                clamped |= (theta != te);
            } else {
                // 2b. inside interval ilo: channels linear in w; Illinois false position with a bisection safeguard
                if (!(have_b && ihi == ilo + 1)) imp_node<MODE>(F, lr, lb, li, ilo + 1, yb);
                const double dy[3] = {yb[0] - ya[0], yb[1] - ya[1], yb[2] - ya[2]};
                auto Fseg = [&](double th, double *fr) {
                    double w = (log10(th) - ax.lo10) * ax.inv10 - (double)ilo;
                    w = fmin(fmax(w, 0.0), 1.0);
                    const double y[3] = {ya[0] + w * dy[0], ya[1] + w * dy[1], ya[2] + w * dy[2]};
                    return imp_loss_y<MODE>(S, c, th, th, y, fr);
                };
                double lo = node_theta(ilo), hi = fmin(node_theta(ilo + 1), c.R);
                double flo_ = lo * opq - c.R + Fseg(lo, nullptr), fhi = hi * opq - c.R + Fseg(hi, nullptr);
                if (!(flo_ < 0.0)) { hi = lo; fhi = 0.0; }           // rounding at the node: the node is the root
                if (fhi <= 2.3e-16 * c.R) fhi = 0.0;                 // weak cooling: F at the bracket end is already rounding noise
                int side = 0, stall = 0;
                for (int it = 0; it < 200 && fhi != 0.0; ++it) {
                    const double width = hi - lo;
                    if (!(width > 4.4408920985006262e-16 * hi)) break;       // two ulps
                    double m = hi - fhi * (width / (fhi - flo_));
                    if (!(m > lo && m < hi) || stall >= 2) { m = lo + 0.5 * width; stall = 0; }   // bisect when the bracket stalls
                    if (m == lo || m == hi) break;
                    const double fm = m * opq - c.R + Fseg(m, nullptr);
                    if (fabs(fm) <= 2.3e-16 * c.R) { hi = m; break; }        // below ulp(R) the sign of F is rounding noise
                    if (fm < 0.0) { lo = m; flo_ = fm; if (side == -1) fhi *= 0.5; side = -1; }
                    else { hi = m; fhi = fm; if (side == 1) flo_ *= 0.5; side = 1; }
                    stall = (hi - lo > 0.5 * width) ? stall + 1 : 0;
                }
                theta = hi;
                de = Fseg(theta, frac);
            }
        }
        de_sum[0] += de; de_sum[1] += de * frac[0]; de_sum[2] += de * frac[1]; de_sum[3] += de * frac[2];
        thi = thi - g * (c.q * (thi - theta));
        the = theta;
    }
    const double wgt = rho * vol;
#pragma unroll
    for (int k = 0; k < 4; ++k) acc.lum[k] += de_sum[k] * wgt;
    acc.flo += floored; acc.cla += clamped;
    shell_add(S, cell, de_sum, wgt, MODE == 4);
    if (flags) flags[cell] = (unsigned char)((floored << 1) | (clamped << 2));
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
        implicit_cell<MODE, Fetch>(T, K, S, F, rho, bsq, the, thi, rr, vv, acc, c, d_diag ? C.flags : nullptr);
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
    CellPtrs C{a.rho, a.bsq, a.the_in, a.thi_in, a.r, a.vol, a.the_out, a.thi_out, a.ncell, a.flags};
    kern<<<grid, THREADS, smem, L.st>>>(L.t->dev, L.t->cst, *L.S, C, a.partials, a.ticket, a.d_diag);
    return cudaGetLastError();
}

// ==========================================================================================
// fp32 cells: the same solve in fp32 on the T' tables (log2 of the rate per unit electron energy, cool_internal.h), where
// h Lambda/u_e = 2^(interp T' + log2 h + rho clamp correction) needs no large-number cancellation.  Same structure:
// binary search over the Theta_e nodes, then false position inside the interval on the contracted column values.
// The bracket is refined to a few fp32 ulps, so the result is within ~1e-6 of the root (tolerance 1e-5, as for the
// explicit fp32 path).  Fetch is one of the fp64 path's lookup policies, constructed over the T' arrays.
// ==========================================================================================
struct Imp32 { float rho, thi0, q, R, opq, kc, hf; };    // kc: clamp correction of the rho axis (log2), hf: h as a factor

template <int MODE, class Fetch>
__device__ __forceinline__ void imp32_node(const Fetch &F, const Loc32 &r, const Loc32 &b, const Loc32 &ii, int ir, int ib, int iii, int i, float (&y)[3])
{
    if constexpr (MODE == 3) {
        const float a0 = lerp(b.w, F.at1(ir, i, ib), F.at1(ir, i, ib + 1)), a1 = lerp(b.w, F.at1(ir + 1, i, ib), F.at1(ir + 1, i, ib + 1));
        y[0] = lerp(r.w, a0, a1); y[1] = y[2] = 0.f;
    } else {
        float v[2][2][3];
#pragma unroll
        for (int cr = 0; cr < 2; ++cr)
#pragma unroll
            for (int ci = 0; ci < 2; ++ci) {
                const float4 t0 = F.at4(ir + cr, i, iii + ci, ib), t1 = F.at4(ir + cr, i, iii + ci, ib + 1);
                v[cr][ci][0] = lerp(b.w, t0.x, t1.x); v[cr][ci][1] = lerp(b.w, t0.y, t1.y); v[cr][ci][2] = lerp(b.w, t0.z, t1.z);
            }
#pragma unroll
        for (int k = 0; k < 3; ++k) y[k] = lerp(r.w, lerp(ii.w, v[0][0][k], v[0][1][k]), lerp(ii.w, v[1][0][k], v[1][1][k]));
    }
}

// 3-D tables in global memory with the quad layout (cool_internal.h: q3[r][e][b] = {T'(r,e,b), T'(r,e,b+1), T'(r,e+1,b),
// T'(r,e+1,b+1)}, edges duplicated): the column values at Theta_e nodes i AND i+1 from two 128-bit loads — a probe of node
// i brings the other end of its interval along, which is the whole bracket when the root lies in the interval below R.
__device__ __forceinline__ void imp32_pair3(const float4 *q3, int sr, int se, const Loc32 &r, const Loc32 &b, int ir, int ib, int i, float &y_i, float &y_i1)
{
    const float4 *p = q3 + (unsigned)(ir * sr + i * se + ib);
    const float4 q0 = ldg_f4(p), q1 = ldg_f4(p + sr);
    y_i = lerp(r.w, lerp(b.w, q0.x, q0.y), lerp(b.w, q1.x, q1.y));
    y_i1 = lerp(r.w, lerp(b.w, q0.z, q0.w), lerp(b.w, q1.z, q1.w));
}
template <int MODE, class Fetch> struct ImpPairFetch { static constexpr bool value = false; };
template <> struct ImpPairFetch<3, FetchGlobal> { static constexpr bool value = true; };

// loss(th)/th = h Lambda(th_c)/u_e(th_c) from the channel values y at th_c; optional process shares
template <int MODE>
__device__ __forceinline__ float imp32_rate(const F32Const &S, const Imp32 &c, float thc, const float (&y)[3], float *frac)
{
    // h multiplies the power of two instead of joining its exponent: one rounding less at magnitude ~40, which matters
    // here because in the strongly cooled limit theta' ~ R/rate carries the full relative error of the rate
    if constexpr (MODE == 3) {
        return ex2_approx(y[0] + c.kc) * c.hf;
    } else {
        const float rbr = ex2_approx(fminf(y[0] + c.kc, 100.f)) * c.hf;
        const float esy = y[1] + c.kc;
        const float rsy = ex2_approx(fminf(esy + y[2], 100.f)) * c.hf;                        // eta * Q_syn
        const float rthin = rbr + rsy;                                                        // eq 10
        const float num = fmaf(S.ae, thc, S.ai * c.thi0), den = fmaf(S.be, thc, fmaf(S.bi, c.thi0, 1.f));
        const float rcs = c.rho * (num * rsqrt_approx(num * den));                            // rho c_s   (eqs 13-14)
        const float th3 = fmaxf(thc * thc * thc, 1e-30f);
        const float tau_abs = rthin * (S.inv_kB * rcs) * rcp_approx(th3);                     // eq 12
        const float tau_sca = S.ksca * rcs;
        if (frac) {
            const float inv = rcp_approx(fmaxf(rthin, 1e-37f));
            const float rs0 = ex2_approx(fminf(esy, 100.f)) * c.hf;
            frac[0] = rbr * inv; frac[1] = rs0 * inv; frac[2] = (rsy - rs0) * inv;
        }
        return rthin * rcp_approx(fmaf(tau_abs, fmaf(1.5f, tau_abs + tau_sca, 1.7320508f), 1.f));   // eq 11
    }
}

// ---- accurate rate inside the bracketing interval -------------------------------------------------------------------------
// In the strongly cooled limit theta' ~ R/rate carries the full relative error of rate = 2^y, and in fp32 y (|y| up to ~40)
// is good to 2-4e-6 only: the roundings of the node contraction and of the exponent sum (measured: 4e-6 per sub-step, adding
// over sub-steps).  The fp32 search over the nodes only has to find the bracketing Theta_e interval; inside it the two node
// values are contracted once more in fp64 and the exponent y = a + w (b - a) + log2 h + clamp terms is summed in fp64; 2^y
// then takes the integer part exactly and the fraction (|f| <= 1/2) from MUFU.EX2 (2e-7).  Everything else stays fp32 (the
// interval weight w is harmless: a weight error moves rate and theta together and cancels to first order in the root).
__device__ __forceinline__ float imp_exp2_d(double y)
{
    y = fmin(fmax(y, -120.0), 120.0);
    const double yi = rint(y);
    return __int_as_float(__float_as_int(ex2_approx((float)(y - yi))) + ((int)yi << 23));      // 2^f in [0.70, 1.42] scaled by 2^yi (|yi| <= 120)
}
__device__ __forceinline__ double imp_dlerp(float w, float a, float b) { return fma((double)w, (double)b - (double)a, (double)a); }
__device__ __forceinline__ double imp_dlerp(float w, double a, double b) { return fma((double)w, b - a, a); }

template <int MODE, class Fetch>
__device__ __forceinline__ void imp_node_d(const Fetch &F, const Loc32 &r, const Loc32 &b, const Loc32 &ii, int ir, int ib, int iii, int i, double (&y)[3])
{
    if constexpr (MODE == 3) {
        y[0] = imp_dlerp(r.w, imp_dlerp(b.w, F.at1(ir, i, ib), F.at1(ir, i, ib + 1)), imp_dlerp(b.w, F.at1(ir + 1, i, ib), F.at1(ir + 1, i, ib + 1)));
        y[1] = y[2] = 0.0;
    } else {
        double v[2][2][3];
#pragma unroll
        for (int cr = 0; cr < 2; ++cr)
#pragma unroll
            for (int ci = 0; ci < 2; ++ci) {
                const float4 t0 = F.at4(ir + cr, i, iii + ci, ib), t1 = F.at4(ir + cr, i, iii + ci, ib + 1);
                v[cr][ci][0] = imp_dlerp(b.w, t0.x, t1.x); v[cr][ci][1] = imp_dlerp(b.w, t0.y, t1.y); v[cr][ci][2] = imp_dlerp(b.w, t0.z, t1.z);
            }
#pragma unroll
        for (int k = 0; k < 3; ++k) y[k] = imp_dlerp(r.w, imp_dlerp(ii.w, v[0][0][k], v[0][1][k]), imp_dlerp(ii.w, v[1][0][k], v[1][1][k]));
    }
}

// imp32_rate with the channel exponents y (+ kd = log2 h + rho clamp correction) given in fp64
template <int MODE>
__device__ __forceinline__ float imp32_rate_d(const F32Const &S, const Imp32 &c, float thc, const double (&y)[3], double kd, float *frac)
{
    if constexpr (MODE == 3) {
        return imp_exp2_d(y[0] + kd);
    } else {
        const float rbr = imp_exp2_d(fmin(y[0] + kd, 100.0));
        const double esy = y[1] + kd;
        const float rsy = imp_exp2_d(fmin(esy + y[2], 100.0));                                // eta * Q_syn
        const float rthin = rbr + rsy;                                                        // eq 10
        const float num = fmaf(S.ae, thc, S.ai * c.thi0), den = fmaf(S.be, thc, fmaf(S.bi, c.thi0, 1.f));
        const float rcs = c.rho * (num * rsqrt_approx(num * den));                            // rho c_s   (eqs 13-14)
        const float th3 = fmaxf(thc * thc * thc, 1e-30f);
        const float tau_abs = rthin * (S.inv_kB * rcs) * rcp_approx(th3);                     // eq 12
        const float tau_sca = S.ksca * rcs;
        if (frac) {
            const float inv = rcp_approx(fmaxf(rthin, 1e-37f));
            const float rs0 = imp_exp2_d(fmin(esy, 100.0));
            frac[0] = rbr * inv; frac[1] = rs0 * inv; frac[2] = (rsy - rs0) * inv;
        }
        return rthin * rcp_approx(fmaf(tau_abs, fmaf(1.5f, tau_abs + tau_sca, 1.7320508f), 1.f));   // eq 11
    }
}

constexpr float kImpF32Rate = 0.03f;      // radiated fraction h Lambda/u_e below which the fp32 rate is accurate enough for the implicit root

template <int MODE, class Fetch>
__device__ void implicit_cell_f32(const DevTable &T, const StepConst &S, const F32Const &S32, const Fetch &F,
                                  float rho, float bsq, float &the, float &thi, float r, float vol, DiagAcc &acc, long long cell,
                                  unsigned char *flags, double k0d, bool want_diag)   // k0d = log2 h in fp64
{
    const float chk = (bsq + the) + (thi + rho);
    if (chk != chk || !(rho > 0.f)) {                // NaN in -> NaN out, no matter -> unchanged; no events
        if (chk != chk) the = thi = __int_as_float(0x7fc00000);
        if (flags) flags[cell] = 0;
        return;
    }
    const int one_bits = 0x3f800000;
    const AxisCoef &ax = T.ax[CAX_THE];
    const int n = ax.n;
    bool clamped = false; int floored = 0;
    const Loc32 lr = locate32<true>(T.ax[CAX_RHO], rho, clamped, one_bits), lb = locate32<true>(T.ax[CAX_BSQ], bsq, clamped, one_bits);
    const int ir = (int)lr.fi, ib = (int)lb.fi;
    Loc32 li{0.f, 0.f, 0.f, 0.f}; int iii = 0;
    const float g = S32.gi1_over_ge1;
    float de_sum[4] = {0.f, 0.f, 0.f, 0.f};
    auto node_theta = [&](int i) { return ex2_approx(fmaf((float)i - ax.cf, ax.d2f, ax.e0)); };
    for (int s = 0; s < S32.nsub; ++s) {
        bool flo = false;
        if (S32.hfloor2 > 0.f && r > 0.f) {
            const float ok = __fdividef(r, fmaf(r, sqrtf(r), S32.spin));
            if ((the + thi) * S32.mr < S32.hfloor2 * ok * ok) { flo = true; floored = 1; }
        }
        if constexpr (MODE == 4) { li = locate32<true>(T.ax[CAX_THI], thi, clamped, one_bits); iii = (int)li.fi; }
        float C = 0.f;
        if (S32.coulomb == 1) {
            bool dummy = false;
            const Loc32 ca = locate32<false>(T.cax[0], thi, dummy, one_bits), cb = locate32<false>(T.cax[1], the, dummy, one_bits);
            C = coulomb_C32<0, false>(T.cax[1].n, 0, T.fcoul, 0u, ca, cb);
        } else if (S32.coulomb == 2) {
            C = (float)coolphys::coulomb_C((double)the, (double)thi / S32.ion_ratio);
        }
        const float a = S32.coul_kh * rho * C;
        Imp32 c;
        c.rho = rho; c.thi0 = thi; c.q = a / (1.f + a * g); c.R = fmaf(c.q, thi, the); c.opq = 1.f + c.q;
        c.kc = lr.d * T.ax[CAX_RHO].d2f; c.hf = ex2_approx(S32.k0);
        auto kd_of = [&]() { return (double)lr.d * (double)T.ax[CAX_RHO].d2f + k0d; };     // log2 h + clamp term, fp64: only the fp64-exponent paths form it
        if (!(c.R > 0.f)) continue;
        float theta, rate = 0.f, frac[3] = {0.f, 0.f, 0.f};
        if (flo) {
            theta = c.R / c.opq;
        } else {
            const float tR = coord32(ax, c.R, one_bits);
            const int imax = tR >= (float)(n - 1) ? n - 1 : (tR < 0.f ? -1 : (int)tR);
            int ilo = -1, ihi = imax + 1;
            float ya[3] = {0.f, 0.f, 0.f}, yb[3] = {0.f, 0.f, 0.f};
            float ra = 0.f, ta = 0.f;                        // rate and Theta_e at node ilo, as the probe that set ilo computed them
            bool have_b = false;
            const bool pair = ImpPairFetch<MODE, Fetch>::value && T.q3 != nullptr;       // warp-uniform
            int pa_idx = -2; float pa_lo = 0.f, pa_hi = 0.f;                            // the last pair loaded: nodes pa_idx, pa_idx + 1
            auto probe = [&](int m) {                        // F at node m; narrows [ilo, ihi]; true when F < 0 there
                float ym[3];
                if (pair) { imp32_pair3(T.q3, T.s_rho, T.s_the, lr, lb, ir, ib, m, pa_lo, pa_hi); pa_idx = m; ym[0] = pa_lo; ym[1] = ym[2] = 0.f; }
                else imp32_node<MODE>(F, lr, lb, li, ir, ib, iii, m, ym);
                const float tm = node_theta(m);
                const float rm = imp32_rate<MODE>(S32, c, tm, ym, nullptr);
                const float fm = fmaf(tm, c.opq, -c.R) + tm * rm;
                if (fm < 0.f) { ilo = m; ya[0] = ym[0]; ya[1] = ym[1]; ya[2] = ym[2]; ra = rm; ta = tm; return true; }
                ihi = m; yb[0] = ym[0]; yb[1] = ym[1]; yb[2] = ym[2]; have_b = true;
                return false;
            };
            // gallop down from the node just below R (weak cooling leaves the root in the interval that holds R: one probe),
            // then bisect what is left
            for (int m = imax, step = 1; m >= 0; m -= step, step <<= 1)
                if (probe(m)) break;
            while (ihi - ilo > 1) probe((ilo + ihi) >> 1);
            if (ilo == -1 || ilo == n - 1) {
                const int e = ilo == -1 ? 0 : n - 1;
                float ye[3];
                if (ilo == -1 && have_b) { ye[0] = yb[0]; ye[1] = yb[1]; ye[2] = yb[2]; }
                else if (ilo == n - 1) { ye[0] = ya[0]; ye[1] = ya[1]; ye[2] = ya[2]; }
                else imp32_node<MODE>(F, lr, lb, li, ir, ib, iii, e, ye);
                const float te = node_theta(e);
                double yed[3];
                imp_node_d<MODE>(F, lr, lb, li, ir, ib, iii, e, yed);
                rate = imp32_rate_d<MODE>(S32, c, te, yed, kd_of(), frac);           // cooling time held outside the range
                theta = c.R / (c.opq + rate);
                clamped = true;
            } else {
                if (pair) {
                    if (pa_idx != ilo) imp32_pair3(T.q3, T.s_rho, T.s_the, lr, lb, ir, ib, ilo, pa_lo, pa_hi);
                    ya[0] = pa_lo; yb[0] = pa_hi;
                } else if (!have_b) imp32_node<MODE>(F, lr, lb, li, ir, ib, iii, ilo + 1, yb);
                const float dy[3] = {yb[0] - ya[0], yb[1] - ya[1], yb[2] - ya[2]};
                float lo = ta, hi = fminf(node_theta(ilo + 1), c.R);
                // The root moves with the rate by d ln(theta) = -[rate/(opq + rate)] d ln(rate), and fp32 exponents give the rate to
                // <= 1e-4 even in the steepest interval (5e-6 nodes x 16 log2 units), so where the radiated fraction is below
                // kImpF32Rate over the bracket [lo, hi] the fp32 rate holds 1e-5 with a wide margin; elsewhere the bracketing
                // nodes are contracted once more in fp64 and the exponent is summed in fp64.  Inside a table interval every process
                // is a power law of Theta_e, so the bracket's two ends bound the rate (the bridged sum of a 4-D table can exceed both
                // only marginally; the threshold leaves a factor 3): the lower end is what the probe of node ilo computed, the
                // upper end is the first evaluation of the iteration anyway.
                bool f32ok = true;
                double yad[3] = {0.0, 0.0, 0.0}, dyd[3] = {0.0, 0.0, 0.0}, kd = 0.0;
                auto Rate = [&](float th, float *fr) {
                    const float w32 = fminf(fmaxf(coord32(ax, th, one_bits) - (float)ilo, 0.f), 1.f);
                    if (f32ok) {
                        const float y32[3] = {fmaf(w32, dy[0], ya[0]), fmaf(w32, dy[1], ya[1]), fmaf(w32, dy[2], ya[2])};
                        return imp32_rate<MODE>(S32, c, th, y32, fr);
                    }
                    const double w = (double)w32;
                    const double y[3] = {fma(w, dyd[0], yad[0]), fma(w, dyd[1], yad[1]), fma(w, dyd[2], yad[2])};
                    return imp32_rate_d<MODE>(S32, c, th, y, kd, fr);
                };
                const float noise = 1.2e-7f * c.R;              // F is a difference of terms of size R: below ~ulp(R) its sign is
                                                                // rounding noise and the point is as good a root as fp32 can tell
                                                                // (F' >= opq + rate where the rate does not fall with Theta_e, so
                                                                // the error in theta is <= ulp(theta))
                float rhi = Rate(hi, nullptr);
                float flo0 = fmaf(lo, c.opq, -c.R) + lo * ra;                  // < 0: that is how the probe chose ilo
                if (!(fmaxf(ra, rhi) < kImpF32Rate)) {
                    double ybd[3];
                    imp_node_d<MODE>(F, lr, lb, li, ir, ib, iii, ilo, yad);
                    imp_node_d<MODE>(F, lr, lb, li, ir, ib, iii, ilo + 1, ybd);
                    dyd[0] = ybd[0] - yad[0]; dyd[1] = ybd[1] - yad[1]; dyd[2] = ybd[2] - yad[2];
                    f32ok = false; kd = kd_of();
                    rhi = Rate(hi, nullptr);
                    flo0 = fmaf(lo, c.opq, -c.R) + lo * Rate(lo, nullptr);
                }
                float fhi = fmaf(hi, c.opq, -c.R) + hi * rhi;
                float rate_hi = rhi;                            // the rate at `hi` wherever the iteration leaves it (3-D tables)
                if (fhi > noise) {
                    if (!(flo0 < 0.f)) { hi = lo; fhi = 0.f; rhi = f32ok ? ra : Rate(lo, nullptr); rate_hi = rhi; }   // rounding at the lower node: it is the root
                    if constexpr (MODE == 3) {
                        // inside the interval the rate is an exact power law, rate ~ theta^p with p = dy invf, so
                        // F' = opq + rate (1 + p): Newton steps, kept inside the bracket
                        const float p1 = fmaf(dy[0], ax.invf, 1.f);
                        float x = hi, fx = fhi, rx = rhi;
                        for (int it = 0; it < 40 && fabsf(fx) > noise; ++it) {
                            const float d = fmaf(rx, p1, c.opq);
                            float m = d > 0.25f * c.opq ? x - fx / d : lo + 0.5f * (hi - lo);
                            if (!(m > lo && m < hi)) m = lo + 0.5f * (hi - lo);
                            if (m == lo || m == hi) break;
                            const float rm = Rate(m, nullptr), fm = fmaf(m, c.opq, -c.R) + m * rm;
                            if (fm < 0.f) lo = m; else hi = m;
                            const bool done = fabsf(m - x) <= 1.2e-7f * m;
                            x = m; fx = fm; rx = rm;
                            if (done) break;
                        }
                        hi = x; rate_hi = rx;
                    } else {
                        float flo_ = flo0;
                        int side = 0, stall = 0;
                        for (int it = 0; it < 48 && fhi != 0.f; ++it) {
                            const float width = hi - lo;
                            if (!(width > 2.4e-7f * hi)) break;                        // two fp32 ulps
                            float m = hi - fhi * (width / (fhi - flo_));
                            if (!(m > lo && m < hi) || stall >= 2) { m = lo + 0.5f * width; stall = 0; }   // bisect when the bracket stalls
                            if (m == lo || m == hi) break;
                            const float fm = fmaf(m, c.opq, -c.R) + m * Rate(m, nullptr);
                            if (fabsf(fm) <= noise) { hi = m; break; }
                            if (fm < 0.f) { lo = m; flo_ = fm; if (side == -1) fhi *= 0.5f; side = -1; }
                            else { hi = m; fhi = fm; if (side == 1) flo_ *= 0.5f; side = 1; }
                            stall = (hi - lo > 0.5f * width) ? stall + 1 : 0;
                        }
                    }
                }
                theta = hi;
                if constexpr (MODE == 3) rate = rate_hi;        // no process split on a 3-D table: the last evaluation is the rate at theta
                else rate = Rate(theta, frac);
            }
        }
        const float de = theta * rate;
        de_sum[0] += de; de_sum[1] = fmaf(de, frac[0], de_sum[1]); de_sum[2] = fmaf(de, frac[1], de_sum[2]); de_sum[3] = fmaf(de, frac[2], de_sum[3]);
        // Theta_i' = Theta_i - g q (Theta_i - theta) in its cancellation-free form (a >> 1 drives Theta_i' -> theta)
        thi = fmaf(g * a, theta, thi) / fmaf(a, g, 1.f);
        the = theta;
    }
    if (!want_diag) return;                          // kernel argument: warp-uniform
    const double wgt = (double)rho * (double)vol;
    const double ds[4] = {(double)de_sum[0], (double)de_sum[1], (double)de_sum[2], (double)de_sum[3]};
#pragma unroll
    for (int k = 0; k < (MODE == 4 ? 4 : 1); ++k) acc.lum[k] += ds[k] * wgt;      // no process split on a 3-D table
    acc.flo += floored; acc.cla += clamped ? 1 : 0;
    shell_add(S, cell, ds, wgt, MODE == 4);
    if (flags) flags[cell] = (unsigned char)((floored << 1) | (clamped ? 4 : 0));
}

// Resident blocks per SM: the solve is bound by the latency of its dependent chains, so warps count.  3-D tables fit 80 registers
// (three blocks of 256 threads: 24 warps, 20 % faster than two); the 4-D solve needs 128 (two blocks; three measured no gain).
template <int MODE, class Fetch, int THREADS>
__global__ void __launch_bounds__(THREADS, MODE == 3 ? 3 : 2)
cool_implicit_f32_kernel(const DevTable T, const StepConst S, const F32Const S32, const CellPtrs C, double *partials, unsigned *ticket, cool_diag *d_diag)
{
    extern __shared__ __align__(16) unsigned char smem_imp32[];
    DevTable Tp = T;                                 // the lookup policies of the fp64 path, pointed at the T' arrays
    Tp.lin1 = T.f1; Tp.lin4 = T.f4; Tp.tex_pt = T.ftex_pt;
    const Fetch F(Tp, smem_imp32);
    if (Fetch::kSmem) __syncthreads();
    DiagAcc acc;
    const double k0d = log2(S.h);
    const long long stride = (long long)gridDim.x * THREADS;
    long long c = (long long)blockIdx.x * THREADS + threadIdx.x;
    // the next cell's values are requested before the current cell is solved: the solve hides the HBM latency
    float n_the = 0.f, n_thi = 0.f, n_rho = 0.f, n_bsq = 0.f, n_rr = 0.f, n_vv = 1.f;
    auto fetch = [&](long long k) {
        n_the = __ldcs((const float *)C.the_in + k); n_thi = __ldcs((const float *)C.thi_in + k);
        n_rho = __ldcs((const float *)C.rho + k); n_bsq = __ldcs((const float *)C.bsq + k);
        if (S.has_r) n_rr = __ldcs((const float *)C.r + k);
        if (S.has_vol) n_vv = __ldcs((const float *)C.vol + k);
    };
    if (c < C.ncell) fetch(c);
    for (; c < C.ncell; c += stride) {
        float the = n_the, thi = n_thi;
        const float rho = n_rho, bsq = n_bsq, rr = n_rr, vv = n_vv;
        if (c + stride < C.ncell) fetch(c + stride);
        implicit_cell_f32<MODE, Fetch>(T, S, S32, F, rho, bsq, the, thi, rr, vv, acc, c, d_diag ? C.flags : nullptr, k0d, d_diag != nullptr);
        __stcs((float *)C.the_out + c, the);
        __stcs((float *)C.thi_out + c, thi);
    }
    if (d_diag) reduce_diag(acc, S.lum_k, partials, ticket, d_diag);
}

template <int MODE, class Fetch>
static cudaError_t launch_implicit_f32_one(const LaunchCtx &L, const F32Const &S32, size_t smem)
{
    constexpr int THREADS = 256;
    auto kern = cool_implicit_f32_kernel<MODE, Fetch, THREADS>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    int occ = 0;
    cudaError_t eo = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, THREADS, smem);
    if (eo != cudaSuccess) return eo;
    if (occ < 1) occ = 1;
    const LaunchArgs &a = *L.a;
    long long need = (a.ncell + THREADS - 1) / THREADS;
    const long long cap = (long long)L.t->sm_count * (occ * 8 < 32 ? occ * 8 : 32);
    const int grid = (int)(need < 1 ? 1 : (need < cap ? need : cap));
    CellPtrs C{a.rho, a.bsq, a.the_in, a.thi_in, a.r, a.vol, a.the_out, a.thi_out, a.ncell, a.flags};
    kern<<<grid, THREADS, smem, L.st>>>(L.t->dev, *L.S, S32, C, a.partials, a.ticket, a.d_diag);
    return cudaGetLastError();
}

cudaError_t launch_implicit(const LaunchCtx &L, const F32Const &S32, int mode, cool_variant v, cool_dtype dt);


}  // namespace cool
