// cool_kernels.cu — hand-written sm_100a kernels of the per-cell cooling step (include/cool.h).
//
// One kernel template, instantiated per (cell dtype) x (table shape) x (lookup variant):
//   * cells are streamed as SoA with 128-bit L1-bypassing loads/stores, 16 B per thread per array;
//   * the table is read through one of four lookup policies (global/L2, shared memory, point
//     texture, hardware-filtered texture) or not at all (analytic);
//   * the luminosity diagnostic is reduced warp -> block -> fixed-order last-block pass, so it is
//     bit-reproducible for a given launch shape.
// No tensor cores: the step is a gather plus scalar arithmetic.
#include <cstdio>

#include "cool_internal.h"

namespace cool {

// ------------------------------------------------------------------------------------------
// Per-launch constants (host fp64 -> rounded copies for the fp32 path).
// ------------------------------------------------------------------------------------------
struct StepConst {
    // fp64 path
    double h, inv_dt, f_limit, mr, ge1, gi1, eq_frac, coul_kh, bb_k, tausca_k, h_per_cs, hth_cm;
    double ae, ai, be, bi;         // c_s^2 = (ae Th_e + ai Th_i)/(1 + be Th_e + bi Th_i)
    double hfloor2, spin;          // floor: (pi/2) h_floor^2 (Omega_K r)^2
    double lum_k;                  // lum = sum(dTheta_rad * rho * vol) * lum_k,  lum_k = mr/(ge1 dt)
    // fp32 path
    float L10h, L10l;              // log2(10) = L10h + L10l
    float ksm;                     // log2(h) - log2(mr/ge1)   (fraction-sized constant of the exponent)
    float f_limitf, mrf, eq_fracf, ge1_over_gi1, gi1_over_ge1, coul_khf;
    float aef, aif, bef, bif;
    float kB_I, kB_F;              // log2( bb_k h ge1 / (h_per_cs mr) ) split integer + fraction (MODE 4)
    float kB3_I, kB3_F;            // same with hth_cm in place of h_per_cs*c_s (unused in MODE 3 table path)
    float kscaf;                   // tau_sca = kscaf * rho * sqrt(cs2)
    float hfloor2f, spinf;
    int nsub, coulomb, want_diag, has_r, has_vol, aligned;
};

// ------------------------------------------------------------------------------------------
// Streaming cell I/O: 128-bit, no L1 allocation (cell data is touched once; L1 is for the table).
// ------------------------------------------------------------------------------------------
template <class Real> struct VecT;
template <> struct VecT<float>  { static constexpr int N = 4; using type = float4; };
template <> struct VecT<double> { static constexpr int N = 2; using type = double2; };

__device__ __forceinline__ float4 ld_stream(const float4 *p)
{
    float4 v;
    asm volatile("ld.global.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ double2 ld_stream(const double2 *p)
{
    double2 v;
    asm volatile("ld.global.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_stream(float4 *p, float4 v)
{
    asm volatile("st.global.L1::no_allocate.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ void st_stream(double2 *p, double2 v)
{
    asm volatile("st.global.L1::no_allocate.v2.f64 [%0], {%1,%2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ float &vget(float4 &v, int j) { return (&v.x)[j]; }
__device__ __forceinline__ double &vget(double2 &v, int j) { return (&v.x)[j]; }

// ------------------------------------------------------------------------------------------
// Lookup policies.  at1/at4 take canonical node indices; the policy knows the layout.
// ------------------------------------------------------------------------------------------
struct FetchGlobal {
    static constexpr bool kHw = false, kSmem = false;
    const float *p1; const float4 *p4; int sr, se, si;
    __device__ FetchGlobal(const DevTable &T, void *) : p1(T.lin1), p4(T.lin4), sr(T.s_rho), se(T.s_the), si(T.s_thi) {}
    __device__ __forceinline__ float at1(int ir, int ie, int ib) const { return __ldg(p1 + (ir * sr + ie * se + ib)); }
    __device__ __forceinline__ float4 at4(int ir, int ie, int ii, int ib) const { return __ldg(p4 + (ir * sr + ie * se + ii * si + ib)); }
};
struct FetchSmem {
    static constexpr bool kHw = false, kSmem = true;
    const float *p1; const float4 *p4; int sr, se, si;
    __device__ FetchSmem(const DevTable &T, void *smem) : p1((const float *)smem), p4((const float4 *)smem), sr(T.s_rho), se(T.s_the), si(T.s_thi)
    {
        const float4 *src = T.mode == 3 ? (const float4 *)T.lin1 : T.lin4;
        float4 *dst = (float4 *)smem;
        const unsigned n16 = T.table_bytes >> 4;          // table_bytes is padded to 16 B at create time
        for (unsigned k = threadIdx.x; k < n16; k += blockDim.x) dst[k] = __ldg(src + k);
        __syncthreads();
    }
    __device__ __forceinline__ float at1(int ir, int ie, int ib) const { return p1[ir * sr + ie * se + ib]; }
    __device__ __forceinline__ float4 at4(int ir, int ie, int ii, int ib) const { return p4[ir * sr + ie * se + ii * si + ib]; }
};
struct FetchTexPoint {
    static constexpr bool kHw = false, kSmem = false;
    cudaTextureObject_t tex; int ne;
    __device__ FetchTexPoint(const DevTable &T, void *) : tex(T.tex_pt), ne(T.ax[CAX_THE].n) {}
    __device__ __forceinline__ float at1(int ir, int ie, int ib) const { return tex3D<float>(tex, ib + 0.5f, ie + 0.5f, ir + 0.5f); }
    __device__ __forceinline__ float4 at4(int ir, int ie, int ii, int ib) const { return tex3D<float4>(tex, ib + 0.5f, ii + 0.5f, (ir * ne + ie) + 0.5f); }
};
struct FetchTexHw {
    static constexpr bool kHw = true, kSmem = false;
    cudaTextureObject_t tex; int ne;
    __device__ FetchTexHw(const DevTable &T, void *) : tex(T.tex_lin), ne(T.ax[CAX_THE].n) {}
    // MODE 3: one trilinear fetch.  MODE 4: hardware bilinear on (bsq, theta_i) at a fixed
    // (rho, theta_e) slice — the paper's scheme (L155-L159): the flattened dimension is manual.
    __device__ __forceinline__ float hw3(float tr, float te, float tb) const { return tex3D<float>(tex, tb + 0.5f, te + 0.5f, tr + 0.5f); }
    __device__ __forceinline__ float4 hw4(int ir, int ie, float ti, float tb) const { return tex3D<float4>(tex, tb + 0.5f, ti + 0.5f, (ir * ne + ie) + 0.5f); }
    __device__ __forceinline__ float at1(int, int, int) const { return 0.f; }
    __device__ __forceinline__ float4 at4(int, int, int, int) const { return make_float4(0, 0, 0, 0); }
};
struct FetchNone {   // analytic
    static constexpr bool kHw = false, kSmem = false;
    __device__ FetchNone(const DevTable &, void *) {}
};

// ------------------------------------------------------------------------------------------
// Diagnostics accumulator
// ------------------------------------------------------------------------------------------
struct DiagAcc {
    double lum[4];
    int lim, flo, cla;
    __device__ DiagAcc() : lum{0, 0, 0, 0}, lim(0), flo(0), cla(0) {}
};

// ==========================================================================================
// fp64 path: mirrors the definition step by step (tolerance 1e-12 against the oracle).
// ==========================================================================================
struct Loc64 { int i; double w; int clamped; };
__device__ __forceinline__ Loc64 locate64(const AxisCoef &a, double q)
{
    Loc64 L;
    double t = (q > 0.0) ? (log10(q) - a.lo10) * a.inv10 : -1.0;      // (x - lo)/Delta; non-positive -> lower edge
    L.clamped = 0;
    if (t < 0.0) { t = 0.0; L.clamped = 1; }
    if (t > (double)(a.n - 1)) { t = (double)(a.n - 1); L.clamped = 1; }
    int i = (int)t;
    if (i > a.n - 2) i = a.n - 2;
    L.i = i; L.w = t - (double)i;
    return L;
}

template <class Fetch>
__device__ __forceinline__ double interp3_f64(const Fetch &F, const Loc64 &r, const Loc64 &e, const Loc64 &b)
{
    if constexpr (Fetch::kHw) {
        return (double)F.hw3((float)(r.i + r.w), (float)(e.i + e.w), (float)(b.i + b.w));
    } else {
        double y = 0.0;
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            int cr = c >> 2, ce = (c >> 1) & 1, cb = c & 1;
            double pw = (cr ? r.w : 1.0 - r.w) * (ce ? e.w : 1.0 - e.w) * (cb ? b.w : 1.0 - b.w);
            y += pw * (double)F.at1(r.i + cr, e.i + ce, b.i + cb);
        }
        return y;
    }
}
template <class Fetch>
__device__ __forceinline__ void interp4_f64(const Fetch &F, const Loc64 &r, const Loc64 &e, const Loc64 &ii, const Loc64 &b, double y[3])
{
    y[0] = y[1] = y[2] = 0.0;
    if constexpr (Fetch::kHw) {
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            int cr = c >> 1, ce = c & 1;
            double pw = (cr ? r.w : 1.0 - r.w) * (ce ? e.w : 1.0 - e.w);
            float4 v = F.hw4(r.i + cr, e.i + ce, (float)(ii.i + ii.w), (float)(b.i + b.w));
            y[0] += pw * v.x; y[1] += pw * v.y; y[2] += pw * v.z;
        }
    } else {
#pragma unroll
        for (int c = 0; c < 16; ++c) {
            int cr = c >> 3, ce = (c >> 2) & 1, ci = (c >> 1) & 1, cb = c & 1;
            double pw = (cr ? r.w : 1.0 - r.w) * (ce ? e.w : 1.0 - e.w) * (ci ? ii.w : 1.0 - ii.w) * (cb ? b.w : 1.0 - b.w);
            float4 v = F.at4(r.i + cr, e.i + ce, ii.i + ci, b.i + cb);
            y[0] += pw * v.x; y[1] += pw * v.y; y[2] += pw * v.z;
        }
    }
}

__device__ __forceinline__ double coulomb_C_table64(const DevTable &T, double the, double thi)
{
    Loc64 a = locate64(T.cax[0], thi), b = locate64(T.cax[1], the);
    const int n1 = T.cax[1].n;
    const float *p = T.coul + a.i * n1 + b.i;
    double y = (1.0 - a.w) * ((1.0 - b.w) * __ldg(p) + b.w * __ldg(p + 1)) +
               a.w * ((1.0 - b.w) * __ldg(p + n1) + b.w * __ldg(p + n1 + 1));
    return exp10(y);
}

// shared by the fp64 table path and the analytic kernel: floor, Coulomb, limited update (B3-B6)
__device__ __forceinline__ void update64(const DevTable &T, const DevConst &K, const StepConst &S, double rho, double r,
                                         double lam, const double frac[3], double &the, double &thi, double de_sum[4],
                                         int &limited, int &floored)
{
    if (S.hfloor2 > 0.0 && r > 0.0) {
        double ok = r / (r * sqrt(r) + S.spin);            // Omega_K r
        if ((the + thi) * S.mr < S.hfloor2 * ok * ok) { lam = 0.0; floored = 1; }
    }
    double dcoul = 0.0;                                    // raw Coulomb change of Theta_e over h
    const double D = thi - the;
    if (S.coulomb != 0 && D != 0.0) {
        double C = (S.coulomb == 1) ? coulomb_C_table64(T, the, thi)
                                    : coolphys::coulomb_C(the, thi / K.units.ion_theta_mass_ratio);
        dcoul = S.coul_kh * rho * C * D;
    }
    // energies per (rho mr): ue = the/ge1, ui = thi/gi1 ; work directly in Theta
    double dth_rad = lam * S.h * S.ge1 / (rho * S.mr);     // dE (ge1/(rho mr))
    if (dth_rad > S.f_limit * the) { dth_rad = S.f_limit * the; limited = 1; }
    double mag = fabs(dcoul);
    double cap1 = (D > 0.0) ? S.f_limit * thi * (S.ge1 / S.gi1) : S.f_limit * the;
    double cap2 = fabs(D) * S.eq_frac;
    mag = fmin(mag, fmin(cap1, cap2));
    double dthe = (D > 0.0) ? mag : -mag;
    de_sum[0] += dth_rad;
    de_sum[1] += dth_rad * frac[0]; de_sum[2] += dth_rad * frac[1]; de_sum[3] += dth_rad * frac[2];
    the = the - dth_rad + dthe;
    thi = thi - dthe * (S.gi1 / S.ge1);
}

template <int MODE, class Fetch>
__device__ __forceinline__ void step_cell_f64(const DevTable &T, const DevConst &K, const StepConst &S, const Fetch &F,
                                              double rho, double bsq, double &the, double &thi, double r, double vol, DiagAcc &acc)
{
    if (isnan(rho) || isnan(bsq) || isnan(the) || isnan(thi)) { the = thi = __longlong_as_double(0x7ff8000000000000LL); return; }
    if (!(rho > 0.0)) return;
    const Loc64 lr = locate64(T.ax[CAX_RHO], rho), lb = locate64(T.ax[CAX_BSQ], bsq);
    int limited = 0, floored = 0, clamped = lr.clamped | lb.clamped;
    double de_sum[4] = {0, 0, 0, 0};
    for (int s = 0; s < S.nsub; ++s) {
        const Loc64 le = locate64(T.ax[CAX_THE], the);
        clamped |= le.clamped;
        double lam, frac[3] = {0, 0, 0};
        if constexpr (MODE == 3) {
            lam = exp10(interp3_f64(F, lr, le, lb));
        } else {
            const Loc64 li = locate64(T.ax[CAX_THI], thi);
            clamped |= li.clamped;
            double y[3];
            interp4_f64(F, lr, le, li, lb, y);
            const double qbr = exp10(y[0]), qsy = exp10(y[1]), eta = exp10(y[2]);
            const double qthin = qbr + eta * qsy;                                         // eq 10
            const double cs2 = (S.ae * the + S.ai * thi) / (1.0 + S.be * the + S.bi * thi);   // eq 14
            const double H = S.h_per_cs * sqrt(cs2);                                      // eq 13
            const double th2 = the * the;
            const double tau_abs = qthin * H / (S.bb_k * th2 * th2);                      // eq 12
            const double tau_sca = S.tausca_k * rho * H;
            lam = qthin / (1.0 + tau_abs * (1.7320508075688772 + 1.5 * (tau_abs + tau_sca)));   // eq 11
            frac[0] = qbr / qthin; frac[1] = qsy / qthin; frac[2] = (eta - 1.0) * qsy / qthin;
        }
        update64(T, K, S, rho, r, lam, frac, the, thi, de_sum, limited, floored);
    }
    if (S.want_diag) {
        const double wgt = rho * vol;
#pragma unroll
        for (int k = 0; k < 4; ++k) acc.lum[k] += de_sum[k] * wgt;
        acc.lim += limited; acc.flo += floored; acc.cla += clamped;
    }
}

// analytic variant (COOL_V_ANALYTIC): eqs 1-12 per cell, fp64 regardless of the cell dtype
template <int MODE>
__device__ __noinline__ void step_cell_analytic(const DevTable &T, const DevConst &K, const StepConst &S,
                                                double rho, double bsq, double &the, double &thi, double r, double vol, DiagAcc &acc)
{
    if (isnan(rho) || isnan(bsq) || isnan(the) || isnan(thi)) { the = thi = __longlong_as_double(0x7ff8000000000000LL); return; }
    if (!(rho > 0.0)) return;
    int limited = 0, floored = 0;
    double de_sum[4] = {0, 0, 0, 0};
    const double ne = K.der.ne_per_rho * rho;
    const double B = sqrt(K.der.b2_per_bsq * fmax(bsq, 0.0));
    for (int s = 0; s < S.nsub; ++s) {
        double H = S.hth_cm;
        if (MODE == 4) H = S.h_per_cs * sqrt((S.ae * the + S.ai * thi) / (1.0 + S.be * the + S.bi * thi));
        coolphys::Cooling c = coolphys::cooling_cgs(H, B, ne, the);
        double frac[3] = {c.brems / c.thin, c.synch / c.thin, (c.eta - 1.0) * c.synch / c.thin};
        update64(T, K, S, rho, r, c.total * K.der.rate_conv, frac, the, thi, de_sum, limited, floored);
    }
    if (S.want_diag) {
        const double wgt = rho * vol;
#pragma unroll
        for (int k = 0; k < 4; ++k) acc.lum[k] += de_sum[k] * wgt;
        acc.lim += limited; acc.flo += floored;
    }
}

// ==========================================================================================
// fp32 path.  log2 of every primitive is kept as (integer exponent e, fraction lm = log2 mantissa)
// so that node coordinates and the exponent of the rate are formed without cancelling large
// fp32 numbers; the rate is applied as the dimensionless ratio rrad = Lambda h / u_e.
// ==========================================================================================
struct L2f { float e, lm; };
__device__ __forceinline__ L2f split_log2(float q)
{
    L2f r;
    if (!(q > 0.f)) { r.e = -300.f; r.lm = 0.f; return r; }            // non-positive -> below every table
    const int b = __float_as_int(q);
    r.e = __int_as_float(((unsigned)b >> 23) | 0x4B000000) - 8388735.0f;   // exponent field - 127, no I2F
    r.lm = __log2f(__int_as_float((b & 0x007fffff) | 0x3f800000));         // MUFU.LG2 on [1,2): abs err 2^-22
    return r;
}
struct Loc32 { int i; float w; int clamped; };
__device__ __forceinline__ Loc32 locate32(const AxisCoef &a, const L2f &q)
{
    Loc32 L;
    float t = fmaf(q.e - a.e0, a.invf, fmaf(q.lm, a.invf, a.cf));
    const float tmax = (float)(a.n - 1);
    L.clamped = (t < 0.f) | (t > tmax);
    t = fminf(fmaxf(t, 0.f), tmax);
    // floor via the 2^23 trick (no F2I/I2F): rint(t - 0.5) equals floor(t) except at exact
    // integers, where either neighbour gives the same interpolant
    const float tf = (t - 0.5f) + 12582912.0f;         // 1.5 * 2^23 keeps the sum in [2^23, 2^24)
    int i = __float_as_int(tf) - 0x4B400000;
    float fi = tf - 12582912.0f;
    if (i < 0) { i = 0; fi = 0.f; }
    if (i > a.n - 2) { i = a.n - 2; fi = (float)(a.n - 2); }
    L.i = i; L.w = t - fi;
    return L;
}

// (base, delta) form: y = base + delta with base an exact table value and |delta| small
template <class Fetch>
__device__ __forceinline__ void interp3_f32(const Fetch &F, const Loc32 &r, const Loc32 &e, const Loc32 &b, float &base, float &delta)
{
    if constexpr (Fetch::kHw) {
        base = 0.f;
        delta = F.hw3(r.i + r.w, e.i + e.w, b.i + b.w);
    } else {
        const float c000 = F.at1(r.i, e.i, b.i), c001 = F.at1(r.i, e.i, b.i + 1);
        const float c010 = F.at1(r.i, e.i + 1, b.i), c011 = F.at1(r.i, e.i + 1, b.i + 1);
        const float c100 = F.at1(r.i + 1, e.i, b.i), c101 = F.at1(r.i + 1, e.i, b.i + 1);
        const float c110 = F.at1(r.i + 1, e.i + 1, b.i), c111 = F.at1(r.i + 1, e.i + 1, b.i + 1);
        base = c000;
        const float d010 = c010 - c000, d100 = c100 - c000, d110 = c110 - c000;
        const float a00 = b.w * (c001 - c000);
        const float a01 = fmaf(b.w, c011 - c010, d010);
        const float a10 = fmaf(b.w, c101 - c100, d100);
        const float a11 = fmaf(b.w, c111 - c110, d110);
        const float b0 = fmaf(e.w, a01 - a00, a00), b1 = fmaf(e.w, a11 - a10, a10);
        delta = fmaf(r.w, b1 - b0, b0);
    }
}
template <class Fetch>
__device__ __forceinline__ void interp4_f32(const Fetch &F, const Loc32 &r, const Loc32 &e, const Loc32 &ii, const Loc32 &b,
                                            float base[3], float delta[3])
{
    if constexpr (Fetch::kHw) {
        const float ti = ii.i + ii.w, tb = b.i + b.w;
        const float4 v00 = F.hw4(r.i, e.i, ti, tb), v01 = F.hw4(r.i, e.i + 1, ti, tb);
        const float4 v10 = F.hw4(r.i + 1, e.i, ti, tb), v11 = F.hw4(r.i + 1, e.i + 1, ti, tb);
        const float *p00 = &v00.x, *p01 = &v01.x, *p10 = &v10.x, *p11 = &v11.x;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            base[k] = p00[k];
            const float a0 = e.w * (p01[k] - p00[k]);
            const float a1 = fmaf(e.w, p11[k] - p10[k], p10[k] - p00[k]);
            delta[k] = fmaf(r.w, a1 - a0, a0);
        }
    } else {
        float acc[2][2][3];          // [cr][ce] after reducing (theta_i, bsq), relative to base
        float4 v0 = F.at4(r.i, e.i, ii.i, b.i);
        base[0] = v0.x; base[1] = v0.y; base[2] = v0.z;
#pragma unroll
        for (int cr = 0; cr < 2; ++cr)
#pragma unroll
            for (int ce = 0; ce < 2; ++ce) {
                const float4 q00 = (cr | ce) ? F.at4(r.i + cr, e.i + ce, ii.i, b.i) : v0;
                const float4 q01 = F.at4(r.i + cr, e.i + ce, ii.i, b.i + 1);
                const float4 q10 = F.at4(r.i + cr, e.i + ce, ii.i + 1, b.i);
                const float4 q11 = F.at4(r.i + cr, e.i + ce, ii.i + 1, b.i + 1);
                const float *a = &q00.x, *bb = &q01.x, *c = &q10.x, *d = &q11.x;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    const float x0 = fmaf(b.w, bb[k] - a[k], a[k] - base[k]);
                    const float x1 = fmaf(b.w, d[k] - c[k], c[k] - base[k]);
                    acc[cr][ce][k] = fmaf(ii.w, x1 - x0, x0);
                }
            }
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const float a0 = fmaf(e.w, acc[0][1][k] - acc[0][0][k], acc[0][0][k]);
            const float a1 = fmaf(e.w, acc[1][1][k] - acc[1][0][k], acc[1][0][k]);
            delta[k] = fmaf(r.w, a1 - a0, a0);
        }
    }
}

// exponent (log2) of 10^(base+delta) * h / u_e as big + small (big: exact sum of large terms)
__device__ __forceinline__ float rate_exponent(const StepConst &S, float base, float delta, const L2f &lr, const L2f &le)
{
    const float P = base * S.L10h;
    const float Pl = fmaf(base, S.L10h, -P);
    const float small = fmaf(base, S.L10l, Pl) + fmaf(delta, S.L10h, S.ksm - lr.lm - le.lm);
    const float big = P - (lr.e + le.e);
    return big + small;
}

__device__ __forceinline__ float coulomb_C_table32(const DevTable &T, const L2f &le, const L2f &li)
{
    const Loc32 a = locate32(T.cax[0], li), b = locate32(T.cax[1], le);
    const int n1 = T.cax[1].n;
    const float *p = T.coul + a.i * n1 + b.i;
    const float c00 = __ldg(p), c01 = __ldg(p + 1), c10 = __ldg(p + n1), c11 = __ldg(p + n1 + 1);
    const float y0 = fmaf(b.w, c01 - c00, c00), y1 = fmaf(b.w, c11 - c10, c10);
    return exp2f(3.3219280948873623f * fmaf(a.w, y1 - y0, y0));
}

template <int MODE, class Fetch>
__device__ __forceinline__ void step_cell_f32(const DevTable &T, const DevConst &K, const StepConst &S, const Fetch &F,
                                              float rho, float bsq, float &the, float &thi, float r, float vol, DiagAcc &acc)
{
    if (isnan(rho) || isnan(bsq) || isnan(the) || isnan(thi)) { the = thi = __int_as_float(0x7fc00000); return; }
    if (!(rho > 0.f)) return;
    const L2f l_r = split_log2(rho), l_b = split_log2(bsq);
    const Loc32 lr = locate32(T.ax[CAX_RHO], l_r), lb = locate32(T.ax[CAX_BSQ], l_b);
    int limited = 0, floored = 0, clamped = lr.clamped | lb.clamped;
    float tfloor = 0.f;
    if (S.hfloor2f > 0.f && r > 0.f) {
        const float ok = r / fmaf(r, sqrtf(r), S.spinf);       // Omega_K r
        tfloor = S.hfloor2f * ok * ok;
    }
    float lsum[4] = {0.f, 0.f, 0.f, 0.f};
    for (int s = 0; s < S.nsub; ++s) {
        const L2f l_e = split_log2(the);
        const Loc32 le = locate32(T.ax[CAX_THE], l_e);
        clamped |= le.clamped;
        float rrad;                       // Lambda h / u_e
        float fr0 = 0.f, fr1 = 0.f, fr2 = 0.f;
        L2f l_i;
        if constexpr (MODE == 3) {
            float base, delta;
            interp3_f32(F, lr, le, lb, base, delta);
            rrad = exp2f(rate_exponent(S, base, delta, l_r, l_e));
            if (S.coulomb == 1) l_i = split_log2(thi);
        } else {
            l_i = split_log2(thi);
            const Loc32 li = locate32(T.ax[CAX_THI], l_i);
            clamped |= li.clamped;
            float base[3], delta[3];
            interp4_f32(F, lr, le, li, lb, base, delta);
            const float zbr = fminf(rate_exponent(S, base[0], delta[0], l_r, l_e), 110.f);
            const float zeta = S.L10h * (base[2] + delta[2]);
            const float zsy = rate_exponent(S, base[1], delta[1], l_r, l_e);
            const float rbr = exp2f(zbr);
            const float rsy = exp2f(fminf(zsy + zeta, 110.f));                // eta * Q_syn
            const float rthin = rbr + rsy;                                     // eq 10 (as ratio to u_e/h)
            // eqs 13-14: c_s^2, and log2 of r_B = (4 sigma T^4 / H) h / u_e
            const float num = fmaf(S.aef, the, S.aif * thi), den = fmaf(S.bef, the, fmaf(S.bif, thi, 1.f));
            const L2f l_n = split_log2(num), l_d = split_log2(den);
            const float lcs_I = l_n.e - l_d.e, lcs_F = l_n.lm - l_d.lm;
            const float lB = (S.kB_I + 3.f * l_e.e - l_r.e - 0.5f * lcs_I) + (S.kB_F + 3.f * l_e.lm - l_r.lm - 0.5f * lcs_F);
            const float inv_rB = exp2f(fminf(fmaxf(-lB, -120.f), 120.f));
            const float tau_abs = rthin * inv_rB;                              // eq 12
            const float tau_sca = S.kscaf * rho * exp2f(0.5f * (lcs_I + lcs_F));
            rrad = __fdividef(rthin, fmaf(tau_abs, fmaf(1.5f, tau_abs + tau_sca, 1.7320508f), 1.f));   // eq 11
            if (S.want_diag) {
                const float inv = __fdividef(1.f, rthin);
                const float eta = exp2f(zeta);
                fr0 = rbr * inv; fr1 = __fdividef(rsy, eta) * inv; fr2 = rsy * inv - fr1;
            }
        }
        if (tfloor > 0.f && (the + thi) * S.mrf < tfloor) { rrad = 0.f; floored = 1; }
        if (rrad > S.f_limitf) { rrad = S.f_limitf; limited = 1; }
        // Coulomb
        float dthe = 0.f;
        const float D = thi - the;
        if (S.coulomb != 0 && D != 0.f) {
            float C;
            if (S.coulomb == 1) C = coulomb_C_table32(T, l_e, l_i);
            else C = (float)coolphys::coulomb_C((double)the, (double)thi / K.units.ion_theta_mass_ratio);
            const float raw = fabsf(S.coul_khf * rho * C * D);
            const float cap1 = (D > 0.f) ? S.f_limitf * thi * S.ge1_over_gi1 : S.f_limitf * the;
            const float mag = fminf(raw, fminf(cap1, fabsf(D) * S.eq_fracf));
            dthe = copysignf(mag, D);
        }
        const float drad = rrad * the;
        lsum[0] += drad; lsum[1] = fmaf(drad, fr0, lsum[1]); lsum[2] = fmaf(drad, fr1, lsum[2]); lsum[3] = fmaf(drad, fr2, lsum[3]);
        the = (the - drad) + dthe;
        thi = fmaf(-dthe, S.gi1_over_ge1, thi);
    }
    if (S.want_diag) {
        const float wgt = rho * vol;
#pragma unroll
        for (int k = 0; k < 4; ++k) acc.lum[k] += (double)(lsum[k] * wgt);
        acc.lim += limited; acc.flo += floored; acc.cla += clamped;
    }
}

// ------------------------------------------------------------------------------------------
// Diagnostics reduction: warp shuffle -> block smem -> per-block partials -> the last block to
// finish sums the partials in a fixed order (bit-reproducible for a given grid).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ void reduce_diag(const DiagAcc &acc, const StepConst &S, double *partials, unsigned *ticket, cool_diag *out)
{
    __shared__ double sh[32][8];
    __shared__ unsigned s_last;
    double v[7] = {acc.lum[0], acc.lum[1], acc.lum[2], acc.lum[3], (double)acc.lim, (double)acc.flo, (double)acc.cla};
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int k = 0; k < 7; ++k) {
        v[k] = warp_sum(v[k]);
        if (lane == 0) sh[wid][k] = v[k];
    }
    __syncthreads();
    if (threadIdx.x < 7) {
        double s = 0.0;
        for (int w = 0; w < nw; ++w) s += sh[w][threadIdx.x];
        partials[(size_t)blockIdx.x * 8 + threadIdx.x] = s;
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // fixed-order final pass: thread t sums blocks t, t+B, ...; then a fixed tree over threads
    __shared__ double fin[256];
    for (int k = 0; k < 7; ++k) {
        double s = 0.0;
        if (threadIdx.x < 256)
            for (unsigned b = threadIdx.x; b < gridDim.x; b += 256) s += ((volatile double *)partials)[(size_t)b * 8 + k];
        if (threadIdx.x < 256) fin[threadIdx.x] = s;
        __syncthreads();
        for (int o = 128; o > 0; o >>= 1) {
            if (threadIdx.x < o && threadIdx.x + o < min(256u, blockDim.x)) fin[threadIdx.x] += fin[threadIdx.x + o];
            __syncthreads();
        }
        if (threadIdx.x == 0) {
            double t = fin[0];
            if (k < 4) (&out->lum_total)[k] = t * S.lum_k;
            else (&out->n_limited)[k - 4] = (long long)(t + 0.5);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) *ticket = 0;       // ready for the next launch on this stream
}

// ------------------------------------------------------------------------------------------
// The kernel
// ------------------------------------------------------------------------------------------
template <class Real, int MODE, class Fetch, bool ANALYTIC>
__device__ __forceinline__ void do_cell(const DevTable &T, const DevConst &K, const StepConst &S, const Fetch &F,
                                        Real rho, Real bsq, Real &the, Real &thi, Real r, Real vol, DiagAcc &acc)
{
    if constexpr (ANALYTIC) {
        double te = (double)the, ti = (double)thi;
        step_cell_analytic<MODE>(T, K, S, (double)rho, (double)bsq, te, ti, (double)r, (double)vol, acc);
        the = (Real)te; thi = (Real)ti;
    } else if constexpr (sizeof(Real) == 8) {
        step_cell_f64<MODE>(T, K, S, F, rho, bsq, the, thi, r, vol, acc);
    } else {
        step_cell_f32<MODE>(T, K, S, F, rho, bsq, the, thi, r, vol, acc);
    }
}

struct CellPtrs { const void *rho, *bsq, *the_in, *thi_in, *r, *vol; void *the_out, *thi_out; long long ncell; };

template <class Real, int MODE, class Fetch, bool ANALYTIC, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
cool_step_kernel(const DevTable T, const DevConst K, const StepConst S, const CellPtrs C, double *partials, unsigned *ticket, cool_diag *d_diag)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Fetch F(T, smem_raw);
    using V = typename VecT<Real>::type;
    constexpr int N = VecT<Real>::N;
    DiagAcc acc;
    const long long nvec = S.aligned ? C.ncell / N : 0;
    const long long stride = (long long)gridDim.x * THREADS;
    for (long long v = (long long)blockIdx.x * THREADS + threadIdx.x; v < nvec; v += stride) {
        V rho = ld_stream((const V *)C.rho + v), bsq = ld_stream((const V *)C.bsq + v);
        V the = ld_stream((const V *)C.the_in + v), thi = ld_stream((const V *)C.thi_in + v);
        V rr, vv;
        if (S.has_r) rr = ld_stream((const V *)C.r + v);
        if (S.has_vol) vv = ld_stream((const V *)C.vol + v);
#pragma unroll
        for (int j = 0; j < N; ++j)
            do_cell<Real, MODE, Fetch, ANALYTIC>(T, K, S, F, vget(rho, j), vget(bsq, j), vget(the, j), vget(thi, j),
                                                 S.has_r ? vget(rr, j) : (Real)0, S.has_vol ? vget(vv, j) : (Real)1, acc);
        st_stream((V *)C.the_out + v, the);
        st_stream((V *)C.thi_out + v, thi);
    }
    // scalar tail (and the whole range when the arrays are not 16-byte aligned)
    for (long long c = nvec * N + (long long)blockIdx.x * THREADS + threadIdx.x; c < C.ncell; c += stride) {
        Real the = ((const Real *)C.the_in)[c], thi = ((const Real *)C.thi_in)[c];
        do_cell<Real, MODE, Fetch, ANALYTIC>(T, K, S, F, ((const Real *)C.rho)[c], ((const Real *)C.bsq)[c], the, thi,
                                             S.has_r ? ((const Real *)C.r)[c] : (Real)0, S.has_vol ? ((const Real *)C.vol)[c] : (Real)1, acc);
        ((Real *)C.the_out)[c] = the;
        ((Real *)C.thi_out)[c] = thi;
    }
    if (S.want_diag) reduce_diag(acc, S, partials, ticket, d_diag);
}

// ------------------------------------------------------------------------------------------
// Host side: per-launch constants and dispatch
// ------------------------------------------------------------------------------------------
static void split_if(double x, float &I, float &Fr)
{
    double fl = floor(x);
    I = (float)fl; Fr = (float)(x - fl);
}
static StepConst make_step_const(const cool_table *t, cool_dtype dt, const LaunchArgs &a)
{
    const DevConst &K = t->cst;
    StepConst S{};
    S.h = a.dt / a.nsub; S.inv_dt = 1.0 / a.dt; S.f_limit = a.f_limit;
    S.mr = K.mr; S.ge1 = K.ge1; S.gi1 = K.gi1; S.eq_frac = K.ge1 / (K.ge1 + K.gi1);
    S.coul_kh = K.coul_k * S.h * K.ge1;
    S.bb_k = K.bb_k; S.tausca_k = K.tausca_k; S.h_per_cs = K.der.h_per_cs; S.hth_cm = K.units.hth_cm;
    S.ae = K.units.gamma_e * K.mr; S.ai = K.units.gamma_i * K.mr;
    S.be = K.mr * K.units.gamma_e / K.ge1; S.bi = K.mr * K.units.gamma_i / K.gi1;
    S.hfloor2 = (a.h_floor > 0.0 && a.r) ? 0.5 * coolphys::kPI * a.h_floor * a.h_floor : 0.0;
    S.spin = K.units.spin;
    S.lum_k = K.mr / (K.ge1 * a.dt);
    const double L10 = 3.321928094887362;
    S.L10h = (float)L10; S.L10l = (float)(L10 - (double)S.L10h);
    S.ksm = (float)(log2(S.h) - K.log2_ue_k);
    S.f_limitf = (float)a.f_limit; S.mrf = (float)K.mr; S.eq_fracf = (float)S.eq_frac;
    S.ge1_over_gi1 = (float)(K.ge1 / K.gi1); S.gi1_over_ge1 = (float)(K.gi1 / K.ge1);
    S.coul_khf = (float)S.coul_kh;
    S.aef = (float)S.ae; S.aif = (float)S.ai; S.bef = (float)S.be; S.bif = (float)S.bi;
    split_if(log2(K.bb_k * S.h * K.ge1 / (K.der.h_per_cs * K.mr)), S.kB_I, S.kB_F);
    split_if(log2(K.bb_k * S.h * K.ge1 / (K.units.hth_cm * K.mr)), S.kB3_I, S.kB3_F);
    S.kscaf = (float)(K.tausca_k * K.der.h_per_cs);
    S.hfloor2f = (float)S.hfloor2; S.spinf = (float)S.spin;
    S.nsub = a.nsub; S.coulomb = a.coulomb; S.want_diag = a.want_diag;
    S.has_r = a.r != nullptr; S.has_vol = a.vol != nullptr;
    const size_t al = dt == COOL_F32 ? 16 : 16;
    auto ok = [&](const void *p) { return p == nullptr || ((size_t)p % al) == 0; };
    S.aligned = ok(a.rho) && ok(a.bsq) && ok(a.the_in) && ok(a.thi_in) && ok(a.the_out) && ok(a.thi_out) && ok(a.r) && ok(a.vol);
    return S;
}

template <class Real, int MODE, class Fetch, bool ANALYTIC, int THREADS, int MINB>
static cudaError_t launch_one(const cool_table *t, const StepConst &S, const LaunchArgs &a, size_t smem, cudaStream_t st)
{
    auto kern = cool_step_kernel<Real, MODE, Fetch, ANALYTIC, THREADS, MINB>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    // persistent grid: exactly the resident blocks (a multiple of the SM count), grid-stride inside
    int occ = 0;
    cudaError_t eo = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, THREADS, smem);
    if (eo != cudaSuccess) return eo;
    if (occ < 1) occ = 1;
    constexpr int N = VecT<Real>::N;
    long long need = (a.ncell / N + THREADS - 1) / THREADS;
    if (need < 1) need = 1;
    const long long cap = (long long)t->sm_count * occ;
    const int grid = (int)(need < cap ? need : cap);
    CellPtrs C{a.rho, a.bsq, a.the_in, a.thi_in, a.r, a.vol, a.the_out, a.thi_out, a.ncell};
    kern<<<grid, THREADS, smem, st>>>(t->dev, t->cst, S, C, a.partials, a.ticket, a.d_diag);
    return cudaGetLastError();
}

static constexpr int kSmemThreads = 1024;

bool variant_supported(const cool_table *t, cool_variant v, cool_dtype, std::string *why)
{
    if (v == COOL_V_ANALYTIC) return true;
    if (t->dev.mode == 0) { if (why) *why = "table has no data (nproc = 0): only COOL_V_ANALYTIC applies"; return false; }
    if (v == COOL_V_SMEM && (size_t)t->dev.table_bytes + 1024 > (size_t)t->max_smem_optin) {
        if (why) *why = "table does not fit in shared memory"; return false;
    }
    return true;
}

cool_status launch_step(const cool_table *t, cool_variant v, cool_dtype dt, const LaunchArgs &a, cudaStream_t st, int *nlaunch)
{
    const StepConst S = make_step_const(t, dt, a);
    const int mode = t->dev.mode == 0 ? (t->desc.ndim == 4 ? 4 : 3) : t->dev.mode;
    cudaError_t e = cudaSuccess;
#define COOL_LAUNCH(REAL, MODE, FETCH, AN, TH, MB, SMEM) e = launch_one<REAL, MODE, FETCH, AN, TH, MB>(t, S, a, SMEM, st)
#define COOL_BY_MODE(REAL, FETCH, AN, TH, MB, SMEM) do { if (mode == 3) COOL_LAUNCH(REAL, 3, FETCH, AN, TH, MB, SMEM); else COOL_LAUNCH(REAL, 4, FETCH, AN, TH, MB, SMEM); } while (0)
#define COOL_BY_DTYPE(FETCH, AN, TH, MB, SMEM) do { if (dt == COOL_F32) COOL_BY_MODE(float, FETCH, AN, TH, MB, SMEM); else COOL_BY_MODE(double, FETCH, AN, TH, MB, SMEM); } while (0)
    switch (v) {
        case COOL_V_GLOBAL: COOL_BY_DTYPE(FetchGlobal, false, 256, 2, 0); break;
        case COOL_V_TEX_POINT: COOL_BY_DTYPE(FetchTexPoint, false, 256, 2, 0); break;
        case COOL_V_TEX_HWFILTER: COOL_BY_DTYPE(FetchTexHw, false, 256, 2, 0); break;
        case COOL_V_SMEM: COOL_BY_DTYPE(FetchSmem, false, kSmemThreads, 1, (size_t)t->dev.table_bytes); break;
        case COOL_V_ANALYTIC: COOL_BY_DTYPE(FetchNone, true, 256, 1, 0); break;
        default: set_error("internal: unresolved variant %d", (int)v); return COOL_EINVAL;
    }
    if (e != cudaSuccess) { set_error("kernel launch failed: %s", cudaGetErrorString(e)); return COOL_ECUDA; }
    if (nlaunch) *nlaunch += 1;
    return COOL_OK;
}

}  // namespace cool
