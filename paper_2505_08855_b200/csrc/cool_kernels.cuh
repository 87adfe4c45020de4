// cool_kernels.cuh — hand-written sm_100a kernels of the per-cell cooling step (include/cool.h):
// the fp64 table variants and the analytic variant (either cell dtype), plus what the fp32 kernels
// of cool_f32.cuh share with them (streaming I/O, diagnostics reduction).
//
// One kernel template, instantiated per (cell dtype) x (table shape) x (lookup variant) x flags:
//   * cells stream as SoA with 128-bit L1-bypassing loads/stores, 16 B per thread per array;
//   * the table is read through one of four lookup policies (global/L2, shared memory, point
//     texture, hardware-filtered texture) or not at all (analytic);
//   * the luminosity diagnostic is reduced warp -> block -> fixed-order last-block pass, so it is
//     bit-reproducible for a given launch shape.
// The fp64 path mirrors the definition step by step (tolerance 1e-12); it is the correctness
// path of configs[0], not the throughput path.
#pragma once
#include "cool_internal.h"

namespace cool {

// ------------------------------------------------------------------------------------------
// Per-launch constants (host fp64 -> rounded copies for the fp32 path).
// ------------------------------------------------------------------------------------------
struct StepConst {
    // fp64 path
    double h, f_limit, mr, ge1, gi1, eq_frac, coul_kh, bb_k, tausca_k, h_per_cs, hth_cm;
    double ae, ai, be, bi;         // c_s^2 = (ae Th_e + ai Th_i)/(1 + be Th_e + bi Th_i)      (eq 14)
    double hfloor2, spin;          // floor: (pi/2) h_floor^2 (Omega_K r)^2                     (eq 19)
    double lum_k;                  // lum = sum(dTheta_rad rho vol) * lum_k,  lum_k = mr/(ge1 dt)
    int nsub, coulomb, has_r, has_vol, aligned;
    int cgs; double omk_ref_inv;   // the paper's table: H_th from the cell's radius; omk_ref_inv = r_ref^1.5 + a
    // radial profile (eq 25): shell = (cell_offset + cell)/shell_cells; sums go to replica (block index & shell_rmask) of lum_shell
    // (this launch's workspace, local shell index); shell_reduce_kernel then adds the replicas into the caller's array
    double *lum_shell; long long shell_cells, cell_offset, shell0; unsigned shell_nloc4, shell_rmask;
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
    // the 8 corners of a MODE-3 cell with one pointer computation; c[cr*4 + ce*2 + cb]
    template <class L> __device__ __forceinline__ void corners3(const L &r, const L &e, const L &b, float (&c)[8]) const
    {
        const float *p = p1 + (r.i * sr + e.i * se + b.i), *q = p + se, *u = p + sr, *v = u + se;
        c[0] = __ldg(p); c[1] = __ldg(p + 1); c[2] = __ldg(q); c[3] = __ldg(q + 1);
        c[4] = __ldg(u); c[5] = __ldg(u + 1); c[6] = __ldg(v); c[7] = __ldg(v + 1);
    }
    // the (rho, bsq) quad of a MODE-4 table at (ie+ce, ii+ci); q[cr*2 + cb]
    template <class L> __device__ __forceinline__ void quad4(const L &r, const L &e, const L &ii, const L &b, int ce, int ci, float4 (&q)[4]) const
    {
        const float4 *p = p4 + (r.i * sr + (e.i + ce) * se + (ii.i + ci) * si + b.i), *u = p + sr;
        q[0] = __ldg(p); q[1] = __ldg(p + 1); q[2] = __ldg(u); q[3] = __ldg(u + 1);
    }
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
    }
    __device__ __forceinline__ float at1(int ir, int ie, int ib) const { return p1[ir * sr + ie * se + ib]; }
    __device__ __forceinline__ float4 at4(int ir, int ie, int ii, int ib) const { return p4[ir * sr + ie * se + ii * si + ib]; }
    template <class L> __device__ __forceinline__ void corners3(const L &r, const L &e, const L &b, float (&c)[8]) const
    {
        const float *p = p1 + (r.i * sr + e.i * se + b.i), *q = p + se, *u = p + sr, *v = u + se;
        c[0] = p[0]; c[1] = p[1]; c[2] = q[0]; c[3] = q[1]; c[4] = u[0]; c[5] = u[1]; c[6] = v[0]; c[7] = v[1];
    }
    template <class L> __device__ __forceinline__ void quad4(const L &r, const L &e, const L &ii, const L &b, int ce, int ci, float4 (&q)[4]) const
    {
        const float4 *p = p4 + (r.i * sr + (e.i + ce) * se + (ii.i + ci) * si + b.i), *u = p + sr;
        q[0] = p[0]; q[1] = p[1]; q[2] = u[0]; q[3] = u[1];
    }
};
struct FetchTexPoint {
    static constexpr bool kHw = false, kSmem = false;
    cudaTextureObject_t tex; int ne; float nef;
    __device__ FetchTexPoint(const DevTable &T, void *) : tex(T.tex_pt), ne(T.ax[CAX_THE].n), nef((float)T.ax[CAX_THE].n) {}
    __device__ __forceinline__ float at1(int ir, int ie, int ib) const { return tex3D<float>(tex, ib + 0.5f, ie + 0.5f, ir + 0.5f); }
    __device__ __forceinline__ float4 at4(int ir, int ie, int ii, int ib) const { return tex3D<float4>(tex, ib + 0.5f, ii + 0.5f, (ir * ne + ie) + 0.5f); }
    // float node indices (L::fi) avoid int->float conversions; texel centres are at +0.5
    template <class L> __device__ __forceinline__ void corners3(const L &r, const L &e, const L &b, float (&c)[8]) const
    {
        const float x = b.fi + 0.5f, y = e.fi + 0.5f, z = r.fi + 0.5f;
        c[0] = tex3D<float>(tex, x, y, z); c[1] = tex3D<float>(tex, x + 1.f, y, z);
        c[2] = tex3D<float>(tex, x, y + 1.f, z); c[3] = tex3D<float>(tex, x + 1.f, y + 1.f, z);
        c[4] = tex3D<float>(tex, x, y, z + 1.f); c[5] = tex3D<float>(tex, x + 1.f, y, z + 1.f);
        c[6] = tex3D<float>(tex, x, y + 1.f, z + 1.f); c[7] = tex3D<float>(tex, x + 1.f, y + 1.f, z + 1.f);
    }
    template <class L> __device__ __forceinline__ void quad4(const L &r, const L &e, const L &ii, const L &b, int ce, int ci, float4 (&q)[4]) const
    {
        const float x = b.fi + 0.5f, y = ii.fi + (float)ci + 0.5f, z = fmaf(r.fi, nef, e.fi + (float)ce + 0.5f);
        q[0] = tex3D<float4>(tex, x, y, z); q[1] = tex3D<float4>(tex, x + 1.f, y, z);
        q[2] = tex3D<float4>(tex, x, y, z + nef); q[3] = tex3D<float4>(tex, x + 1.f, y, z + nef);
    }
};
struct FetchTexHw {
    static constexpr bool kHw = true, kSmem = false;
    cudaTextureObject_t tex; int ne; float nef;
    __device__ FetchTexHw(const DevTable &T, void *) : tex(T.tex_lin), ne(T.ax[CAX_THE].n), nef((float)T.ax[CAX_THE].n) {}
    // MODE 3: one trilinear fetch.  MODE 4: hardware bilinear on (bsq, theta_i) at a fixed
    // (rho, theta_e) slice — the paper's scheme (L155-L159): the flattened dimension is manual.
    __device__ __forceinline__ float hw3(float tr, float te, float tb) const { return tex3D<float>(tex, tb + 0.5f, te + 0.5f, tr + 0.5f); }
    __device__ __forceinline__ float4 hw4(int ir, int ie, float ti, float tb) const { return tex3D<float4>(tex, tb + 0.5f, ti + 0.5f, (ir * ne + ie) + 0.5f); }
    __device__ __forceinline__ float4 hw4(float fr, float fe, float ti, float tb) const { return tex3D<float4>(tex, tb + 0.5f, ti + 0.5f, fmaf(fr, nef, fe) + 0.5f); }
    __device__ __forceinline__ float at1(int, int, int) const { return 0.f; }
    __device__ __forceinline__ float4 at4(int, int, int, int) const { return make_float4(0, 0, 0, 0); }
    template <class L> __device__ __forceinline__ void corners3(const L &, const L &, const L &, float (&)[8]) const {}
    template <class L> __device__ __forceinline__ void quad4(const L &, const L &, const L &, const L &, int, int, float4 (&)[4]) const {}
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
// one cell's luminosity terms into its radial shell (fp64 / analytic / implicit kernels: one atomic per term)
__device__ __forceinline__ void shell_add(const StepConst &S, long long cell, const double de_sum[4], double wgt, bool split)
{
    if (!S.lum_shell) return;
    double *p = S.lum_shell + (size_t)(blockIdx.x & S.shell_rmask) * S.shell_nloc4 + 4 * ((S.cell_offset + cell) / S.shell_cells - S.shell0);
    atomicAdd(p, de_sum[0] * wgt * S.lum_k);
    if (split) { atomicAdd(p + 1, de_sum[1] * wgt * S.lum_k); atomicAdd(p + 2, de_sum[2] * wgt * S.lum_k); atomicAdd(p + 3, de_sum[3] * wgt * S.lum_k); }
}

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

// shared by the fp64 table path, the analytic kernel and the paper's-table kernel: floor, limited update (B3-B6);
// dcoul = raw Coulomb change of Theta_e over h
__device__ __forceinline__ void update64_core(const StepConst &S, double rho, double r, double lam, const double frac[3], double &the, double &thi,
                                              double de_sum[4], int &limited, int &floored, double dcoul)
{
    if (S.hfloor2 > 0.0 && r > 0.0) {
        double ok = r / (r * sqrt(r) + S.spin);            // Omega_K r
        if ((the + thi) * S.mr < S.hfloor2 * ok * ok) { lam = 0.0; floored = 1; }
    }
    const double D = thi - the;
    // energies per (rho mr): u_e = the/ge1, u_i = thi/gi1; work directly in Theta
    double dth_rad = lam * S.h * S.ge1 / (rho * S.mr);
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
__device__ __forceinline__ void update64(const DevTable &T, const DevConst &K, const StepConst &S, double rho, double r,
                                         double lam, const double frac[3], double &the, double &thi, double de_sum[4],
                                         int &limited, int &floored)
{
    double dcoul = 0.0;
    const double D = thi - the;
    if (S.coulomb != 0 && D != 0.0) {
        double C = (S.coulomb == 1) ? coulomb_C_table64(T, the, thi)
                                    : coolphys::coulomb_C(the, thi / K.units.ion_theta_mass_ratio);
        dcoul = S.coul_kh * rho * C * D;
    }
    update64_core(S, rho, r, lam, frac, the, thi, de_sum, limited, floored, dcoul);
}
// Coulomb term given as Q_cc/(Theta_i - Theta_e) in code units (the paper's Q_cc(n_e, T_i, T_e) table, cool_cgs.cu):
// dTheta_e = Q_cc h (gamma_e - 1)/(rho m_e/m_p)
__device__ __forceinline__ void update64_q(const StepConst &S, double rho, double r, double lam, const double frac[3], double &the, double &thi,
                                           double de_sum[4], int &limited, int &floored, double qcc_per_D)
{
    const double D = thi - the;
    update64_core(S, rho, r, lam, frac, the, thi, de_sum, limited, floored, D != 0.0 ? qcc_per_D * D * S.h * S.ge1 / (rho * S.mr) : 0.0);
}

template <int MODE, class Fetch, bool DIAG>
__device__ __forceinline__ void step_cell_f64(const DevTable &T, const DevConst &K, const StepConst &S, const Fetch &F,
                                              double rho, double bsq, double &the, double &thi, double r, double vol, DiagAcc &acc, long long cell,
                                              int *cell_flags = nullptr)
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
    if constexpr (DIAG) {
        const double wgt = rho * vol;
#pragma unroll
        for (int k = 0; k < 4; ++k) acc.lum[k] += de_sum[k] * wgt;
        acc.lim += limited; acc.flo += floored; acc.cla += clamped;
        shell_add(S, cell, de_sum, wgt, MODE == 4);
        if (cell_flags) *cell_flags = limited | (floored << 1) | (clamped << 2);
    }
}

// analytic variant (COOL_V_ANALYTIC): eqs 1-12 per cell, fp64 regardless of the cell dtype
template <int MODE, bool DIAG>
__device__ __noinline__ void step_cell_analytic(const DevTable &T, const DevConst &K, const StepConst &S,
                                                double rho, double bsq, double &the, double &thi, double r, double vol, DiagAcc &acc, long long cell,
                                                int *cell_flags)
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
        if (MODE == 4 && S.cgs && r > 0.0) H *= (r * sqrt(r) + S.spin) / S.omk_ref_inv;      // the paper's table: H_th at the cell's own radius (eq 13)
        coolphys::Cooling c = coolphys::cooling_cgs(H, B, ne, the);
        double frac[3] = {c.brems / c.thin, c.synch / c.thin, (c.eta - 1.0) * c.synch / c.thin};
        update64(T, K, S, rho, r, c.total * K.der.rate_conv, frac, the, thi, de_sum, limited, floored);
    }
    if constexpr (DIAG) {
        const double wgt = rho * vol;
#pragma unroll
        for (int k = 0; k < 4; ++k) acc.lum[k] += de_sum[k] * wgt;
        acc.lim += limited; acc.flo += floored;
        shell_add(S, cell, de_sum, wgt, true);
        if (cell_flags) *cell_flags = limited | (floored << 1);
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
// Takes the sums BY VALUE: passing the accumulator by reference to this non-inlined function would pin it in local
// memory for the whole kernel (one st.local per accumulation).
static __device__ __noinline__ void reduce_diag_vals(double l0, double l1, double l2, double l3, int lim, int flo, int cla,
                                                     double lum_k, double *partials, unsigned *ticket, cool_diag *out)
{
    __shared__ double sh[32][8];
    __shared__ unsigned s_last;
    __shared__ double fin[256];
    double v[7] = {l0, l1, l2, l3, (double)lim, (double)flo, (double)cla};
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
    // fixed-order final pass: thread t sums blocks t, t+256, ...; then a fixed tree over threads
    for (int k = 0; k < 7; ++k) {
        double s = 0.0;
        if (threadIdx.x < 256)
            for (unsigned b = threadIdx.x; b < gridDim.x; b += 256) s += ((volatile double *)partials)[(size_t)b * 8 + k];
        if (threadIdx.x < 256) fin[threadIdx.x] = s;
        __syncthreads();
        for (int o = 128; o > 0; o >>= 1) {
            if (threadIdx.x < o) fin[threadIdx.x] += fin[threadIdx.x + o];
            __syncthreads();
        }
        if (threadIdx.x == 0) {
            double t = fin[0];
            if (k < 4) (&out->lum_total)[k] = t * lum_k;
            else (&out->n_limited)[k - 4] = (long long)(t + 0.5);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) *ticket = 0;       // ready for the next launch on this stream
}
__device__ __forceinline__ void reduce_diag(const DiagAcc &acc, double lum_k, double *partials, unsigned *ticket, cool_diag *out)
{
    reduce_diag_vals(acc.lum[0], acc.lum[1], acc.lum[2], acc.lum[3], acc.lim, acc.flo, acc.cla, lum_k, partials, ticket, out);
}
// ------------------------------------------------------------------------------------------
// The kernel
// ------------------------------------------------------------------------------------------
struct CellPtrs { const void *rho, *bsq, *the_in, *thi_in, *r, *vol; void *the_out, *thi_out; long long ncell; unsigned char *flags; };

// NV cells of one thread through the right path
template <class Real, int MODE, class Fetch, bool ANALYTIC, bool DIAG, int CM, int NV>
__device__ __forceinline__ void do_cells(const DevTable &T, const DevConst &K, const StepConst &S, const Fetch &F, const float *coul,
                                         const Real *rho, const Real *bsq, Real *the, Real *thi, const Real *r, const Real *vol, DiagAcc &acc, long long cell0,
                                         unsigned char *flags)
{
    if constexpr (ANALYTIC) {
#pragma unroll 1
        for (int j = 0; j < NV; ++j) {
            double te = (double)the[j], ti = (double)thi[j];
            int fl = 0;
            step_cell_analytic<MODE, DIAG>(T, K, S, (double)rho[j], (double)bsq[j], te, ti, (double)r[j], (double)vol[j], acc, cell0 + j, &fl);
            the[j] = (Real)te; thi[j] = (Real)ti;
            if (DIAG && flags) flags[cell0 + j] = (unsigned char)fl;
        }
    } else {
        static_assert(sizeof(Real) == 8, "fp32 table variants live in cool_f32.cuh");
#pragma unroll
        for (int j = 0; j < NV; ++j) {
            int fl = 0;
            step_cell_f64<MODE, Fetch, DIAG>(T, K, S, F, rho[j], bsq[j], the[j], thi[j], r[j], vol[j], acc, cell0 + j, &fl);
            if (DIAG && flags) flags[cell0 + j] = (unsigned char)fl;
        }
    }
}

constexpr int kCoulSmemMax = 16384;      // Coulomb tables up to 64^2 floats are staged in shared memory

template <class Real, int MODE, class Fetch, bool ANALYTIC, bool DIAG, int CM, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
cool_step_kernel(const DevTable T, const DevConst K, const StepConst S, const CellPtrs C, double *partials, unsigned *ticket, cool_diag *d_diag)
{
    // dynamic shared memory: [table image (SMEM variant)] [Coulomb coefficient table (fp32 path, if small)]
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Fetch F(T, smem_raw);
    const float *coul = T.coul;
    if (Fetch::kSmem) __syncthreads();
    using V = typename VecT<Real>::type;
    constexpr int N = VecT<Real>::N;
    DiagAcc acc;
    const long long nvec = S.aligned ? C.ncell / N : 0;
    const long long stride = (long long)gridDim.x * THREADS;
    for (long long v = (long long)blockIdx.x * THREADS + threadIdx.x; v < nvec; v += stride) {
        V rho = ld_stream((const V *)C.rho + v), bsq = ld_stream((const V *)C.bsq + v);
        V the = ld_stream((const V *)C.the_in + v), thi = ld_stream((const V *)C.thi_in + v);
        V rr, vv;
#pragma unroll
        for (int j = 0; j < N; ++j) { vget(rr, j) = (Real)0; vget(vv, j) = (Real)1; }
        if (S.has_r) rr = ld_stream((const V *)C.r + v);
        if (S.has_vol) vv = ld_stream((const V *)C.vol + v);
        do_cells<Real, MODE, Fetch, ANALYTIC, DIAG, CM, N>(T, K, S, F, coul, &rho.x, &bsq.x, &the.x, &thi.x, &rr.x, &vv.x, acc, v * N, C.flags);
        st_stream((V *)C.the_out + v, the);
        st_stream((V *)C.thi_out + v, thi);
    }
    // scalar tail (and the whole range when the arrays are not 16-byte aligned)
    for (long long c = nvec * N + (long long)blockIdx.x * THREADS + threadIdx.x; c < C.ncell; c += stride) {
        Real the = ((const Real *)C.the_in)[c], thi = ((const Real *)C.thi_in)[c];
        const Real rho = ((const Real *)C.rho)[c], bsq = ((const Real *)C.bsq)[c];
        const Real rr = S.has_r ? ((const Real *)C.r)[c] : (Real)0, vv = S.has_vol ? ((const Real *)C.vol)[c] : (Real)1;
        do_cells<Real, MODE, Fetch, ANALYTIC, DIAG, CM, 1>(T, K, S, F, coul, &rho, &bsq, &the, &thi, &rr, &vv, acc, c, C.flags);
        ((Real *)C.the_out)[c] = the;
        ((Real *)C.thi_out)[c] = thi;
    }
    if constexpr (DIAG) reduce_diag(acc, S.lum_k, partials, ticket, d_diag);
}

// ------------------------------------------------------------------------------------------
// Host-side launch of one instantiation (persistent grid = resident blocks, grid-stride inside)
// ------------------------------------------------------------------------------------------
struct LaunchCtx { const cool_table *t; const StepConst *S; const LaunchArgs *a; cudaStream_t st; };

template <class Real, int MODE, class Fetch, bool ANALYTIC, bool DIAG, int CM, int THREADS, int MINB>
static cudaError_t launch_one(const LaunchCtx &L, size_t smem)
{
    auto kern = cool_step_kernel<Real, MODE, Fetch, ANALYTIC, DIAG, CM, THREADS, MINB>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    // asked per call (a host-side computation of a few microseconds): a cached value would be shared by threads and devices
    int occ_cache = 0;
    cudaError_t eo = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_cache, kern, THREADS, smem);
    if (eo != cudaSuccess) return eo;
    if (occ_cache < 1) occ_cache = 1;
    const LaunchArgs &a = *L.a;
    constexpr int N = VecT<Real>::N;
    long long need = (a.ncell / N + THREADS - 1) / THREADS;
    if (need < 1) need = 1;
    const long long cap = (long long)L.t->sm_count * occ_cache;
    const int grid = (int)(need < cap ? need : cap);
    CellPtrs C{a.rho, a.bsq, a.the_in, a.thi_in, a.r, a.vol, a.the_out, a.thi_out, a.ncell, a.flags};
    kern<<<grid, THREADS, smem, L.st>>>(L.t->dev, L.t->cst, *L.S, C, a.partials, a.ticket, a.d_diag);
    return cudaGetLastError();
}

// one function per translation unit of instantiations (cool_inst_*.cu)
cudaError_t launch_f64(const LaunchCtx &L, int mode, cool_variant v, bool diag);
cudaError_t launch_analytic(const LaunchCtx &L, int mode, cool_dtype dt, bool diag);
cudaError_t launch_cgs(const LaunchCtx &L, cool_variant v, cool_dtype dt, bool diag);      // the paper's table (cool_cgs.cu)


constexpr int kSmemThreads = 512;

// dispatch over the four table variants for fixed <Real, MODE, DIAG, CM>
template <class Real, int MODE, bool DIAG, int CM>
static cudaError_t launch_by_variant(const LaunchCtx &L, cool_variant v)
{
    switch (v) {
        case COOL_V_GLOBAL: return launch_one<Real, MODE, FetchGlobal, false, DIAG, CM, 256, 2>(L, 0);
        case COOL_V_TEX_POINT: return launch_one<Real, MODE, FetchTexPoint, false, DIAG, CM, 256, 2>(L, 0);
        case COOL_V_TEX_HWFILTER: return launch_one<Real, MODE, FetchTexHw, false, DIAG, CM, 256, 2>(L, 0);
        case COOL_V_SMEM: return launch_one<Real, MODE, FetchSmem, false, DIAG, CM, kSmemThreads, 1>(L, (size_t)L.t->dev.table_bytes);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace cool
