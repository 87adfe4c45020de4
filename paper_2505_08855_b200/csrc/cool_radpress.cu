// Radiation-pressure temperature correction (eq 29; reading C-20): per cell, where
// tau_sca = n_e sigma_T H > tau_crit, Theta_e is replaced by the root of  a T^4 + N k_B (T - T_e) = 0.
//
// With y = T/T_e and beta = a T_e^3/(N k_B) the equation is  beta y^4 + y - 1 = 0,  0 < y <= 1.  Newton's step for it,
//     y <- (3 beta y^4 + 1)/(4 beta y^3 + 1),
// has only positive terms (no cancellation at either end of beta's 40 decades) and converges quadratically from the
// seed (1 + beta)^(-1/4), which is exact in both limits: 4 steps reach fp32 rounding, 6 steps fp64 rounding, for every
// beta (a fixed count keeps the warp converged).  The kernel is a pure stream: 12 B read + 4 B written per fp32 cell.
#include <cuda_runtime.h>
#include <cmath>
#include "cool_internal.h"

namespace {

constexpr int kRpThreads = 256;

struct RpConst {
    double c_tau;        // tau_sca = c_tau rho hscale : (rho_scale/m_p) sigma_T r_g
    double c_beta;       // beta = c_beta Theta^3/rho  : a (m_e c^2/k_B)^3 m_p/(k_B rho_scale)
    double tau_crit;
};

__device__ __forceinline__ float rp_cell(float rho, float the, float hs, float c_tau, float c_beta, float tau_crit, int &cnt)
{
    const bool thick = rho > 0.f && the > 0.f && rho * hs * c_tau > tau_crit;      // false for NaN: the cell passes through
    const float beta = fminf(__fdividef(c_beta * the * the * the, rho), 1e38f);
    float y = rsqrtf(sqrtf(1.f + beta));
#pragma unroll
    for (int it = 0; it < 4; ++it) {
        const float by3 = beta * y * y * y;
        y = __fdividef(fmaf(3.f * by3, y, 1.f), fmaf(4.f, by3, 1.f));
    }
    cnt += thick;
    return thick ? the * y : the;
}

__device__ __forceinline__ double rp_cell(double rho, double the, double hs, double c_tau, double c_beta, double tau_crit, int &cnt)
{
    const bool thick = rho > 0.0 && the > 0.0 && rho * hs * c_tau > tau_crit;
    const double beta = fmin(c_beta * the * the * the / rho, 1e300);
    double y = 1.0 / sqrt(sqrt(1.0 + beta));
#pragma unroll
    for (int it = 0; it < 6; ++it) {
        const double by3 = beta * y * y * y;
        y = fma(3.0 * by3, y, 1.0) / fma(4.0, by3, 1.0);
    }
    cnt += thick;
    return thick ? the * y : the;
}

template <typename Real> struct Vec;
template <> struct Vec<float> { using type = float4; static constexpr int n = 4; };
template <> struct Vec<double> { using type = double2; static constexpr int n = 2; };

template <typename Real, typename V> __device__ __forceinline__ V rp_vec(V r, V t, V h, Real ct, Real cb, Real tc, int &cnt)
{
    V o;
    o.x = rp_cell(r.x, t.x, h.x, ct, cb, tc, cnt);
    o.y = rp_cell(r.y, t.y, h.y, ct, cb, tc, cnt);
    if constexpr (sizeof(V) == 4 * sizeof(Real)) {
        o.z = rp_cell(r.z, t.z, h.z, ct, cb, tc, cnt);
        o.w = rp_cell(r.w, t.w, h.w, ct, cb, tc, cnt);
    }
    return o;
}

// VEC: all four arrays 16-byte aligned -> 128-bit streaming loads/stores, two vectors per thread in flight.
template <typename Real, bool VEC, bool COUNT>
__global__ void __launch_bounds__(kRpThreads)
cool_radpress_kernel(const Real *__restrict__ rho, const Real *the, const Real *__restrict__ hs,
                     Real *out, long long ncell, RpConst K, unsigned long long *__restrict__ ncorrected)
{
    const Real ct = (Real)K.c_tau, cb = (Real)K.c_beta, tc = (Real)K.tau_crit;
    int cnt = 0;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long nth = (long long)gridDim.x * blockDim.x;
    long long done = 0;
    if constexpr (VEC) {
        using V = typename Vec<Real>::type;
        constexpr int W = Vec<Real>::n;
        const long long nvec = ncell / W;
        const V *r4 = reinterpret_cast<const V *>(rho), *t4 = reinterpret_cast<const V *>(the), *h4 = reinterpret_cast<const V *>(hs);
        V *o4 = reinterpret_cast<V *>(out);
        long long v = tid;
        for (; v + nth < nvec; v += 2 * nth) {
            const V ra = __ldcs(r4 + v), ta = __ldcs(t4 + v), ha = __ldcs(h4 + v);
            const V rb = __ldcs(r4 + v + nth), tb = __ldcs(t4 + v + nth), hb = __ldcs(h4 + v + nth);
            __stcs(o4 + v, rp_vec<Real, V>(ra, ta, ha, ct, cb, tc, cnt));
            __stcs(o4 + v + nth, rp_vec<Real, V>(rb, tb, hb, ct, cb, tc, cnt));
        }
        if (v < nvec)
            __stcs(o4 + v, rp_vec<Real, V>(__ldcs(r4 + v), __ldcs(t4 + v), __ldcs(h4 + v), ct, cb, tc, cnt));
        done = nvec * W;
    }
    for (long long k = done + tid; k < ncell; k += nth)          // ragged tail, or everything when unaligned
        out[k] = rp_cell(rho[k], the[k], hs[k], ct, cb, tc, cnt);
    if constexpr (COUNT) {
        __shared__ int s_cnt;
        if (threadIdx.x == 0) s_cnt = 0;
        __syncthreads();
        const int w = __reduce_add_sync(0xffffffffu, cnt);
        if ((threadIdx.x & 31) == 0 && w) atomicAdd(&s_cnt, w);
        __syncthreads();
        if (threadIdx.x == 0 && s_cnt) atomicAdd(ncorrected, (unsigned long long)s_cnt);
    }
}

template <typename Real>
cudaError_t rp_launch(const void *rho, const void *the, const void *hs, void *out, long long ncell, const RpConst &K,
                      long long *d_cnt, int nsm, cudaStream_t st)
{
    constexpr int W = Vec<Real>::n;
    const bool vec = (((uintptr_t)rho | (uintptr_t)the | (uintptr_t)hs | (uintptr_t)out) & 15) == 0;
    const long long per_cta = (long long)kRpThreads * W * 2;
    long long grid = (ncell + per_cta - 1) / per_cta;
    auto *cnt = reinterpret_cast<unsigned long long *>(d_cnt);
    const Real *r = (const Real *)rho, *t = (const Real *)the, *h = (const Real *)hs;
    Real *o = (Real *)out;
    // one wave: as many CTAs as are resident at once (registers decide: 5 per SM for the fp32 vector kernel), each
    // striding over the whole array, so that no partial second wave runs on a part of the machine
    auto go = [&](auto kern) {
        int per_sm = 1;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kRpThreads, 0) != cudaSuccess || per_sm < 1) per_sm = 1;
        const long long cap = (long long)nsm * per_sm;
        if (grid > cap) grid = cap;
        if (grid < 1) grid = 1;
        kern<<<(unsigned)grid, kRpThreads, 0, st>>>(r, t, h, o, ncell, K, cnt);
    };
    if (vec) {
        if (d_cnt) go(cool_radpress_kernel<Real, true, true>);
        else go(cool_radpress_kernel<Real, true, false>);
    } else {
        if (d_cnt) go(cool_radpress_kernel<Real, false, true>);
        else go(cool_radpress_kernel<Real, false, false>);
    }
    return cudaGetLastError();
}

}  // namespace

using cool::set_error;
using cool::note_launches;

extern "C" cool_status cool_radpress_correct(const cool_units *units, long long ncell, cool_dtype dtype, const void *d_rho,
                                             const void *d_theta_e, const void *d_hscale, double tau_crit,
                                             void *d_theta_e_out, long long *d_ncorrected, void *cuda_stream)
{
    if (!units) { set_error("cool_radpress_correct: units is NULL"); return COOL_EINVAL; }
    if (ncell < 0) { set_error("cool_radpress_correct: ncell < 0"); return COOL_EINVAL; }
    if (dtype != COOL_F32 && dtype != COOL_F64) { set_error("cool_radpress_correct: unknown dtype"); return COOL_EINVAL; }
    if (ncell > 0 && (!d_rho || !d_theta_e || !d_hscale || !d_theta_e_out)) { set_error("cool_radpress_correct: NULL cell array"); return COOL_EINVAL; }
    if (!(tau_crit >= 0.0) || !std::isfinite(tau_crit)) { set_error("cool_radpress_correct: tau_crit must be finite and >= 0"); return COOL_EINVAL; }
    if (!(units->rho_scale_cgs > 0.0) || !(units->mbh_msun > 0.0)) { set_error("cool_radpress_correct: rho_scale_cgs and mbh_msun must be > 0"); return COOL_EINVAL; }
    int dev = 0, nsm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) { set_error("cool_radpress_correct: no usable CUDA device: %s", cudaGetErrorString(e)); return COOL_ECUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // CODATA-2018 cgs; the radiation constant is the value the paper prints (L345)
    const double kB = 1.380649e-16, me = 9.1093837015e-28, mp = 1.67262192369e-24, cl = 2.99792458e10;
    const double sigT = 6.6524587321e-25, gmsun = 1.32712440018e26, arad = 7.5646e-15;
    const double n_per_rho = units->rho_scale_cgs / mp, rg = gmsun * units->mbh_msun / (cl * cl), tk = me * cl * cl / kB;
    RpConst K;
    K.c_tau = n_per_rho * sigT * rg;
    K.c_beta = arad * tk * tk * tk / (n_per_rho * kB);
    K.tau_crit = tau_crit;
    if (dtype == COOL_F32 && !(K.c_beta < 1e30 && K.c_tau < 1e30)) { set_error("cool_radpress_correct: units out of fp32 range"); return COOL_EINVAL; }
    if (d_ncorrected) {
        e = cudaMemsetAsync(d_ncorrected, 0, sizeof(long long), st);
        if (e != cudaSuccess) { set_error("cool_radpress_correct: cudaMemsetAsync: %s", cudaGetErrorString(e)); return COOL_ECUDA; }
    }
    note_launches(0);
    if (ncell == 0) return COOL_OK;
    e = dtype == COOL_F32 ? rp_launch<float>(d_rho, d_theta_e, d_hscale, d_theta_e_out, ncell, K, d_ncorrected, nsm, st)
                          : rp_launch<double>(d_rho, d_theta_e, d_hscale, d_theta_e_out, ncell, K, d_ncorrected, nsm, st);
    if (e != cudaSuccess) { set_error("cool_radpress_correct: launch: %s", cudaGetErrorString(e)); return COOL_ECUDA; }
    note_launches(1);
    return COOL_OK;
}
