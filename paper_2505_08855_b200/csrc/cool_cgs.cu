// cool_cgs.cu — the cooling step on THE PAPER'S OWN TABLE: Q(H_th, B, n_e, T_e) in cgs units on
// log-spaced axes, the Coulomb table Q_cc(n_e, T_i, T_e) (L147), and the paper's texture layout
// (L155-L159).  Per cell and sub-step (L181: "the values of H_th, B, n_e and T_e obtained from the simulation"):
//   H_th = c_s/Omega_K (eqs 13-14) with the CELL'S OWN radius,  B = sqrt(4 pi b^2 rho_scale c^2),  n_e = rho rho_scale/m_p,
//   T_e = Theta_e m_e c^2/k_B  ->  log10 coordinates, edge clamp  ->  4-D interpolation of log10 Q  ->  Lambda = 10^y conv
// and then the floor, Coulomb exchange, 30 % limiter and update of update64 (cool_kernels.cuh), shared with the fp64 path.
//
// Lookup variants (north_star: they compete):
//   GLOBAL       16 corner gathers from the linear array [H][B][n_e][T_e] (T_e fastest: the (n_e, T_e) pair of a cell's
//                neighbourhood lies in two runs of two floats per (H, B) corner);
//   TEX_POINT    the same 16 corners as point fetches from the 3-D texture (x = B, y = H_th, z = i_ne n_Te + i_Te);
//   TEX_HWFILTER the paper's scheme: the hardware filters (H_th, B) bilinearly at the four (n_e, T_e) corners, the flattened
//                axis is interpolated by hand — 4 fetches instead of 16, with the filter's 8-bit weights (reported, not gated);
//   ANALYTIC     eqs 1-12 per cell with the cell's H_th (cool_kernels.cuh, step_cell_analytic).
// All arithmetic is fp64 for both cell dtypes: at 100^4 (400 MB, beyond L2) the step is bound by the 16 scattered sectors
// per cell, not by arithmetic, and the table's T_e axis contains the K2 -> 2 theta^2 step of L87, which fp32 coordinates
// cannot carry.  One thread per cell, 128-bit streaming loads and stores of the SoA arrays.
#include "cool_kernels.cuh"

namespace cool {

enum { CGS_GLOBAL = 0, CGS_TEXPT = 1, CGS_TEXHW = 2 };

struct CgsConst {
    double ne_per_rho, b2_per_bsq, theta_to_K, rate_conv, rg_cm;        // unit conversions (cool_physics.cuh, Derived)
    int coulomb3;                                                       // Coulomb from the paper's 3-D table
};

template <int VAR>
__device__ __forceinline__ double cgs_lookup(const DevTable &T, const Loc64 &lh, const Loc64 &lb, const Loc64 &ln, const Loc64 &lt)
{
    const int nB = T.ax[1].n, nN = T.ax[2].n, nT = T.ax[3].n;
    double y = 0.0;
    if constexpr (VAR == CGS_TEXHW) {
        // hardware bilinear on (B, H_th) at the four (n_e, T_e) corners; manual interpolation on the flattened axis (L159)
        const float x = (float)(lb.i + lb.w) + 0.5f, yy = (float)(lh.i + lh.w) + 0.5f;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int cn = c >> 1, ct = c & 1;
            const double pw = (cn ? ln.w : 1.0 - ln.w) * (ct ? lt.w : 1.0 - lt.w);
            y += pw * (double)tex3D<float>(T.tex_lin, x, yy, (float)((ln.i + cn) * nT + (lt.i + ct)) + 0.5f);
        }
    } else {
#pragma unroll
        for (int c = 0; c < 16; ++c) {
            const int ch = c >> 3, cb = (c >> 2) & 1, cn = (c >> 1) & 1, ct = c & 1;
            const double pw = (ch ? lh.w : 1.0 - lh.w) * (cb ? lb.w : 1.0 - lb.w) * (cn ? ln.w : 1.0 - ln.w) * (ct ? lt.w : 1.0 - lt.w);
            float v;
            if constexpr (VAR == CGS_GLOBAL) v = __ldg(T.lin1 + ((((size_t)(lh.i + ch) * nB + (lb.i + cb)) * nN + (ln.i + cn)) * nT + (lt.i + ct)));
            else v = tex3D<float>(T.tex_pt, (float)(lb.i + cb) + 0.5f, (float)(lh.i + ch) + 0.5f, (float)((ln.i + cn) * nT + (lt.i + ct)) + 0.5f);
            y += pw * (double)v;
        }
    }
    return y;
}

template <int VAR, bool DIAG>
__device__ __forceinline__ void cgs_cell(const DevTable &T, const DevConst &K, const StepConst &S, const CgsConst &G,
                                         double rho, double bsq, double &the, double &thi, double r, double vol, DiagAcc &acc, long long cell, int *flags)
{
    if (isnan(rho) || isnan(bsq) || isnan(the) || isnan(thi)) { the = thi = __longlong_as_double(0x7ff8000000000000LL); return; }
    if (!(rho > 0.0)) return;
    const double ne = G.ne_per_rho * rho;
    const Loc64 ln = locate64(T.ax[2], ne), lb = locate64(T.ax[1], sqrt(G.b2_per_bsq * fmax(bsq, 0.0)));
    const double h_per_cs = G.rg_cm * ((r > 0.0 ? r * sqrt(r) : K.units.r_ref_rg * sqrt(K.units.r_ref_rg)) + S.spin);      // 1/Omega_K of THIS cell (eq 13)
    int limited = 0, floored = 0, clamped = ln.clamped | lb.clamped;
    double de_sum[4] = {0, 0, 0, 0};
    const double frac[3] = {0, 0, 0};
    for (int s = 0; s < S.nsub; ++s) {
        const double cs2 = (S.ae * the + S.ai * thi) / (1.0 + S.be * the + S.bi * thi);              // eq 14
        const Loc64 lh = locate64(T.ax[0], h_per_cs * sqrt(cs2)), lt = locate64(T.ax[3], the * G.theta_to_K);
        clamped |= lh.clamped | lt.clamped;
        const double lam = exp10(cgs_lookup<VAR>(T, lh, lb, ln, lt)) * G.rate_conv;
        if (G.coulomb3) {
            // update64 with the Coulomb term of the paper's table: Q_cc = 10^(interp) (T_i - T_e), per kelvin (C-23)
            const Loc64 a = locate64(T.cax3[0], ne), b = locate64(T.cax3[1], thi * G.theta_to_K), c = locate64(T.cax3[2], the * G.theta_to_K);
            const int n1 = T.cax3[1].n, n2 = T.cax3[2].n;
            double yk = 0.0;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int ca = q >> 2, cb = (q >> 1) & 1, cc = q & 1;
                yk += (ca ? a.w : 1.0 - a.w) * (cb ? b.w : 1.0 - b.w) * (cc ? c.w : 1.0 - c.w) *
                      (double)__ldg(T.coul3 + (((size_t)(a.i + ca) * n1 + (b.i + cb)) * n2 + (c.i + cc)));
            }
            // dTheta_e/dt = Q_cc (gamma_e - 1)/(rho m_e/m_p): hand update64 the same product it forms from coul_kh rho C D
            const double qcc_per_D = exp10(yk) * G.theta_to_K * G.rate_conv;                          // Q_cc / (Theta_i - Theta_e), code units
            update64_q(S, rho, r, lam, frac, the, thi, de_sum, limited, floored, qcc_per_D);
        } else {
            update64(T, K, S, rho, r, lam, frac, the, thi, de_sum, limited, floored);
        }
    }
    if constexpr (DIAG) {
        const double wgt = rho * vol;
        acc.lum[0] += de_sum[0] * wgt;
        acc.lim += limited; acc.flo += floored; acc.cla += clamped;
        shell_add(S, cell, de_sum, wgt, false);
        if (flags) *flags = limited | (floored << 1) | (clamped << 2);
    }
}

template <class Real, int VAR, bool DIAG>
__global__ void __launch_bounds__(256)
cool_cgs_kernel(const DevTable T, const DevConst K, const StepConst S, const CgsConst G, const CellPtrs C, double *partials, unsigned *ticket, cool_diag *d_diag)
{
    using V = typename VecT<Real>::type;
    constexpr int N = VecT<Real>::N;
    DiagAcc acc;
    const long long nvec = S.aligned ? C.ncell / N : 0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < nvec; v += stride) {
        V rho = ld_stream((const V *)C.rho + v), bsq = ld_stream((const V *)C.bsq + v);
        V the = ld_stream((const V *)C.the_in + v), thi = ld_stream((const V *)C.thi_in + v);
        V rr, vv;
#pragma unroll
        for (int j = 0; j < N; ++j) { vget(rr, j) = (Real)0; vget(vv, j) = (Real)1; }
        if (C.r) rr = ld_stream((const V *)C.r + v);
        if (S.has_vol) vv = ld_stream((const V *)C.vol + v);
#pragma unroll
        for (int j = 0; j < N; ++j) {
            double te = (double)vget(the, j), ti = (double)vget(thi, j);
            int fl = 0;
            cgs_cell<VAR, DIAG>(T, K, S, G, (double)vget(rho, j), (double)vget(bsq, j), te, ti, (double)vget(rr, j), (double)vget(vv, j), acc, v * N + j, &fl);
            vget(the, j) = (Real)te; vget(thi, j) = (Real)ti;
            if (DIAG && C.flags) C.flags[v * N + j] = (unsigned char)fl;
        }
        st_stream((V *)C.the_out + v, the);
        st_stream((V *)C.thi_out + v, thi);
    }
    for (long long c = nvec * N + (long long)blockIdx.x * blockDim.x + threadIdx.x; c < C.ncell; c += stride) {
        double te = (double)((const Real *)C.the_in)[c], ti = (double)((const Real *)C.thi_in)[c];
        int fl = 0;
        cgs_cell<VAR, DIAG>(T, K, S, G, (double)((const Real *)C.rho)[c], (double)((const Real *)C.bsq)[c], te, ti,
                            C.r ? (double)((const Real *)C.r)[c] : 0.0, S.has_vol ? (double)((const Real *)C.vol)[c] : 1.0, acc, c, &fl);
        ((Real *)C.the_out)[c] = (Real)te; ((Real *)C.thi_out)[c] = (Real)ti;
        if (DIAG && C.flags) C.flags[c] = (unsigned char)fl;
    }
    if constexpr (DIAG) reduce_diag(acc, S.lum_k, partials, ticket, d_diag);
}

template <class Real, int VAR, bool DIAG>
static cudaError_t launch_cgs_one(const LaunchCtx &L, const CgsConst &G)
{
    auto kern = cool_cgs_kernel<Real, VAR, DIAG>;
    int occ = 0;
    cudaError_t eo = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, 256, 0);
    if (eo != cudaSuccess) return eo;
    if (occ < 1) occ = 1;
    const LaunchArgs &a = *L.a;
    constexpr int N = VecT<Real>::N;
    long long need = (a.ncell / N + 255) / 256;
    if (need < 1) need = 1;
    const long long cap = (long long)L.t->sm_count * (occ < 32 ? occ : 32);
    const int grid = (int)(need < cap ? need : cap);
    CellPtrs C{a.rho, a.bsq, a.the_in, a.thi_in, a.r, a.vol, a.the_out, a.thi_out, a.ncell, a.flags};
    kern<<<grid, 256, 0, L.st>>>(L.t->dev, L.t->cst, *L.S, G, C, a.partials, a.ticket, a.d_diag);
    return cudaGetLastError();
}

cudaError_t launch_cgs(const LaunchCtx &L, cool_variant v, cool_dtype dt, bool diag)
{
    const DevConst &K = L.t->cst;
    CgsConst G{K.der.ne_per_rho, K.der.b2_per_bsq, coolphys::kTHETA_TO_K, K.der.rate_conv, K.der.rg_cm, (L.S->coulomb == 1 && L.t->dev.coul3) ? 1 : 0};
#define COOL_CGS_GO(R, VAR) (diag ? launch_cgs_one<R, VAR, true>(L, G) : launch_cgs_one<R, VAR, false>(L, G))
    const int var = v == COOL_V_GLOBAL ? CGS_GLOBAL : (v == COOL_V_TEX_POINT ? CGS_TEXPT : CGS_TEXHW);
    if (dt == COOL_F32) return var == CGS_GLOBAL ? COOL_CGS_GO(float, CGS_GLOBAL) : (var == CGS_TEXPT ? COOL_CGS_GO(float, CGS_TEXPT) : COOL_CGS_GO(float, CGS_TEXHW));
    return var == CGS_GLOBAL ? COOL_CGS_GO(double, CGS_GLOBAL) : (var == CGS_TEXPT ? COOL_CGS_GO(double, CGS_TEXPT) : COOL_CGS_GO(double, CGS_TEXHW));
#undef COOL_CGS_GO
}

// ---- device table builder for the paper's table ---------------------------------------------------------------------------
// 100^4 nodes take the host builder minutes; the same cool_physics.cuh code on the device takes a second.
__global__ void __launch_bounds__(128) cgs_build_kernel(int n0, int n1, int n2, int n3, double lo0, double lo1, double lo2, double lo3,
                                                        double d0, double d1, double d2, double d3, float *out, long long total)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long f = (long long)blockIdx.x * blockDim.x + threadIdx.x; f < total; f += stride) {
        long long rem = f;
        const int i3 = (int)(rem % n3); rem /= n3;
        const int i2 = (int)(rem % n2); rem /= n2;
        const int i1 = (int)(rem % n1); const int i0 = (int)(rem / n1);
        (void)n0;
        const coolphys::Cooling c = coolphys::cooling_cgs(pow(10.0, lo0 + i0 * d0), pow(10.0, lo1 + i1 * d1), pow(10.0, lo2 + i2 * d2),
                                                          pow(10.0, lo3 + i3 * d3) / coolphys::kTHETA_TO_K);
        out[f] = (float)log10(c.total);
    }
}

}  // namespace cool

extern "C" cool_status cool_table_build_device(const cool_table_desc *shape, int device, float *host_out)
{
    using namespace cool;
    std::string why;
    if (!desc_valid(shape, false, &why)) { set_error("cool_table_build_device: %s", why.c_str()); return COOL_EINVAL; }
    if (!desc_is_cgs(shape) || shape->nproc != 1) { set_error("cool_table_build_device: only the paper's table (axes LOG_HTH, LOG_B, LOG_NE, LOG_TE; nproc = 1)"); return COOL_EUNSUPPORTED; }
    if (!host_out) { set_error("cool_table_build_device: host_out is NULL"); return COOL_EINVAL; }
    int prev = -1;
    if (cudaGetDevice(&prev) != cudaSuccess || cudaSetDevice(device) != cudaSuccess) { set_error("cool_table_build_device: no usable CUDA device %d", device); return COOL_ECUDA; }
    const long long total = (long long)shape->n[0] * shape->n[1] * shape->n[2] * shape->n[3];
    float *d = nullptr;
    cudaError_t e = cudaMalloc(&d, (size_t)total * sizeof(float));
    if (e == cudaSuccess) {
        double dd[4];
        for (int k = 0; k < 4; ++k) dd[k] = (shape->hi[k] - shape->lo[k]) / (shape->n[k] - 1);
        const long long blocks = (total + 127) / 128;
        cgs_build_kernel<<<(int)(blocks < 148 * 64 ? blocks : 148 * 64), 128>>>(shape->n[0], shape->n[1], shape->n[2], shape->n[3], shape->lo[0], shape->lo[1],
                                                                               shape->lo[2], shape->lo[3], dd[0], dd[1], dd[2], dd[3], d, total);
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaMemcpy(host_out, d, (size_t)total * sizeof(float), cudaMemcpyDeviceToHost);
    }
    if (d) cudaFree(d);
    if (prev >= 0) cudaSetDevice(prev);
    if (e != cudaSuccess) { set_error("cool_table_build_device: %s", cudaGetErrorString(e)); return e == cudaErrorMemoryAllocation ? COOL_ENOMEM : COOL_ECUDA; }
    return COOL_OK;
}
