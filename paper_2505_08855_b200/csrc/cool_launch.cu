// cool_launch.cu — per-launch constants and dispatch to the kernel instantiations.
#include <algorithm>
#include <cstring>

#include "cool_implicit.cuh"

namespace cool {

// Radial profile, second (tiny) launch: add the replicas of the step launch's shells into the caller's array, in a fixed
// order over the replicas.  Kept out of reduce_diag_vals on purpose: growing that non-inlined function cost the step
// kernels that call it 8 % more instructions in their hot loops (measured).
static __global__ void shell_reduce_kernel(const double *rep, double *out, unsigned nloc4, long long shell0, unsigned rmask)
{
    const unsigned idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= nloc4) return;
    double s = 0.0;
    for (unsigned r = 0; r <= rmask; ++r) s += rep[(size_t)r * nloc4 + idx];
    if (s != 0.0) atomicAdd(out + 4 * shell0 + idx, s);
}

static StepConst make_step_const(const cool_table *t, cool_dtype dt, const LaunchArgs &a)
{
    const DevConst &K = t->cst;
    StepConst S{};
    S.h = a.dt / a.nsub; S.f_limit = a.f_limit;
    S.mr = K.mr; S.ge1 = K.ge1; S.gi1 = K.gi1; S.eq_frac = K.ge1 / (K.ge1 + K.gi1);
    S.coul_kh = K.coul_k * S.h * K.ge1;
    S.bb_k = K.bb_k; S.tausca_k = K.tausca_k; S.h_per_cs = K.der.h_per_cs; S.hth_cm = K.units.hth_cm;
    S.ae = K.units.gamma_e * K.mr; S.ai = K.units.gamma_i * K.mr;
    S.be = K.mr * K.units.gamma_e / K.ge1; S.bi = K.mr * K.units.gamma_i / K.gi1;
    S.hfloor2 = (a.h_floor > 0.0 && a.r) ? 0.5 * coolphys::kPI * a.h_floor * a.h_floor : 0.0;
    S.spin = K.units.spin;
    S.lum_k = K.mr / (K.ge1 * a.dt);
    S.nsub = a.nsub; S.coulomb = a.coulomb;
    S.cgs = desc_is_cgs(&t->desc); S.omk_ref_inv = pow(K.units.r_ref_rg, 1.5) + K.units.spin;
    S.has_r = a.r != nullptr && (S.hfloor2 > 0.0 || S.cgs); S.has_vol = a.vol != nullptr && a.want_diag;      // arrays nobody uses are not read
    auto ok = [&](const void *p) { return p == nullptr || ((size_t)p % 16) == 0; };
    S.lum_shell = a.lum_shell ? a.shell_rep : nullptr; S.shell_cells = a.shell_cells > 0 ? a.shell_cells : 1;
    S.cell_offset = a.cell_offset; S.shell0 = a.shell0; S.shell_nloc4 = a.shell_nloc4; S.shell_rmask = a.shell_rmask;
    S.aligned = ok(a.rho) && ok(a.bsq) && ok(a.the_in) && ok(a.thi_in) && ok(a.the_out) && ok(a.thi_out) && ok(a.r) && ok(a.vol);
    return S;
}

// Coulomb coefficient table staged in shared memory (not needed when it rides in the 4-D texels): returns the kernels'
// CM — 0 not staged, 1 quads (<= 72 KiB; the SMEM variant stores the plain table under CM = 1), 2 plain table (<= 16 KiB)
// for launches with diagnostics that are small or stage no radius array.  Measured on B200 (table 128^3, Coulomb 64^2):
// 288x192x144 cells with the floor 0.089 (quads) / 0.077 ms (plain); 512^3 with the floor (6 cell arrays) 0.910 / 0.927 ms;
// 512^3 without it (5 arrays: the plain table keeps the CTA under the 164 KiB carve-out) 0.849 / 0.784 ms.
constexpr long long kCoulPlainBelowCells = 1ll << 25;
static int coulomb_smem_mode(const cool_table *t, const LaunchArgs &a, cool_variant v)
{
    const DevTable &D = t->dev;
    if (a.coulomb != 1 || !D.fcoul || (D.mode == 4 && D.f4_has_coul)) return 0;
    if (v == COOL_V_SMEM) return D.coul_bytes <= kCoulSmemMax ? 1 : 0;
    if (a.want_diag && (a.ncell < kCoulPlainBelowCells || a.r == nullptr) && D.coul_bytes <= kCoulSmemMax) return 2;
    return D.coulq_bytes <= kCoulQuadSmemMax ? 1 : 0;
}

static F32Const make_f32_const(const cool_table *t, const LaunchArgs &a)
{
    const DevConst &K = t->cst;
    F32Const S{};
    const double h = a.dt / a.nsub;
    S.k0 = (float)log2(h);
    S.f_limit = (float)a.f_limit; S.mr = (float)K.mr; S.eq_frac = (float)(K.ge1 / (K.ge1 + K.gi1));
    S.gi1_over_ge1 = (float)(K.gi1 / K.ge1);
    S.coul_kh = (float)(K.coul_k * h * K.ge1);
    S.cap1e = (float)a.f_limit; S.cap1i = (float)(a.f_limit * K.ge1 / K.gi1);
    S.ae = (float)(K.units.gamma_e * K.mr); S.ai = (float)(K.units.gamma_i * K.mr);
    S.be = (float)(K.mr * K.units.gamma_e / K.ge1); S.bi = (float)(K.mr * K.units.gamma_i / K.gi1);
    S.inv_kB = (float)(K.der.h_per_cs * K.mr / (K.bb_k * h * K.ge1));
    S.ksca = (float)(K.tausca_k * K.der.h_per_cs);
    S.hfloor2 = (float)((a.h_floor > 0.0 && a.r) ? 0.5 * coolphys::kPI * a.h_floor * a.h_floor : 0.0);
    S.spin = (float)K.units.spin;
    S.lum_k = K.mr / (K.ge1 * a.dt);
    S.ion_ratio = K.units.ion_theta_mass_ratio;
    S.nsub = a.nsub; S.coulomb = a.coulomb;
    S.has_r = a.r != nullptr && S.hfloor2 > 0.f; S.has_vol = a.vol != nullptr && a.want_diag;      // arrays nobody uses are neither staged nor read
    S.nf = 4 + S.has_r + S.has_vol;
    S.fixmap = a.fixmap;
    {
        // precise-pass criterion (cool_internal.h): a band cell left to the fp32 path errs by at most r/(1-r) x step x ln 2 x dt_nodes,
        // dt_nodes = the fp32 path's worst node-coordinate error inside a band: 1e-5 (the tolerance itself) of Theta_e in
        // node units plus the coordinate's own 1e-5
        const DevTable &D0 = t->dev;
        const double dt_nodes = 1e-5 * 1.4426950408889634 / (double)D0.ax[CAX_THE].d2f + 1e-5;
        const double sens = 0.6931471805599453 * (double)D0.band_step * dt_nodes;
        const bool on = D0.nband != 0 && (a.fixmap != nullptr || (D0.mode == 3 && a.nsub == 1));
        auto bits = [](double x) { const float f = (float)x; unsigned u; memcpy(&u, &f, 4); return u; };
        const float hi = std::min(D0.band_hi, 3.0e38f);               // keep the width a finite-float difference
        const unsigned lo_b = bits(D0.band_lo), rmin_b = bits(1.5e-6 / sens), rmax_b = bits(a.f_limit * (1.0 + 2.0 * sens) + 1e-6);
        S.band_lo_bits = lo_b; S.band_w = on ? bits(hi) - lo_b : 0u;
        S.rmin_bits = rmin_b; S.r_w = (on && rmax_b > rmin_b) ? rmax_b - rmin_b : 0u;
    }
    S.lum_shell = a.lum_shell ? a.shell_rep : nullptr;
    S.shell_tiles = a.shell_cells > 0 ? (unsigned)(a.shell_cells / kWarpTile) : 1u; S.tile_offset = (unsigned)(a.cell_offset / kWarpTile);
    S.shell0 = (unsigned)a.shell0; S.shell_nloc4 = a.shell_nloc4; S.shell_rmask = a.shell_rmask;
    S.shell_magic = ((1ull << 40) + S.shell_tiles - 1) / S.shell_tiles;
    auto ok = [&](const void *p) { return p == nullptr || ((size_t)p % 16) == 0; };
    S.use_tma = ok(a.rho) && ok(a.bsq) && ok(a.the_in) && ok(a.thi_in) && ok(a.the_out) && ok(a.thi_out) && ok(a.r) && ok(a.vol) && ((size_t)a.flags % 4) == 0;
    // Coulomb-table node coordinates as an affine map of the table's own node coordinates
    const DevTable &D = t->dev;
    if (D.fcoul && D.mode != 0) {
        const AxisCoef &te = D.ax[CAX_THE], &ce = D.cax[1];
        S.cme_s = (float)(ce.inv10 / te.inv10); S.cme_o = (float)((te.lo10 - ce.lo10) * ce.inv10);
        if (D.mode == 4) {
            const AxisCoef &ti = D.ax[CAX_THI], &ci = D.cax[0];
            S.cmi_s = (float)(ci.inv10 / ti.inv10); S.cmi_o = (float)((ti.lo10 - ci.lo10) * ci.inv10);
        }
    }
    return S;
}

bool variant_supported(const cool_table *t, cool_variant v, cool_dtype, std::string *why)
{
    if (v == COOL_V_ANALYTIC) return true;
    if (t->dev.mode == 5 && v == COOL_V_SMEM) { if (why) *why = "the paper's table runs on the GLOBAL, TEX_POINT, TEX_HWFILTER and ANALYTIC lookups"; return false; }
    if (t->dev.mode == 0) { if (why) *why = "table has no data (nproc = 0): only COOL_V_ANALYTIC applies"; return false; }
    // SMEM variant: table image + the warps' 6-array cell stages + plain Coulomb table + barriers
    if (v == COOL_V_SMEM && (size_t)t->dev.table_bytes + kCoulSmemMax + (size_t)kF32SmemStages * 6 * (size_t)kF32SmemThreads * kF32CellsPerThread * 4 + kF32BarBytes > (size_t)t->max_smem_optin) {
        if (why) *why = "table does not fit in shared memory"; return false;
    }
    return true;
}

// The precise pass follows the fp32 software-interpolation kernels of the explicit scheme when the table has steep Theta_e
// intervals.  Not the hardware-filtered texture (its 8-bit weights miss the tolerance everywhere: reported, not gated), not
// fp64 cells or the analytic variant (already fp64), not the implicit scheme (a root solve is insensitive to the coordinate).
bool uses_fixmap(const cool_table *t, cool_variant v, cool_dtype dt, const LaunchArgs &a)
{
    // (a single update of a 3-D table needs no second kernel: its cells are exact inputs, and the step re-evaluates the rate of
    // a band cell in place, precise_rate3 of cool_f32.cuh)
    return t->dev.mode != 5 && t->dev.nband != 0 && dt == COOL_F32 && a.scheme == COOL_SCHEME_EXPLICIT && (v == COOL_V_GLOBAL || v == COOL_V_SMEM || v == COOL_V_TEX_POINT) &&
           (t->dev.mode == 4 || a.nsub > 1);
}

cool_status launch_step(const cool_table *t, cool_variant v, cool_dtype dt, const LaunchArgs &a_in, cudaStream_t st, int *nlaunch)
{
    LaunchArgs a_loc = a_in;
    // the analytic variant has no use for the paper's Coulomb TABLE: eq 15 analytically
    if (desc_is_cgs(&t->desc) && v == COOL_V_ANALYTIC && a_loc.coulomb == 1) a_loc.coulomb = 2;
    const LaunchArgs &a = a_loc;
    const StepConst S = make_step_const(t, dt, a);
    const LaunchCtx L{t, &S, &a, st};
    const int mode = t->dev.mode == 0 ? (t->desc.ndim == 4 ? 4 : 3) : t->dev.mode;
    const bool diag = a.want_diag != 0;
    cudaError_t e;
    bool fix = false;
    static const char *const vname[] = {"auto", "tex_point", "tex_hwfilter", "smem", "global", "analytic"};
    if (a.scheme == COOL_SCHEME_IMPLICIT) {
        note_kernel("%s<MODE=%d,%s>", dt == COOL_F64 ? "cool_implicit_kernel" : "cool_implicit_f32_kernel", mode, vname[v]);
        e = launch_implicit(L, make_f32_const(t, a), mode, v, dt);
    } else if (v == COOL_V_ANALYTIC) {
        note_kernel("cool_step_kernel<%s,MODE=%d,analytic,DIAG=%d>", dt == COOL_F64 ? "double" : "float", mode, (int)diag);
        e = launch_analytic(L, mode, dt, diag);
    } else if (t->dev.mode == 5) {
        note_kernel("cool_cgs_kernel<%s,%s,DIAG=%d>", dt == COOL_F64 ? "double" : "float", vname[v], (int)diag);
        e = launch_cgs(L, v, dt, diag);
    } else if (dt == COOL_F64) {
        note_kernel("cool_step_kernel<double,MODE=%d,%s,DIAG=%d>", mode, vname[v], (int)diag);
        e = launch_f64(L, mode, v, diag);
    }
    else {
        fix = a.fixmap && uses_fixmap(t, v, dt, a);
        LaunchArgs af = a;                                   // the fp32 kernels list cells for the precise pass only when it will run
        if (!fix) af.fixmap = nullptr;
        LaunchCtx32 L32{t, make_f32_const(t, af), &a, st};
        const int csm = coulomb_smem_mode(t, a, v);
        L32.S.coul_smem = csm != 0;
        // fast path: Coulomb from the coefficient table staged in shared memory (or riding in the 4-D texels)
        const int cm = a.coulomb == 1 ? (csm ? csm : (mode == 4 && t->dev.f4_has_coul ? 1 : 0)) : 0;
        e = (mode == 3) ? launch_f32_m3(L32, v, diag, cm, a.nsub == 1) : launch_f32_m4(L32, v, diag, cm);
    }
    if (e != cudaSuccess) { set_error("kernel launch failed: %s", cudaGetErrorString(e)); return COOL_ECUDA; }
    if (nlaunch) *nlaunch += 1;
    if (fix) {                                           // precise pass over the cells the fp32 kernel listed (steep table intervals)
        e = launch_fix(L, mode, diag);
        if (e != cudaSuccess) { set_error("kernel launch failed: %s", cudaGetErrorString(e)); return COOL_ECUDA; }
        if (nlaunch) *nlaunch += 1;
    }
    if (a.lum_shell) {                       // radial profile: fold this launch's replicas into the caller's array
        shell_reduce_kernel<<<(a.shell_nloc4 + 255) / 256, 256, 0, st>>>(a.shell_rep, a.lum_shell, a.shell_nloc4, a.shell0, a.shell_rmask);
        e = cudaGetLastError();
        if (e != cudaSuccess) { set_error("kernel launch failed: %s", cudaGetErrorString(e)); return COOL_ECUDA; }
        if (nlaunch) *nlaunch += 1;
    }
    return COOL_OK;
}

}  // namespace cool
