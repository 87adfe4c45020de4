// cool_internal.h — private declarations shared by the translation units of libcool_b200.so.
#pragma once
#include <cuda_runtime.h>
#include <map>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/cool.h"
#include "cool_physics.cuh"

namespace cool {

// Canonical device axis order (the library re-lays the caller's table out at create time):
//   MODE 3 (ndim 3, nproc 1):  [rho][theta_e][bsq]            bsq fastest, float texels
//   MODE 4 (ndim 4, nproc 3):  [rho][theta_e][theta_i][bsq]   bsq fastest, float4 texels
//                              {log10 Qbrem, log10 Qsyn, log10 eta, 0}
// bsq is fastest because in GRMHD fields plasma-beta varies cell to cell far more than rho or
// Theta do along a grid line, so the scattered index stays inside one contiguous table row.
enum { CAX_RHO = 0, CAX_THE = 1, CAX_THI = 2, CAX_BSQ = 3 };   // canonical slots (THI unused in MODE 3)

struct AxisCoef {          // node-index coordinate t of a primitive q along one table axis
    int n;
    // fp64 path
    double lo10, inv10;    // t = (log10 q - lo10) * inv10
    // fp32 path: log2 q = e + lm (e integer, lm in [0,1)):  t = (e - e0)*invf + (lm*invf + cf)
    float e0, invf, cf;
    float nm1f, tmaxf;     // n-1 (clamp flag) and the largest float below n-1 (keeps floor(t) <= n-2)
    float ke;              // 2^23 + 127 + e0: (2^23 + biased exponent) - ke = e - e0, exactly
    float d2f;             // node spacing in log2 units (clamp correction of the fp32 path)
    float c2f;             // t = log2(q)*invf + c2f (single-lg2 form)
};

struct DevTable {
    int mode;                      // 3 or 4; 0 = no data (analytic only)
    AxisCoef ax[4];                // indexed by CAX_*
    int s_rho, s_the, s_thi;       // strides in texels (bsq stride = 1)
    const float *lin1;             // MODE 3 linear copy
    const float4 *lin4;            // MODE 4 linear copy
    cudaTextureObject_t tex_pt, tex_lin;   // 3-D array: x = bsq, y = theta_e (MODE 3) / theta_i (MODE 4),
                                           // z = rho (MODE 3) / rho*n_the + i_the (MODE 4, the paper's flattening)
    unsigned table_bytes;          // bytes of the linear copy (for the smem variant)
    // fp32 path: the same nodes re-expressed as log2 of the rate per unit electron energy,
    //   MODE 3: f1 = log2(Lambda ge1 / (mr rho_node Theta_e_node))
    //   MODE 4: f4 = {log2(Q_brem ge1/(mr rho Theta_e)), log2(Q_syn ge1/(mr rho Theta_e)), log2 eta, log2 C or 0}
    // so that Lambda h / u_e = 2^(interp + log2 h) without cancelling large fp32 numbers.
    const float *f1;
    const float4 *f4;
    const float4 *o3;              // MODE 3 oct layout: 8 corners of a table cell per 32-byte element (2 float4), plain strides; NULL when too large
    const float4 *q3;              // MODE 3 quad layout {T'(r,e,b), T'(r,e,b+1), T'(r,e+1,b), T'(r,e+1,b+1)}, plain strides; NULL when too large
    cudaTextureObject_t ftex_pt, ftex_lin;
    const float *fcoul;            // log2 C [theta_i][theta_e] (allocation padded to 16 B)
    const float4 *fcoulq;          // the same as quads {C(i,e), C(i,e+1), C(i+1,e), C(i+1,e+1)}
    int coulq_bytes, coulq_stride;  // row stride of the quads in float4 units (nc[1] + 2: bank skew, see cool_api.cu)
    int f4_has_coul;               // MODE 4: f4.w = log2 C (Coulomb axes identical to the table's Theta axes)
    // Coulomb coefficient table log10 C [theta_i][theta_e]
    const float *coul;
    AxisCoef cax[2];               // 0: theta_i, 1: theta_e
    int coul_bytes;                // size of the Coulomb table (staged in shared memory when small)
    int coul_share_the, coul_share_thi;   // Coulomb axis identical to the table's Theta_e / Theta_i axis
    // Steep Theta_e intervals (fp32 path): where neighbouring Theta_e nodes of T' differ by more than kSteepLog2 (weighted by
    // the channel's share of Q_thin for the process tables) the fp32 node coordinate (<= 5e-6 nodes) and the fp32 state
    // carried between sub-steps cannot hold the 1e-5 tolerance: the K2 -> 2 theta^2 switch of PAPER.md L87 is a 16-19
    // log2-unit step between two nodes, a local power-law index of 60-140.  All steep intervals together make one band
    // band_lo < Theta_e < band_hi (a margin included; the paper's tables have exactly one steep interval).  A cell that is inside a band at the start of a
    // sub-step in which it radiates a fraction r of its electron energy with fix_rmin < r < fix_rmax (F32Const) is left to
    // the precise pass (cool_fix.cu: the fp64 step on the canonical log10 tables): below fix_rmin the steep rate cannot move
    // the result by more than 1.5e-6, above fix_rmax the 30 % limiter decides whatever the rate.
    // mode 5, the paper's table (cool_cgs.cu): lin1 = [H][B][n_e][T_e] float (T_e fastest), ax[0..3] = those axes in this
    // order; tex_pt / tex_lin: 3-D array x = B, y = H_th, z = i_ne * n_Te + i_Te (the paper's flattening, L155-L159);
    // coul3 = log10 [Q_cc/(T_i - T_e)] over [n_e][T_i][T_e], axes cax3[0..2]
    const float *coul3;
    AxisCoef cax3[3];
    int nband;                     // 0: none, 1: band_lo < Theta_e < band_hi
    float band_lo, band_hi;
    float band_step;               // steepest step of the band [log2 units per node]
    int band_k0, band_k1;          // first and last steep Theta_e interval (0 .. n-2); the whole axis when another axis is steep
};
constexpr double kSteepLog2 = 6.0;        // |Delta T'| per Theta_e node above which an interval is steep (precision budget)
constexpr double kBandMargin = 1.0 / 128; // nodes; far above the distance between the fp32 and the fp64 trajectory of a cell (<= 2e-4 nodes)

struct DevConst {
    coolphys::Units units;
    coolphys::Derived der;
    double mr, ge1, gi1;           // m_e/m_p, gamma_e - 1, gamma_i - 1
    double coul_k;                 // dTheta_e/dt from Coulomb = coul_k * rho * C * (Th_i - Th_e) * ge1
    // MODE 4 combine (eqs 10-14) in code units
    double bb_k;                   // (4 sigma_SB T^4 conv) = bb_k * Theta_e^4
    double tausca_k;               // tau_sca = tausca_k * rho * H_cm
    double log2_ue_k;              // log2(u_e) = log2 rho + log2 Theta_e + this
};

struct LaunchArgs {
    long long ncell;
    const void *rho, *bsq, *the_in, *thi_in, *r, *vol;
    void *the_out, *thi_out;
    double dt; int nsub; double f_limit, h_floor;
    int coulomb;                   // 0 off, 1 table, 2 analytic
    int scheme;                    // 0 explicit, 1 implicit
    int want_diag;
    double *partials;              // [grid][8]
    unsigned *ticket;
    cool_diag *d_diag;
    double *lum_shell;             // device [nshell][4] or NULL (zeroed by the caller; the launch ADDS its shells)
    double *shell_rep;             // workspace [kShellReplicas][shell_nloc4], zeroed per launch
    long long shell_cells, cell_offset, shell0;   // shell0: first shell this launch touches
    unsigned shell_nloc4;          // 4 x number of shells this launch touches
    unsigned shell_rmask;          // number of replicas - 1
    unsigned char *flags;          // per-cell event flags (device) or NULL
    unsigned *fixmap;              // precise pass workspace (see fix_layout); NULL: no pass
    mutable unsigned fix_warps, fix_cap;   // set by the fp32 launch: its number of warps and the list slots each of them owns
};
// Precise-pass work lists inside LaunchArgs::fixmap, for an fp32 launch of `warps` warps over `ntiles` warp tiles:
//   count[warps] | tile[warps * cap] | words[warps * cap] (uint4, 16-byte aligned),  cap = ceil(ntiles / warps)
// warp w lists the tiles in which it marked cells at slots [w * cap, w * cap + count[w]); bit `lane` of word j of a tile
// stands for cell tile*128 + lane*4 + j.
constexpr int kFixMaxWarpsPerSm = 32;
struct FixLists { unsigned *count, *tile; uint4 *words; unsigned cap; };
inline FixLists fix_layout(unsigned *base, unsigned warps, long long ntiles)
{
    FixLists f;
    f.cap = (unsigned)((ntiles + warps - 1) / warps);
    f.count = base;
    f.tile = base + warps;
    size_t off = ((size_t)warps + (size_t)warps * f.cap) * 4;
    off = (off + 15) & ~(size_t)15;
    f.words = (uint4 *)((char *)base + off);
    return f;
}

// radial-profile atomics are spread over 32 (small launches) or 256 copies (by block / warp index): at any moment nearly all
// warps work in the same shell, and the L2 serialises atomics to one address
constexpr int kShellReplicasSmall = 32, kShellReplicasLarge = 256;
struct DiagWorkspace { double *partials = nullptr; unsigned *ticket = nullptr; int capacity_blocks = 0; double *shell_rep = nullptr; size_t shell_cap = 0;
                       unsigned *fixmap = nullptr; size_t fixmap_cap = 0; };

}  // namespace cool

struct cool_table {
    int device = 0;
    cool_table_desc desc{};        // host_data pointers nulled
    cool::DevTable dev{};
    cool::DevConst cst{};
    float *d_lin = nullptr;        // owns lin1 / lin4
    float *d_f32 = nullptr;        // owns f1 / f4
    float *d_coul = nullptr, *d_fcoul = nullptr, *d_fcoulq = nullptr, *d_q3 = nullptr, *d_o3 = nullptr, *d_coul3 = nullptr;
    cudaArray_t arr = nullptr, arr32 = nullptr;
    int sm_count = 148;
    int max_smem_optin = 0;
    bool persist_l2 = false;
    mutable std::mutex mu, host_mu;
    mutable std::map<cudaStream_t, cool::DiagWorkspace> diag_ws;     // per-stream, so concurrent streams never share
    // host-path staging (cool_apply_host), created lazily, used under mu
    struct HostStage { cudaStream_t s = nullptr; void *buf[8] = {}; cool_diag *d_diag = nullptr; unsigned char *flags = nullptr; };
    mutable std::vector<HostStage> stages;
    mutable size_t stage_bytes = 0;         // per staging buffer
    mutable cool_diag *h_diag_pinned = nullptr;
    mutable size_t h_diag_cap = 0;
    mutable double *d_shell = nullptr;       // host path: device copy of the radial profile
    mutable size_t d_shell_cap = 0;
};

namespace cool {
void set_error(const char *fmt, ...);
void note_launches(int n);           // what cool_last_launch_count() reports for this thread
void note_kernel(const char *fmt, ...);   // what cool_last_kernel_name() reports for this thread
bool desc_valid(const cool_table_desc *d, bool need_coulomb_shape, std::string *why);
bool desc_is_cgs(const cool_table_desc *d);          // the paper's table: axes (log H_th, log B, log n_e, log T_e)
coolphys::Units to_units(const cool_units &u);
cool_status launch_step(const cool_table *t, cool_variant v, cool_dtype dt, const LaunchArgs &a, cudaStream_t s, int *nlaunch);
bool variant_supported(const cool_table *t, cool_variant v, cool_dtype dt, std::string *why);
bool uses_fixmap(const cool_table *t, cool_variant v, cool_dtype dt, const LaunchArgs &a);
}
