// cool_api.cu — the C ABI of include/cool.h: table objects, argument checking, launches,
// the host-buffer (end-to-end) path.  No compute happens here.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "cool_internal.h"

// Row skew of the Coulomb quads in float4 units: rows i and i+1 of one column would share their banks (a row of 64 quads is
// 1024 B), and the cells of a warp straddle both; 2 quads keep the 2 x 2 neighbourhood of a lookup in distinct bank groups.
// 64 x 66 quads + the stages of the 768-thread kernel fill the 163 KiB a CTA can have at the 164 KiB carve-out exactly
// (measured at 512^3: skew 0 0.627 ms, 1 0.619 ms, 2 0.614 ms; 3 needs the next carve-out step and is slower).
#ifndef COOL_COULQ_SKEW
#define COOL_COULQ_SKEW 2
#endif

namespace cool {

static thread_local char g_err[512] = "";
static thread_local int g_launches = 0;

void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}

void note_launches(int n) { g_launches = n; }

static thread_local char g_kernel[256] = "";
void note_kernel(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_kernel, sizeof g_kernel, fmt, ap);
    va_end(ap);
}

// restores the caller's current device when an entry point that had to switch to the table's device returns
struct DeviceGuard {
    int prev = -1;
    cudaError_t enter(int dev)
    {
        cudaError_t e = cudaGetDevice(&prev);
        if (e != cudaSuccess) { prev = -1; return e; }
        if (prev == dev) { prev = -1; return cudaSuccess; }
        return cudaSetDevice(dev);
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

#define CUDA_TRY(call, what)                                                            \
    do {                                                                                \
        cudaError_t e_ = (call);                                                        \
        if (e_ != cudaSuccess) {                                                        \
            set_error("%s: %s", what, cudaGetErrorString(e_));                          \
            return e_ == cudaErrorMemoryAllocation ? COOL_ENOMEM : COOL_ECUDA;          \
        }                                                                               \
    } while (0)

static int canon_slot(int axis_kind)
{
    switch (axis_kind) {
        case COOL_AX_LOG_RHO: return CAX_RHO;
        case COOL_AX_LOG_THETA_E: return CAX_THE;
        case COOL_AX_LOG_THETA_I: return CAX_THI;
        default: return CAX_BSQ;
    }
}

static AxisCoef make_axis(int n, double lo, double hi)
{
    AxisCoef a{};
    const double L10 = 3.321928094887362;
    const double delta = (hi - lo) / (n - 1);
    a.n = n;
    a.lo10 = lo; a.inv10 = 1.0 / delta;
    const double lo2 = lo * L10, inv2 = 1.0 / (delta * L10);
    const double e0 = floor(lo2);
    a.e0 = (float)e0; a.invf = (float)inv2;
    a.cf = (float)(-(lo2 - e0) * inv2);
    a.nm1f = (float)(n - 1);
    a.tmaxf = nextafterf(a.nm1f, 0.f);
    a.ke = (float)(8388608.0 + 127.0 + e0);
    a.d2f = (float)(delta * L10);
    a.c2f = (float)(-lo2 * inv2);
    return a;
}

// 3-D cudaArray + point / linear texture objects over a canonical host array (x = bsq fastest)
static cudaError_t make_textures(const float *host, int chan, size_t ex, size_t ey, size_t ez, cudaArray_t *arr,
                                 cudaTextureObject_t *pt, cudaTextureObject_t *lin)
{
    cudaChannelFormatDesc cd = chan == 1 ? cudaCreateChannelDesc<float>() : cudaCreateChannelDesc<float4>();
    cudaError_t e = cudaMalloc3DArray(arr, &cd, make_cudaExtent(ex, ey, ez));
    if (e != cudaSuccess) return e;
    cudaMemcpy3DParms cp{};
    cp.srcPtr = make_cudaPitchedPtr((void *)host, ex * chan * sizeof(float), ex, ey);
    cp.dstArray = *arr;
    cp.extent = make_cudaExtent(ex, ey, ez);
    cp.kind = cudaMemcpyHostToDevice;
    e = cudaMemcpy3D(&cp);
    if (e != cudaSuccess) return e;
    cudaResourceDesc rd{};
    rd.resType = cudaResourceTypeArray; rd.res.array.array = *arr;
    cudaTextureDesc td{};
    td.addressMode[0] = td.addressMode[1] = td.addressMode[2] = cudaAddressModeClamp;
    td.readMode = cudaReadModeElementType; td.normalizedCoords = 0;
    td.filterMode = cudaFilterModePoint;
    e = cudaCreateTextureObject(pt, &rd, &td, nullptr);
    if (e != cudaSuccess) return e;
    td.filterMode = cudaFilterModeLinear;
    return cudaCreateTextureObject(lin, &rd, &td, nullptr);
}

static void free_table(cool_table *t)
{
    if (!t) return;
    DeviceGuard dg;
    dg.enter(t->device);
    if (t->dev.tex_pt) cudaDestroyTextureObject(t->dev.tex_pt);
    if (t->dev.tex_lin) cudaDestroyTextureObject(t->dev.tex_lin);
    if (t->dev.ftex_pt) cudaDestroyTextureObject(t->dev.ftex_pt);
    if (t->dev.ftex_lin) cudaDestroyTextureObject(t->dev.ftex_lin);
    if (t->arr) cudaFreeArray(t->arr);
    if (t->arr32) cudaFreeArray(t->arr32);
    if (t->d_lin) cudaFree(t->d_lin);
    if (t->d_f32) cudaFree(t->d_f32);
    if (t->d_coul) cudaFree(t->d_coul);
    if (t->d_fcoul) cudaFree(t->d_fcoul);
    if (t->d_fcoulq) cudaFree(t->d_fcoulq);
    if (t->d_coul3) cudaFree(t->d_coul3);
    if (t->d_q3) cudaFree(t->d_q3);
    if (t->d_o3) cudaFree(t->d_o3);
    for (auto &kv : t->diag_ws) { cudaFree(kv.second.partials); cudaFree(kv.second.ticket); if (kv.second.shell_rep) cudaFree(kv.second.shell_rep); if (kv.second.fixmap) cudaFree(kv.second.fixmap); }
    for (auto &s : t->stages) {
        for (void *b : s.buf) if (b) cudaFree(b);
        if (s.d_diag) cudaFree(s.d_diag);
        if (s.flags) cudaFree(s.flags);
        if (s.s) cudaStreamDestroy(s.s);
    }
    if (t->h_diag_pinned) cudaFreeHost(t->h_diag_pinned);
    if (t->d_shell) cudaFree(t->d_shell);
    delete t;
}

// fills the radial-profile fields of `a` for a launch over cells [off, off + n) and zeroes the replica workspace on `st`
static cool_status prepare_shells(const cool_table *t, cudaStream_t st, LaunchArgs &a, double *d_out, long long shell_cells, long long off, long long n);

static cool_status get_diag_ws(const cool_table *t, cudaStream_t st, DiagWorkspace *out, size_t shell_bytes = 0, size_t fixmap_bytes = 0)
{
    std::lock_guard<std::mutex> lk(t->mu);
    auto it = t->diag_ws.find(st);
    if (it == t->diag_ws.end()) {
        DiagWorkspace w;
        w.capacity_blocks = t->sm_count * 32;
        CUDA_TRY(cudaMalloc(&w.partials, sizeof(double) * 8 * (size_t)w.capacity_blocks), "cudaMalloc(diag partials)");
        cudaError_t e = cudaMalloc(&w.ticket, sizeof(unsigned));
        // zeroed on the stream whose kernels use it (a plain cudaMemset runs on the legacy default stream, which
        // non-blocking streams do not wait for); the kernels leave it at zero again
        if (e == cudaSuccess) e = cudaMemsetAsync(w.ticket, 0, sizeof(unsigned), st);
        if (e != cudaSuccess) {
            set_error("diag ticket: %s", cudaGetErrorString(e));
            cudaFree(w.partials); if (w.ticket) cudaFree(w.ticket);
            return e == cudaErrorMemoryAllocation ? COOL_ENOMEM : COOL_ECUDA;
        }
        it = t->diag_ws.emplace(st, w).first;
    }
    if (fixmap_bytes > it->second.fixmap_cap) {
        CUDA_TRY(cudaStreamSynchronize(st), "cudaStreamSynchronize(precise-pass bitmap)");
        if (it->second.fixmap) cudaFree(it->second.fixmap);
        it->second.fixmap = nullptr; it->second.fixmap_cap = 0;
        CUDA_TRY(cudaMalloc(&it->second.fixmap, fixmap_bytes), "cudaMalloc(precise-pass bitmap)");
        it->second.fixmap_cap = fixmap_bytes;
    }
    if (shell_bytes > it->second.shell_cap) {
        // growing the workspace of a stream that may still be running an earlier launch: wait for it first
        CUDA_TRY(cudaStreamSynchronize(st), "cudaStreamSynchronize(shell workspace)");
        if (it->second.shell_rep) cudaFree(it->second.shell_rep);
        it->second.shell_rep = nullptr; it->second.shell_cap = 0;
        CUDA_TRY(cudaMalloc(&it->second.shell_rep, shell_bytes), "cudaMalloc(shell workspace)");
        it->second.shell_cap = shell_bytes;
    }
    *out = it->second;
    return COOL_OK;
}

static cool_status prepare_shells(const cool_table *t, cudaStream_t st, LaunchArgs &a, double *d_out, long long shell_cells, long long off, long long n)
{
    a.lum_shell = d_out; a.shell_cells = shell_cells; a.cell_offset = off;
    a.shell0 = off / shell_cells;
    const long long nloc = (off + n - 1) / shell_cells - a.shell0 + 1;
    a.shell_nloc4 = (unsigned)(4 * nloc);
    const int nrep = n >= (1ll << 24) ? kShellReplicasLarge : kShellReplicasSmall;
    a.shell_rmask = (unsigned)(nrep - 1);
    const size_t bytes = (size_t)nrep * a.shell_nloc4 * sizeof(double);
    DiagWorkspace w;
    cool_status s = get_diag_ws(t, st, &w, bytes);
    if (s != COOL_OK) return s;
    a.shell_rep = w.shell_rep;
    CUDA_TRY(cudaMemsetAsync(a.shell_rep, 0, bytes, st), "cudaMemsetAsync(shell workspace)");
    return COOL_OK;
}

// work lists of the precise pass (cool_fix.cu): per fp32-kernel warp a count, and per listed tile its index and four 32-bit
// words of cell bits.  Every warp owns ceil(ntiles / warps) slots, so ntiles + warps slots always suffice.
static size_t fixmap_bytes(const cool_table *t, long long ncell)
{
    const size_t ntiles = (size_t)((ncell + 127) / 128), warps = (size_t)t->sm_count * kFixMaxWarpsPerSm;
    return warps * 4 + (ntiles + warps) * 20 + 64;
}

static cool_status check_args(const cool_table *t, const cool_cells *c, const cool_params *p, cool_variant *v, int *coul)
{
    if (!t || !c || !p) { set_error("NULL table, cells or params"); return COOL_EINVAL; }
    if (c->ncell < 0) { set_error("ncell < 0"); return COOL_EINVAL; }
    if (c->dtype != COOL_F32 && c->dtype != COOL_F64) { set_error("unknown dtype"); return COOL_EINVAL; }
    if (c->ncell >= (1ll << 32)) { set_error("ncell must be below 2^32"); return COOL_EINVAL; }
    if (c->ncell > 0 && (!c->rho || !c->bsq || !c->theta_e_in || !c->theta_i_in || !c->theta_e_out || !c->theta_i_out)) {
        set_error("NULL cell array"); return COOL_EINVAL;
    }
    if (c->lum_shell && (c->shell_cells <= 0 || c->shell_cells % 128 != 0)) { set_error("lum_shell needs shell_cells > 0 and a multiple of 128"); return COOL_EINVAL; }
    if (c->lum_shell && (c->ncell / 128 + 1) * (c->shell_cells / 128) >= (1ll << 40)) { set_error("lum_shell: ncell x shell_cells too large"); return COOL_EINVAL; }
    if (!(p->dt > 0.0) || !std::isfinite(p->dt)) { set_error("dt must be finite and > 0"); return COOL_EINVAL; }
    if (p->nsub < 1 || p->nsub > 1024) { set_error("nsub must be in [1, 1024]"); return COOL_EINVAL; }
    if (!(p->f_limit > 0.0 && p->f_limit < 0.5)) { set_error("f_limit must be in (0, 0.5)"); return COOL_EINVAL; }
    if (!(p->h_floor >= 0.0)) { set_error("h_floor must be >= 0"); return COOL_EINVAL; }
    cool_variant vv = p->variant;
    if (vv == COOL_V_AUTO) vv = cool_table_auto_variant(t);
    if (vv < COOL_V_TEX_POINT || vv > COOL_V_ANALYTIC) { set_error("unknown variant"); return COOL_EINVAL; }
    std::string why;
    if (!variant_supported(t, vv, c->dtype, &why)) { set_error("variant unsupported: %s", why.c_str()); return COOL_EUNSUPPORTED; }
    if ((vv == COOL_V_TEX_POINT || vv == COOL_V_TEX_HWFILTER) && !t->dev.tex_pt) { set_error("variant unsupported: table too large for a 3-D texture"); return COOL_EUNSUPPORTED; }
    int cm;
    switch (p->coulomb) {
        case COOL_COULOMB_AUTO: cm = (t->dev.coul || t->dev.coul3) ? 1 : 2; break;
        case COOL_COULOMB_OFF: cm = 0; break;
        case COOL_COULOMB_TABLE:
            if (!t->dev.coul && !t->dev.coul3) { set_error("COOL_COULOMB_TABLE but the table has no Coulomb coefficient table"); return COOL_EINVAL; }
            cm = 1; break;
        case COOL_COULOMB_ANALYTIC: cm = 2; break;
        default: set_error("unknown coulomb mode"); return COOL_EINVAL;
    }
    if (p->scheme != COOL_SCHEME_EXPLICIT && p->scheme != COOL_SCHEME_IMPLICIT) { set_error("unknown scheme"); return COOL_EINVAL; }
    if (p->scheme == COOL_SCHEME_IMPLICIT && desc_is_cgs(&t->desc)) { set_error("variant unsupported: the implicit scheme is not defined on the paper's cgs table"); return COOL_EUNSUPPORTED; }
    if (p->scheme == COOL_SCHEME_IMPLICIT && (vv == COOL_V_TEX_HWFILTER || vv == COOL_V_ANALYTIC)) {
        set_error("variant unsupported: the implicit scheme runs on the GLOBAL, SMEM and TEX_POINT lookups"); return COOL_EUNSUPPORTED;
    }
    *v = vv; *coul = cm;
    return COOL_OK;
}

}  // namespace cool

using namespace cool;

extern "C" const char *cool_last_error(void) { return g_err; }
extern "C" const char *cool_version(void) { return "cool_b200 0.2 (sm_100a)"; }
extern "C" int cool_last_launch_count(void) { return g_launches; }
extern "C" const char *cool_last_kernel_name(void) { return g_kernel; }

extern "C" cool_variant cool_table_auto_variant(const cool_table *t)
{
    if (!t || t->dev.mode == 0) return COOL_V_ANALYTIC;
    if (variant_supported(t, COOL_V_SMEM, COOL_F32, nullptr)) return COOL_V_SMEM;
    return COOL_V_GLOBAL;
}

extern "C" cool_status cool_table_create(const cool_table_desc *desc, int device, cool_table **out)
{
    if (!out) { set_error("cool_table_create: out is NULL"); return COOL_EINVAL; }
    *out = nullptr;
    std::string why;
    if (!desc_valid(desc, desc && (desc->host_coulomb != nullptr || (desc_is_cgs(desc) && desc->host_coulomb3 != nullptr)), &why)) { set_error("cool_table_create: %s", why.c_str()); return COOL_EINVAL; }
    for (int p = 0; p < desc->nproc; ++p)
        if (!desc->host_data[p]) { set_error("cool_table_create: host_data[%d] is NULL", p); return COOL_EINVAL; }
    int ndev = 0;
    CUDA_TRY(cudaGetDeviceCount(&ndev), "cudaGetDeviceCount");
    if (device < 0 || device >= ndev) { set_error("cool_table_create: device %d of %d", device, ndev); return COOL_ECUDA; }
    CUDA_TRY(cudaSetDevice(device), "cudaSetDevice");

    cool_table *t = new (std::nothrow) cool_table();
    if (!t) { set_error("out of host memory"); return COOL_ENOMEM; }
    t->device = device;
    t->desc = *desc;
    t->desc.host_data[0] = t->desc.host_data[1] = t->desc.host_data[2] = nullptr;
    t->desc.host_coulomb = nullptr;
    cudaDeviceProp prop;
    cudaError_t pe = cudaGetDeviceProperties(&prop, device);
    if (pe != cudaSuccess) { set_error("cudaGetDeviceProperties: %s", cudaGetErrorString(pe)); free_table(t); return COOL_ECUDA; }
    t->sm_count = prop.multiProcessorCount;
    t->max_smem_optin = (int)prop.sharedMemPerBlockOptin;

    // unit constants
    DevConst &K = t->cst;
    K.units = to_units(desc->units);
    K.der = coolphys::derive(K.units);
    K.mr = coolphys::kMR; K.ge1 = K.units.gamma_e - 1.0; K.gi1 = K.units.gamma_i - 1.0;
    K.coul_k = K.der.coul_pref_code / K.mr;
    const double t1 = coolphys::kTHETA_TO_K;
    K.bb_k = 4.0 * coolphys::kSIGSB * t1 * t1 * t1 * t1 * K.der.rate_conv;
    K.tausca_k = 2.0 * coolphys::kSIGT * K.der.ne_per_rho;
    K.log2_ue_k = log2(K.mr / K.ge1);

    DevTable &D = t->dev;
    auto fail = [&](cool_status s) { free_table(t); return s; };
    const int nd = desc->ndim;
    if (desc_is_cgs(desc)) {
        // ---- the paper's table (mode 5): kept in the caller's order [H_th][B][n_e][T_e]; the 3-D texture flattens (n_e, T_e)
        // into z and puts (B, H_th) on x, y, which the hardware can filter (L155-L159)
        D.mode = desc->nproc == 0 ? 0 : 5;
        for (int k = 0; k < 4; ++k) D.ax[k] = make_axis(desc->n[k], desc->lo[k], desc->hi[k]);
        const size_t nH = desc->n[0], nB = desc->n[1], nN = desc->n[2], nT = desc->n[3], total = nH * nB * nN * nT;
        if (desc->nproc > 0) {
            const size_t bytes = total * sizeof(float);
            if (bytes > 0xffffffffull) { set_error("table too large"); return fail(COOL_EINVAL); }
            for (size_t f = 0; f < total; ++f)
                if (!std::isfinite(desc->host_data[0][f])) { set_error("cool_table_create: non-finite value in host_data[0]"); return fail(COOL_EINVAL); }
            cudaError_t e = cudaMalloc(&t->d_lin, bytes);
            if (e == cudaSuccess) e = cudaMemcpy(t->d_lin, desc->host_data[0], bytes, cudaMemcpyHostToDevice);
            if (e != cudaSuccess) { set_error("table upload: %s", cudaGetErrorString(e)); return fail(e == cudaErrorMemoryAllocation ? COOL_ENOMEM : COOL_ECUDA); }
            D.lin1 = t->d_lin; D.table_bytes = (unsigned)bytes;
            if (nB <= 16384 && nH <= 16384 && nN * nT <= 16384) {
                std::vector<float> tx;
                try { tx.resize(total); } catch (...) { set_error("out of host memory"); return fail(COOL_ENOMEM); }
                for (size_t ih = 0; ih < nH; ++ih)
                    for (size_t ib = 0; ib < nB; ++ib) {
                        const float *src = desc->host_data[0] + (ih * nB + ib) * nN * nT;
                        for (size_t z = 0; z < nN * nT; ++z) tx[(z * nH + ih) * nB + ib] = src[z];
                    }
                e = make_textures(tx.data(), 1, nB, nH, nN * nT, &t->arr, &D.tex_pt, &D.tex_lin);
                if (e != cudaSuccess) { set_error("texture setup: %s", cudaGetErrorString(e)); return fail(e == cudaErrorMemoryAllocation ? COOL_ENOMEM : COOL_ECUDA); }
            }
        }
        if (desc->host_coulomb3) {
            const size_t n3 = (size_t)desc->nc3[0] * desc->nc3[1] * desc->nc3[2];
            for (size_t k = 0; k < n3; ++k)
                if (!std::isfinite(desc->host_coulomb3[k])) { set_error("cool_table_create: non-finite value in host_coulomb3"); return fail(COOL_EINVAL); }
            cudaError_t e = cudaMalloc(&t->d_coul3, n3 * sizeof(float));
            if (e == cudaSuccess) e = cudaMemcpy(t->d_coul3, desc->host_coulomb3, n3 * sizeof(float), cudaMemcpyHostToDevice);
            if (e != cudaSuccess) { set_error("Coulomb table upload: %s", cudaGetErrorString(e)); return fail(e == cudaErrorMemoryAllocation ? COOL_ENOMEM : COOL_ECUDA); }
            D.coul3 = t->d_coul3;
            for (int k = 0; k < 3; ++k) D.cax3[k] = make_axis(desc->nc3[k], desc->c3lo[k], desc->c3hi[k]);
        }
        t->desc.host_coulomb3 = nullptr;
        *out = t;
        return COOL_OK;
    }
    D.mode = desc->nproc == 0 ? 0 : nd;
    int ncan[4] = {1, 1, 1, 1};
    for (int k = 0; k < nd; ++k) {
        const int slot = canon_slot(desc->axis[k]);
        D.ax[slot] = make_axis(desc->n[k], desc->lo[k], desc->hi[k]);
        ncan[slot] = desc->n[k];
    }
    if (nd == 3) D.ax[CAX_THI] = make_axis(2, 0.0, 1.0);
    D.s_thi = ncan[CAX_BSQ];
    D.s_the = ncan[CAX_THI] * D.s_thi;
    D.s_rho = ncan[CAX_THE] * D.s_the;

    if (desc->nproc > 0) {
        const long long total = (long long)ncan[0] * ncan[1] * ncan[2] * ncan[3];
        const int chan = (nd == 3) ? 1 : 4;
        const size_t bytes = ((size_t)total * chan * sizeof(float) + 15) & ~(size_t)15;
        if (bytes > 0xffffffffull) { set_error("table too large"); return fail(COOL_EINVAL); }
        std::vector<float> canon;
        try { canon.assign(bytes / sizeof(float), 0.f); } catch (...) { set_error("out of host memory"); return fail(COOL_ENOMEM); }
        long long cstride_of_src[4];          // canonical stride (in nodes) for source axis k
        for (int k = 0; k < nd; ++k) {
            const int slot = canon_slot(desc->axis[k]);
            cstride_of_src[k] = slot == CAX_RHO ? D.s_rho : slot == CAX_THE ? D.s_the : slot == CAX_THI ? D.s_thi : 1;
        }
        int idx[4] = {0, 0, 0, 0};
        for (long long f = 0; f < total; ++f) {
            long long coff = 0;
            for (int k = 0; k < nd; ++k) coff += idx[k] * cstride_of_src[k];
            for (int p = 0; p < desc->nproc; ++p) {
                const float v = desc->host_data[p][f];
                if (!std::isfinite(v)) { set_error("cool_table_create: non-finite value in host_data[%d]", p); return fail(COOL_EINVAL); }
                canon[(size_t)coff * chan + p] = v;
            }
            for (int k = nd - 1; k >= 0; --k) { if (++idx[k] < desc->n[k]) break; idx[k] = 0; }
        }
        cudaError_t e = cudaMalloc(&t->d_lin, bytes);
        if (e != cudaSuccess) { set_error("cudaMalloc(table): %s", cudaGetErrorString(e)); return fail(e == cudaErrorMemoryAllocation ? COOL_ENOMEM : COOL_ECUDA); }
        e = cudaMemcpy(t->d_lin, canon.data(), bytes, cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { set_error("cudaMemcpy(table): %s", cudaGetErrorString(e)); return fail(COOL_ECUDA); }
        D.table_bytes = (unsigned)bytes;
        if (nd == 3) D.lin1 = t->d_lin; else D.lin4 = (const float4 *)t->d_lin;

        // fp32-path copy: log2 of the rate per unit electron energy at the node (see cool_internal.h)
        auto same = [](const AxisCoef &x, const AxisCoef &y) { return x.n == y.n && x.lo10 == y.lo10 && x.inv10 == y.inv10; };
        AxisCoef c0{}, c1{};
        if (desc->host_coulomb) { c0 = make_axis(desc->nc[0], desc->clo[0], desc->chi[0]); c1 = make_axis(desc->nc[1], desc->clo[1], desc->chi[1]); }
        D.f4_has_coul = nd == 4 && desc->host_coulomb && same(c0, D.ax[CAX_THI]) && same(c1, D.ax[CAX_THE]);
        std::vector<float> canon32;
        try { canon32.assign(bytes / sizeof(float), 0.f); } catch (...) { set_error("out of host memory"); return fail(COOL_ENOMEM); }
        {
            const double L10 = 3.321928094887362, lue = log2(K.mr / K.ge1);
            const AxisCoef &ar = D.ax[CAX_RHO], &ae = D.ax[CAX_THE];
            const int nr = ncan[CAX_RHO], ne = ncan[CAX_THE], ni = ncan[CAX_THI], nb = ncan[CAX_BSQ];
            for (int ir = 0; ir < nr; ++ir)
                for (int ie = 0; ie < ne; ++ie) {
                    // log2(u_e / (rho Theta_e)) + log2 rho_node + log2 Theta_e_node
                    const double sub = lue + L10 * ((ar.lo10 + ir / ar.inv10) + (ae.lo10 + ie / ae.inv10));
                    for (int ii = 0; ii < ni; ++ii)
                        for (int ib = 0; ib < nb; ++ib) {
                            const size_t o = ((((size_t)ir * ne + ie) * ni + ii) * nb + ib) * chan;
                            if (nd == 3) canon32[o] = (float)(L10 * (double)canon[o] - sub);
                            else {
                                canon32[o + 0] = (float)(L10 * (double)canon[o + 0] - sub);
                                canon32[o + 1] = (float)(L10 * (double)canon[o + 1] - sub);
                                canon32[o + 2] = (float)(L10 * (double)canon[o + 2]);
                                canon32[o + 3] = D.f4_has_coul ? (float)(L10 * (double)desc->host_coulomb[(size_t)ii * desc->nc[1] + ie]) : 0.f;
                            }
                        }
                }
        }
        // Steep intervals of the fp32 tables (cool_internal.h, cool_fix.cu): along Theta_e they become bands whose cells the
        // precise pass recomputes; a steep interval along any other axis sends every cell there (not seen in the paper's tables).
        {
            double steep = kSteepLog2;
            if (const char *ev = getenv("COOL_STEEP_LOG2")) steep = atof(ev);          // experiments; <= 0 switches the pass off
            const int nr = ncan[CAX_RHO], ne = ncan[CAX_THE], ni = ncan[CAX_THI], nb = ncan[CAX_BSQ];
            std::vector<double> de(ne > 1 ? ne - 1 : 0, 0.0);
            double dother = 0.0;
            const size_t sb = chan, si = (size_t)nb * chan, se = (size_t)ni * si, sr = (size_t)ne * se;
            // What counts is the sensitivity of the TOTAL rate to a coordinate error.  nproc = 3: Q_thin = Q_brem + eta Q_syn, so
            // a channel's node-to-node step is weighted by its share of Q_thin (a synchrotron table that falls by 100 log2
            // units where bremsstrahlung dominates a million-fold is harmless); the shares are monotone between two nodes
            // (the ratio of two log-linear interpolants), so the larger of the two end-point values bounds the interval.
            auto step = [&](size_t o, size_t o2) {
                if (nd == 3) return std::fabs((double)canon32[o2] - (double)canon32[o]);
                const double d0 = std::fabs((double)canon32[o2] - (double)canon32[o]);
                const double d1 = std::fabs(((double)canon32[o2 + 1] + (double)canon32[o2 + 2]) - ((double)canon32[o + 1] + (double)canon32[o + 2]));
                double m = 0.0;
                for (size_t q : {o, o2}) {
                    const double ssy = 1.0 / (1.0 + exp2((double)canon32[q] - ((double)canon32[q + 1] + (double)canon32[q + 2])));
                    m = std::max(m, (1.0 - ssy) * d0 + ssy * d1);
                }
                return m;
            };
            for (int ir = 0; ir < nr; ++ir)
                for (int ie = 0; ie < ne; ++ie)
                    for (int ii = 0; ii < ni; ++ii)
                        for (int ib = 0; ib < nb; ++ib) {
                            const size_t o = ir * sr + ie * se + ii * si + ib * sb;
                            if (ie + 1 < ne) de[ie] = std::max(de[ie], step(o, o + se));
                            if (ir + 1 < nr) dother = std::max(dother, step(o, o + sr));
                            if (ii + 1 < ni) dother = std::max(dother, step(o, o + si));
                            if (ib + 1 < nb) dother = std::max(dother, step(o, o + sb));
                        }
            D.nband = 0;
            if (steep > 0.0) {
                int first = -1, last = -1;                            // first and last steep interval: one band covers them all (over-marking is safe)
                D.band_step = 0.f;
                for (int ie = 0; ie + 1 < ne; ++ie)
                    if (de[ie] > steep) { if (first < 0) first = ie; last = ie; D.band_step = std::max(D.band_step, (float)de[ie]); }
                const AxisCoef &axe = D.ax[CAX_THE];
                auto node_theta = [&](double tnode) { return pow(10.0, axe.lo10 + tnode / axe.inv10); };
                D.band_k0 = first; D.band_k1 = last;
                if (dother > steep) {                                 // every positive Theta_e is inside the band
                    D.nband = 1; D.band_lo = 0.f; D.band_hi = INFINITY;
                    D.band_step = std::max(D.band_step, (float)dother);
                    D.band_k0 = 0; D.band_k1 = ne - 2;
                } else if (first >= 0) {
                    D.nband = 1;
                    D.band_lo = (float)node_theta(first - kBandMargin);
                    D.band_hi = (float)node_theta(last + 1 + kBandMargin);
                }
            }
        }
        e = cudaMalloc(&t->d_f32, bytes);
        if (e == cudaSuccess) e = cudaMemcpy(t->d_f32, canon32.data(), bytes, cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { set_error("fp32 table upload: %s", cudaGetErrorString(e)); return fail(e == cudaErrorMemoryAllocation ? COOL_ENOMEM : COOL_ECUDA); }
        if (nd == 3) D.f1 = t->d_f32; else D.f4 = (const float4 *)t->d_f32;

        // MODE 3 quad layout (4x the bytes): one float4 holds the four (Theta_e, bsq) corners of a table cell.
        // Built while it stays L2-resident (default limit 64 MiB; COOL_QUAD_MAX_MB overrides, 0 disables).
        if (nd == 3) {
            size_t quad_max = (size_t)64 << 20;
            if (const char *ev = getenv("COOL_QUAD_MAX_MB")) quad_max = (size_t)atoll(ev) << 20;
            const size_t qbytes = (size_t)total * 4 * sizeof(float);
            if (qbytes <= quad_max) {
                std::vector<float> quad;
                try { quad.resize((size_t)total * 4); } catch (...) { set_error("out of host memory"); return fail(COOL_ENOMEM); }
                const int nr = ncan[CAX_RHO], ne = ncan[CAX_THE], nb = ncan[CAX_BSQ];
                for (int ir = 0; ir < nr; ++ir)
                    for (int ie = 0; ie < ne; ++ie) {
                        const int ie1 = std::min(ie + 1, ne - 1);
                        const float *row0 = &canon32[((size_t)ir * ne + ie) * nb], *row1 = &canon32[((size_t)ir * ne + ie1) * nb];
                        float *q = &quad[((size_t)ir * ne + ie) * nb * 4];
                        for (int ib = 0; ib < nb; ++ib) {
                            const int ib1 = std::min(ib + 1, nb - 1);
                            q[4 * ib + 0] = row0[ib]; q[4 * ib + 1] = row0[ib1]; q[4 * ib + 2] = row1[ib]; q[4 * ib + 3] = row1[ib1];
                        }
                    }
                e = cudaMalloc(&t->d_q3, qbytes);
                if (e == cudaSuccess) e = cudaMemcpy(t->d_q3, quad.data(), qbytes, cudaMemcpyHostToDevice);
                if (e != cudaSuccess) { set_error("quad table upload: %s", cudaGetErrorString(e)); return fail(e == cudaErrorMemoryAllocation ? COOL_ENOMEM : COOL_ECUDA); }
                D.q3 = (const float4 *)t->d_q3;
            }
            // oct layout (8x the bytes): all eight corners of a table cell in one 32-byte sector, one 256-bit gather per
            // lookup.  Wins while it sits comfortably in L2 (64^3: 8 MiB, 0.61 -> 0.40 ms on 2^26 log-uniform cells); at 128^3
            // (64 MiB) it ties with the quads and costs L1 when the diagnostics shrink it, so the default limit is 16 MiB
            // (COOL_OCT_MAX_MB overrides, 0 disables).
            size_t oct_max = (size_t)16 << 20;
            if (const char *ev = getenv("COOL_OCT_MAX_MB")) oct_max = (size_t)atoll(ev) << 20;
            const size_t obytes = (size_t)total * 8 * sizeof(float);
            if (obytes <= oct_max) {
                std::vector<float> oct;
                try { oct.resize((size_t)total * 8); } catch (...) { set_error("out of host memory"); return fail(COOL_ENOMEM); }
                const int nr = ncan[CAX_RHO], ne = ncan[CAX_THE], nb = ncan[CAX_BSQ];
                for (int ir = 0; ir < nr; ++ir)
                    for (int ie = 0; ie < ne; ++ie)
                        for (int ib = 0; ib < nb; ++ib) {
                            float *o = &oct[((((size_t)ir * ne + ie) * nb) + ib) * 8];
                            for (int c = 0; c < 8; ++c) {
                                const int jr = std::min(ir + (c >> 2), nr - 1), je = std::min(ie + ((c >> 1) & 1), ne - 1), jb = std::min(ib + (c & 1), nb - 1);
                                o[c] = canon32[((size_t)jr * ne + je) * nb + jb];
                            }
                        }
                e = cudaMalloc(&t->d_o3, obytes);
                if (e == cudaSuccess) e = cudaMemcpy(t->d_o3, oct.data(), obytes, cudaMemcpyHostToDevice);
                if (e != cudaSuccess) { set_error("oct table upload: %s", cudaGetErrorString(e)); return fail(e == cudaErrorMemoryAllocation ? COOL_ENOMEM : COOL_ECUDA); }
                D.o3 = (const float4 *)t->d_o3;
            }
        }

        // cudaArray + texture objects (x = bsq, y = theta_e | theta_i, z = rho | rho*n_the + i_the)
        const size_t ex = ncan[CAX_BSQ];
        const size_t ey = nd == 3 ? ncan[CAX_THE] : ncan[CAX_THI];
        const size_t ez = nd == 3 ? ncan[CAX_RHO] : (size_t)ncan[CAX_RHO] * ncan[CAX_THE];
        if (ex <= 16384 && ey <= 16384 && ez <= 16384) {
            e = make_textures(canon.data(), chan, ex, ey, ez, &t->arr, &D.tex_pt, &D.tex_lin);
            if (e == cudaSuccess) e = make_textures(canon32.data(), chan, ex, ey, ez, &t->arr32, &D.ftex_pt, &D.ftex_lin);
            if (e != cudaSuccess) { set_error("texture setup: %s", cudaGetErrorString(e)); return fail(e == cudaErrorMemoryAllocation ? COOL_ENOMEM : COOL_ECUDA); }
        }
    }
    if (desc->host_coulomb) {
        const size_t n = (size_t)desc->nc[0] * desc->nc[1];
        for (size_t k = 0; k < n; ++k)
            if (!std::isfinite(desc->host_coulomb[k])) { set_error("cool_table_create: non-finite value in host_coulomb"); return fail(COOL_EINVAL); }
        cudaError_t e = cudaMalloc(&t->d_coul, n * sizeof(float));
        if (e == cudaSuccess) e = cudaMemcpy(t->d_coul, desc->host_coulomb, n * sizeof(float), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { set_error("Coulomb table upload: %s", cudaGetErrorString(e)); return fail(e == cudaErrorMemoryAllocation ? COOL_ENOMEM : COOL_ECUDA); }
        D.coul = t->d_coul;
        {   // fp32 path: log2 C, plain (padded to 16 B) and as quads {C(i,e), C(i,e+1), C(i+1,e), C(i+1,e+1)}
            const size_t npad = (n + 3) & ~(size_t)3;
            const int n0 = desc->nc[0], n1 = desc->nc[1];
            const int qs = n1 + COOL_COULQ_SKEW;                 // quad row stride
            std::vector<float> c2(npad, 0.f), cq((size_t)n0 * qs * 4, 0.f);
            for (size_t k = 0; k < n; ++k) c2[k] = (float)(3.321928094887362 * (double)desc->host_coulomb[k]);
            for (int i = 0; i < n0; ++i)
                for (int j = 0; j < n1; ++j) {
                    const int i1 = std::min(i + 1, n0 - 1), j1 = std::min(j + 1, n1 - 1);
                    float *q = &cq[((size_t)i * qs + j) * 4];
                    q[0] = c2[(size_t)i * n1 + j]; q[1] = c2[(size_t)i * n1 + j1]; q[2] = c2[(size_t)i1 * n1 + j]; q[3] = c2[(size_t)i1 * n1 + j1];
                }
            e = cudaMalloc(&t->d_fcoul, npad * sizeof(float));
            if (e == cudaSuccess) e = cudaMemcpy(t->d_fcoul, c2.data(), npad * sizeof(float), cudaMemcpyHostToDevice);
            if (e == cudaSuccess) e = cudaMalloc(&t->d_fcoulq, cq.size() * sizeof(float));
            if (e == cudaSuccess) e = cudaMemcpy(t->d_fcoulq, cq.data(), cq.size() * sizeof(float), cudaMemcpyHostToDevice);
            if (e != cudaSuccess) { set_error("Coulomb table upload: %s", cudaGetErrorString(e)); return fail(e == cudaErrorMemoryAllocation ? COOL_ENOMEM : COOL_ECUDA); }
            D.fcoul = t->d_fcoul;
            D.fcoulq = (const float4 *)t->d_fcoulq;
            D.coulq_bytes = (int)(cq.size() * sizeof(float));
            D.coulq_stride = qs;
        }
        D.cax[0] = make_axis(desc->nc[0], desc->clo[0], desc->chi[0]);
        D.cax[1] = make_axis(desc->nc[1], desc->clo[1], desc->chi[1]);
        D.coul_bytes = (int)(n * sizeof(float));
        auto same = [](const AxisCoef &x, const AxisCoef &y) { return x.n == y.n && x.lo10 == y.lo10 && x.inv10 == y.inv10; };
        D.coul_share_the = D.mode != 0 && same(D.cax[1], D.ax[CAX_THE]);
        D.coul_share_thi = D.mode == 4 && same(D.cax[0], D.ax[CAX_THI]);
    }
    *out = t;
    return COOL_OK;
}

extern "C" cool_status cool_table_destroy(cool_table *t)
{
    if (!t) return COOL_OK;
    free_table(t);
    return COOL_OK;
}

extern "C" cool_status cool_apply(const cool_table *t, const cool_cells *c, const cool_params *p, cool_diag *d_diag, void *stream)
{
    g_launches = 0;
    cool_variant v; int coul;
    cool_status s = check_args(t, c, p, &v, &coul);
    if (s != COOL_OK) return s;
    DeviceGuard dg;
    CUDA_TRY(dg.enter(t->device), "cudaSetDevice");
    cudaStream_t st = (cudaStream_t)stream;
    LaunchArgs a{};
    a.ncell = c->ncell; a.rho = c->rho; a.bsq = c->bsq; a.the_in = c->theta_e_in; a.thi_in = c->theta_i_in;
    a.r = c->r; a.vol = c->vol; a.the_out = c->theta_e_out; a.thi_out = c->theta_i_out;
    a.dt = p->dt; a.nsub = p->nsub; a.f_limit = p->f_limit; a.h_floor = p->h_floor; a.coulomb = coul; a.scheme = p->scheme;
    a.want_diag = d_diag != nullptr; a.d_diag = d_diag;
    if (c->flags && !d_diag) { set_error("flags needs d_diag"); return COOL_EINVAL; }
    a.flags = c->flags;
    if (c->ncell > 0 && uses_fixmap(t, v, c->dtype, a)) {
        DiagWorkspace w;
        s = get_diag_ws(t, st, &w, 0, fixmap_bytes(t, c->ncell));
        if (s != COOL_OK) return s;
        a.fixmap = w.fixmap; a.partials = w.partials; a.ticket = w.ticket;
    }
    if (c->lum_shell) {
        if (!d_diag) { set_error("lum_shell needs d_diag"); return COOL_EINVAL; }
        const long long nshell = (c->ncell + c->shell_cells - 1) / c->shell_cells;
        if (nshell > 0) CUDA_TRY(cudaMemsetAsync(c->lum_shell, 0, (size_t)nshell * 4 * sizeof(double), st), "cudaMemsetAsync(lum_shell)");
        if (c->ncell > 0) {
            s = prepare_shells(t, st, a, c->lum_shell, c->shell_cells, 0, c->ncell);
            if (s != COOL_OK) return s;
        }
    }
    if (d_diag) {
        DiagWorkspace w;
        s = get_diag_ws(t, st, &w);
        if (s != COOL_OK) return s;
        a.partials = w.partials; a.ticket = w.ticket;
    }
    if (c->ncell == 0) {
        if (d_diag) CUDA_TRY(cudaMemsetAsync(d_diag, 0, sizeof(cool_diag), st), "cudaMemsetAsync(diag)");
        return COOL_OK;
    }
    return launch_step(t, v, c->dtype, a, st, &g_launches);
}

// ------------------------------------------------------------------------------------------
// cool_apply_noalloc (include/cool.h): the step with its scratch in a file-scope device array instead of the per-stream
// workspace get_diag_ws() allocates.  Layout: [0, 256) the ticket | per-block partial sums | precise-pass lists.
// In host code `g_noalloc_scratch` is only a stand-in for the symbol: its device address comes from cudaGetSymbolAddress,
// once per device, with that device current.
// ------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_noalloc_scratch[COOL_NOALLOC_SCRATCH_BYTES];

namespace cool {
constexpr int kNoAllocMaxDevices = 64;
static std::mutex g_noalloc_mu;
static unsigned char *g_noalloc_ptr[kNoAllocMaxDevices] = {};

// device address of the scratch array on the CURRENT device (`device`)
static cool_status noalloc_scratch(int device, unsigned char **out)
{
    if (device < 0 || device >= kNoAllocMaxDevices) { set_error("cool_apply_noalloc: device index %d out of range", device); return COOL_EINVAL; }
    std::lock_guard<std::mutex> lk(g_noalloc_mu);
    if (!g_noalloc_ptr[device]) {
        void *ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
        if (e != cudaSuccess || !ptr) { set_error("cudaGetSymbolAddress(no-alloc scratch): %s", cudaGetErrorString(e)); return COOL_ECUDA; }
        g_noalloc_ptr[device] = (unsigned char *)ptr;
    }
    *out = g_noalloc_ptr[device];
    return COOL_OK;
}
}  // namespace cool

extern "C" cool_status cool_apply_noalloc(const cool_table *t, const cool_cells *c, const cool_params *p, cool_diag *d_diag, void *stream)
{
    g_launches = 0;
    cool_variant v; int coul;
    cool_status s = check_args(t, c, p, &v, &coul);
    if (s != COOL_OK) return s;
    if (c->ncell > COOL_NOALLOC_MAX_CELLS) {
        set_error("cool_apply_noalloc: ncell = %lld exceeds COOL_NOALLOC_MAX_CELLS = %lld (split the batch or use cool_apply)", c->ncell, (long long)COOL_NOALLOC_MAX_CELLS);
        return COOL_EINVAL;
    }
    if (c->lum_shell) { set_error("cool_apply_noalloc: the radial profile (lum_shell) needs a workspace that grows with the shells; use cool_apply"); return COOL_EUNSUPPORTED; }
    if (c->flags && !d_diag) { set_error("flags needs d_diag"); return COOL_EINVAL; }
    DeviceGuard dg;
    CUDA_TRY(dg.enter(t->device), "cudaSetDevice");
    unsigned char *scratch = nullptr;
    s = noalloc_scratch(t->device, &scratch);
    if (s != COOL_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    LaunchArgs a{};
    a.ncell = c->ncell; a.rho = c->rho; a.bsq = c->bsq; a.the_in = c->theta_e_in; a.thi_in = c->theta_i_in;
    a.r = c->r; a.vol = c->vol; a.the_out = c->theta_e_out; a.thi_out = c->theta_i_out;
    a.dt = p->dt; a.nsub = p->nsub; a.f_limit = p->f_limit; a.h_floor = p->h_floor; a.coulomb = coul; a.scheme = p->scheme;
    a.want_diag = d_diag != nullptr; a.d_diag = d_diag;
    a.flags = c->flags;
    if (c->ncell == 0) {
        if (d_diag) CUDA_TRY(cudaMemsetAsync(d_diag, 0, sizeof(cool_diag), st), "cudaMemsetAsync(diag)");
        return COOL_OK;
    }
    const bool fix = uses_fixmap(t, v, c->dtype, a);
    const size_t part_off = 256, part_bytes = sizeof(double) * 8 * (size_t)t->sm_count * 32;      // as get_diag_ws sizes them
    const size_t fix_off = (part_off + part_bytes + 255) & ~(size_t)255;
    const size_t need = fix_off + (fix ? fixmap_bytes(t, c->ncell) : 0);
    if (need > (size_t)COOL_NOALLOC_SCRATCH_BYTES) {
        set_error("cool_apply_noalloc: this launch needs %zu bytes of scratch, the static array holds %u", need, (unsigned)COOL_NOALLOC_SCRATCH_BYTES);
        return COOL_EINVAL;
    }
    if (d_diag || fix) {
        a.ticket = (unsigned *)scratch; a.partials = (double *)(scratch + part_off);
        // the array keeps the last call's contents: the ticket must start at zero (the kernels leave it at zero, but a
        // launch that failed half way would not have)
        CUDA_TRY(cudaMemsetAsync(a.ticket, 0, sizeof(unsigned), st), "cudaMemsetAsync(no-alloc ticket)");
    }
    if (fix) a.fixmap = (unsigned *)(scratch + fix_off);       // every list counter is written by every launch: nothing to clear
    return launch_step(t, v, c->dtype, a, st, &g_launches);
}

extern "C" cool_status cool_apply_host(const cool_table *t, const cool_cells *c, const cool_params *p, cool_diag *h_diag)
{
    g_launches = 0;
    cool_variant v; int coul;
    cool_status s = check_args(t, c, p, &v, &coul);
    if (s != COOL_OK) return s;
    DeviceGuard dg;
    CUDA_TRY(dg.enter(t->device), "cudaSetDevice");
    if (h_diag) memset(h_diag, 0, sizeof *h_diag);
    if (c->lum_shell && !h_diag) { set_error("lum_shell needs h_diag"); return COOL_EINVAL; }
    if (c->flags && !h_diag) { set_error("flags needs h_diag"); return COOL_EINVAL; }
    if (c->ncell == 0) return COOL_OK;

    std::lock_guard<std::mutex> lk_host(t->host_mu);
    const size_t es = c->dtype == COOL_F32 ? 4 : 8;
    const int NST = 3;
    size_t chunk = (size_t)1 << 22;                               // cells per staged chunk
    if ((size_t)c->ncell < chunk) chunk = ((size_t)c->ncell + 3) & ~(size_t)3;
    const size_t need_bytes = chunk * es;
    if (t->stages.empty()) {
        t->stages.resize(NST);
        for (auto &sg : t->stages) {
            CUDA_TRY(cudaStreamCreateWithFlags(&sg.s, cudaStreamNonBlocking), "cudaStreamCreate");
            CUDA_TRY(cudaMalloc(&sg.d_diag, sizeof(cool_diag)), "cudaMalloc(stage diag)");
        }
    }
    if (t->stage_bytes < need_bytes) {
        for (auto &sg : t->stages) {
            CUDA_TRY(cudaStreamSynchronize(sg.s), "cudaStreamSynchronize");
            for (void *&b : sg.buf) {
                if (b) { cudaFree(b); b = nullptr; }
                CUDA_TRY(cudaMalloc(&b, need_bytes), "cudaMalloc(stage buffer)");
            }
            if (sg.flags) { cudaFree(sg.flags); sg.flags = nullptr; }
            CUDA_TRY(cudaMalloc(&sg.flags, chunk), "cudaMalloc(stage flags)");
        }
        t->stage_bytes = need_bytes;
    }
    // a failure inside the chunk loop must not return while copies into the caller's buffers are still in flight
    auto fail_sync = [&](cool_status st_) { for (auto &sg : t->stages) cudaStreamSynchronize(sg.s); return st_; };
#define CUDA_TRY_SYNC(call, what)                                                       \
    do {                                                                                \
        cudaError_t e_ = (call);                                                        \
        if (e_ != cudaSuccess) {                                                        \
            set_error("%s: %s", what, cudaGetErrorString(e_));                          \
            return fail_sync(e_ == cudaErrorMemoryAllocation ? COOL_ENOMEM : COOL_ECUDA); \
        }                                                                               \
    } while (0)
    const size_t nchunks = ((size_t)c->ncell + chunk - 1) / chunk;
    if (h_diag && t->h_diag_cap < nchunks) {
        if (t->h_diag_pinned) cudaFreeHost(t->h_diag_pinned);
        t->h_diag_pinned = nullptr; t->h_diag_cap = 0;
        CUDA_TRY(cudaMallocHost(&t->h_diag_pinned, nchunks * sizeof(cool_diag)), "cudaMallocHost(diag)");
        t->h_diag_cap = nchunks;
    }
    const void *src[6] = {c->rho, c->bsq, c->theta_e_in, c->theta_i_in, c->r, c->vol};
    const size_t shell_bytes = c->lum_shell ? (size_t)((c->ncell + c->shell_cells - 1) / c->shell_cells) * 4 * sizeof(double) : 0;
    if (shell_bytes > t->d_shell_cap) {
        if (t->d_shell) cudaFree(t->d_shell);
        t->d_shell = nullptr; t->d_shell_cap = 0;
        CUDA_TRY(cudaMalloc(&t->d_shell, shell_bytes), "cudaMalloc(shell sums)");
        t->d_shell_cap = shell_bytes;
    }
    if (shell_bytes) {
        // zeroed on stage stream 0 and waited for: every stage stream (non-blocking: they do not wait for the legacy default
        // stream a plain cudaMemset would run on) adds into these sums
        CUDA_TRY(cudaMemsetAsync(t->d_shell, 0, shell_bytes, t->stages[0].s), "cudaMemsetAsync(shell sums)");
        CUDA_TRY(cudaStreamSynchronize(t->stages[0].s), "cudaStreamSynchronize(shell sums)");
    }
    int nl = 0;
    for (size_t k = 0; k < nchunks; ++k) {
        auto &sg = t->stages[k % NST];
        const size_t off = k * chunk;
        const size_t n = std::min(chunk, (size_t)c->ncell - off);
        for (int j = 0; j < 6; ++j)
            if (src[j]) CUDA_TRY_SYNC(cudaMemcpyAsync(sg.buf[j], (const char *)src[j] + off * es, n * es, cudaMemcpyHostToDevice, sg.s), "cudaMemcpyAsync(H2D)");
        LaunchArgs a{};
        a.ncell = (long long)n; a.rho = sg.buf[0]; a.bsq = sg.buf[1]; a.the_in = sg.buf[2]; a.thi_in = sg.buf[3];
        a.r = c->r ? sg.buf[4] : nullptr; a.vol = c->vol ? sg.buf[5] : nullptr;
        a.the_out = sg.buf[6]; a.thi_out = sg.buf[7];
        a.dt = p->dt; a.nsub = p->nsub; a.f_limit = p->f_limit; a.h_floor = p->h_floor; a.coulomb = coul; a.scheme = p->scheme;
        a.want_diag = h_diag != nullptr; a.d_diag = h_diag ? sg.d_diag : nullptr;
        a.flags = c->flags ? sg.flags : nullptr;
        if (shell_bytes) {
            s = prepare_shells(t, sg.s, a, t->d_shell, c->shell_cells, (long long)off, (long long)n);
            if (s != COOL_OK) return fail_sync(s);
        }
        const bool fix = uses_fixmap(t, v, c->dtype, a);
        if (h_diag || fix) {
            DiagWorkspace w;
            s = get_diag_ws(t, sg.s, &w, 0, fix ? fixmap_bytes(t, (long long)n) : 0);
            if (s != COOL_OK) return fail_sync(s);
            a.partials = w.partials; a.ticket = w.ticket; a.fixmap = fix ? w.fixmap : nullptr;
            if (shell_bytes) a.shell_rep = w.shell_rep;
        }
        s = launch_step(t, v, c->dtype, a, sg.s, &nl);
        if (s != COOL_OK) return fail_sync(s);
        CUDA_TRY_SYNC(cudaMemcpyAsync((char *)c->theta_e_out + off * es, sg.buf[6], n * es, cudaMemcpyDeviceToHost, sg.s), "cudaMemcpyAsync(D2H)");
        CUDA_TRY_SYNC(cudaMemcpyAsync((char *)c->theta_i_out + off * es, sg.buf[7], n * es, cudaMemcpyDeviceToHost, sg.s), "cudaMemcpyAsync(D2H)");
        if (c->flags) CUDA_TRY_SYNC(cudaMemcpyAsync(c->flags + off, sg.flags, n, cudaMemcpyDeviceToHost, sg.s), "cudaMemcpyAsync(flags)");
        if (h_diag) CUDA_TRY_SYNC(cudaMemcpyAsync(&t->h_diag_pinned[k], sg.d_diag, sizeof(cool_diag), cudaMemcpyDeviceToHost, sg.s), "cudaMemcpyAsync(diag)");
    }
#undef CUDA_TRY_SYNC
    for (auto &sg : t->stages) CUDA_TRY(cudaStreamSynchronize(sg.s), "cudaStreamSynchronize");
    if (shell_bytes) CUDA_TRY(cudaMemcpy(c->lum_shell, t->d_shell, shell_bytes, cudaMemcpyDeviceToHost), "cudaMemcpy(shell sums)");
    g_launches = nl;
    if (h_diag)
        for (size_t k = 0; k < nchunks; ++k) {
            const cool_diag &d = t->h_diag_pinned[k];
            h_diag->lum_total += d.lum_total; h_diag->lum_brems += d.lum_brems; h_diag->lum_synch += d.lum_synch;
            h_diag->lum_compton += d.lum_compton; h_diag->n_limited += d.n_limited; h_diag->n_floored += d.n_floored;
            h_diag->n_clamped += d.n_clamped;
        }
    return COOL_OK;
}
