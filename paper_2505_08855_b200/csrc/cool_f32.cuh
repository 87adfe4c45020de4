// cool_f32.cuh — the fp32 kernels of the cooling step (include/cool.h), written for sm_100a.
//
// Structure of one launch (one persistent CTA per SM; every WARP runs its own pipeline):
//   * a warp tile = 128 consecutive cells (4 per lane).  The cell arrays of a tile (rho, bsq,
//     Theta_e, Theta_i [, vol, r]) are staged into the warp's own shared-memory stages by 1-D TMA
//     bulk copies (cp.async.bulk + one mbarrier per stage, NST stages deep), so HBM latency never
//     sits on a warp's scoreboard and no CTA-wide barrier exists after the prologue; outputs leave
//     as 128-bit streaming stores;
//   * the table is read through one of five lookup policies: L1/L2-resident global gathers from
//     the plain layout or from the quad layout (one float4 = the four (Theta_e, bsq) corners of a
//     table cell: 2 LDG.128 instead of 8 LDG.32 per trilinear lookup, 2 instead of up to 8 sectors
//     per cell from L2), shared-memory image, point texture, hardware-filtered texture;
//   * the Coulomb coefficient table sits in shared memory, in the same quad layout (1 LDS.128);
//   * the luminosity diagnostic is reduced warp -> block -> fixed-order last-block pass.
// The step is a gather plus scalar arithmetic: no tensor cores.  On B200 it
// is bound by the L1 data pipe and instruction issue, not by HBM, so the code is written to
// minimise L1 wavefronts and instructions:
//   * the table nodes are stored as T' = log2(rate / u_e at the node) (cool_internal.h), so that
//     Lambda h / u_e = 2^(interp(T') + log2 h + clamp correction): no large-number cancellation, no
//     compensated products;
//   * log2 of a primitive is (exponent, log2 mantissa) folded straight into the node coordinate;
//   * floor() is a round-down add of 1.5*2^23 whose mantissa bits are the node index, and the
//     bias is folded into the address constant (no F2I/I2F, no masking);
//   * the Coulomb table's coordinates are an affine map of the table's own node coordinates
//     (one FMA instead of a second logarithm);
//   * MODE 4: the (rho, bsq) contraction of the 16 corners is loop invariant over sub-steps, so a
//     bilinear patch in (w_e, w_i) is cached per visited (i_e, i_i) table cell — 3 FMAs per channel
//     per sub-step — and the Coulomb coefficient rides in the 4th texel channel;
//   * a sub-step that leaves both temperatures bit-identical repeats itself: exact early exit.
#pragma once
#include <cstdlib>
#include "cool_kernels.cuh"

namespace cool {

// Per-launch constants of the fp32 path (host fp64 -> rounded once).
struct F32Const {
    float k0;                         // log2(h)
    float f_limit, mr, eq_frac, gi1_over_ge1, coul_kh, cap1e, cap1i;
    float ae, ai, be, bi;             // c_s^2 = (ae Th_e + ai Th_i)/(1 + be Th_e + bi Th_i)           (eq 14)
    float inv_kB;                     // tau_abs = r_thin * inv_kB rho c_s / Theta_e^3                  (eq 12 in ratio form)
    float ksca;                       // tau_sca = ksca rho c_s
    float hfloor2, spin;              // floor: (pi/2) h_floor^2 (Omega_K r)^2                          (eq 19)
    double lum_k;                     // lum = sum(dTheta_rad rho vol) * lum_k
    double ion_ratio;                 // theta_i of eq 15 = Theta_i / ion_ratio (analytic Coulomb only)
    float cme_s, cme_o, cmi_s, cmi_o; // Coulomb-table node coordinate = table node coordinate * s + o (Theta_e; Theta_i in MODE 4)
    int nsub, coulomb, has_r, has_vol, use_tma, coul_smem, nf;
    unsigned wstage_bytes;            // bytes of one warp stage = nf * 512
    unsigned stage_off, coul_off, table_off;       // dynamic shared memory layout
    // radial profile (eq 25): shell = (tile_offset + warp tile)/shell_tiles; sums go to replica (warp index & shell_rmask) of lum_shell
    // (this launch's workspace, local shell index), shell_reduce_kernel then adds the replicas into the caller's array
    double *lum_shell; unsigned shell_tiles, tile_offset, shell0, shell_nloc4, shell_rmask;
    unsigned long long shell_magic;                          // ceil(2^40 / shell_tiles): (t * magic) >> 40 == t / shell_tiles for t * shell_tiles < 2^40
    // precise pass (cool_fix.cu): a cell goes there when band_lo < Theta_e < band_hi (the table's steep band, DevTable) at the
    // start of a sub-step in which fix_rmin < h Lambda/u_e < fix_rmax (cool_internal.h).  Both windows are tested on the bit
    // patterns (positive floats order like their bits): bits(x) - lo_bits < width as unsigned, false for negative, zero and
    // NaN x; width 0 = empty (no precise pass).  Such a cell is treated like a cell with rho <= 0 here (passed through,
    // neither summed nor counted) and its tile is listed for the precise pass (cool_internal.h, fix_layout).
    unsigned band_lo_bits, band_w, rmin_bits, r_w;
    unsigned *fixmap;                 // NULL: no precise pass
    FixLists fix;
};

// ------------------------------------------------------------------------------------------
// mbarrier / TMA 1-D bulk copy
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_1d(unsigned dst, const void *src, unsigned bytes, unsigned bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile("{\n\t.reg .pred p;\n"
                 "COOL_WAIT:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@p bra COOL_DONE;\n\tbra COOL_WAIT;\n"
                 "COOL_DONE:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
// one elected lane of a converged warp (ptxas then keeps the TMA operands on the uniform datapath without a per-copy election loop)
__device__ __forceinline__ bool elect_one()
{
    unsigned r;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(r));
    return r != 0;
}
__device__ __forceinline__ float lg2_approx(float x)
{
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// opaque register copy of a constant: lets ptxas fold (b & m) | c into one LOP3 (one immediate per LOP3)
__device__ __forceinline__ int opaque_const(int c)
{
    int r;
    asm("mov.b32 %0, %1;" : "=r"(r) : "r"(c));
    return r;
}
__device__ __forceinline__ int and_or(int a, int andmask, int orbits)          // (a & andmask) | orbits
{
    int r;
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(r) : "r"(a), "r"(andmask), "r"(orbits));
    return r;
}
// address of element `off` (>= 0) of a float / float4 array: unsigned offset -> one IMAD.WIDE.U32
__device__ __forceinline__ const float *elem_addr(const float *base, int off) { return base + (unsigned)off; }
__device__ __forceinline__ const float4 *elem_addr(const float4 *base, int off) { return base + (unsigned)off; }
__device__ __forceinline__ float rsqrt_approx(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ------------------------------------------------------------------------------------------
// Node coordinate of a primitive along one table axis.
//   coord32 : t = (log2 q - lo)/Delta in node units, unclamped
//   split32 : tf = t_clamped + 1.5*2^23 rounded down (bit pattern 0x4B400000 + floor(t)),
//             fi = floor(t) as a float, w = t_clamped - floor(t) in [0,1),
//             d  = t_clamped - t (0 inside the table): the clamp correction of the T' form is d * d2f
// ------------------------------------------------------------------------------------------
constexpr float kMagic = 12582912.0f;              // 1.5 * 2^23
constexpr unsigned kMagicBits = 0x4B400000u;
struct Loc32 { float tf, fi, w, d; };
__device__ __forceinline__ float coord32(const AxisCoef &a, float q, int one_bits)
{
    // non-positive (and negative-NaN) -> bits 0 -> exponent -127: below every table (lower-edge clamp)
    const int b = max(__float_as_int(q), 0);
    const float u = __int_as_float((b >> 23) | 0x4B000000);                     // 2^23 + biased exponent, exact
    const float lm = lg2_approx(__int_as_float(and_or(b, 0x007fffff, one_bits)));   // MUFU.LG2 on [1,2): abs err 2^-22
    return fmaf(u - a.ke, a.invf, fmaf(lm, a.invf, a.cf));
}
template <bool DIAG>
__device__ __forceinline__ Loc32 split32(const AxisCoef &a, float t, bool &clamped)
{
    // t < 0 or t > n-1 in one unsigned compare of the bit patterns (negative floats compare above every positive one;
    // t is never -0: it is a sum that cancels to +0; a NaN t belongs to a cell that is not counted)
    if constexpr (DIAG) clamped |= __float_as_uint(t) > __float_as_uint(a.nm1f);
    const float tc = fminf(fmaxf(t, 0.f), a.tmaxf);
    Loc32 L;
    L.tf = __fadd_rd(tc, kMagic);
    L.fi = L.tf - kMagic;
    L.w = tc - L.fi;
    L.d = tc - t;
    return L;
}
template <bool DIAG>
__device__ __forceinline__ Loc32 locate32(const AxisCoef &a, float q, bool &clamped, int one_bits)
{
    return split32<DIAG>(a, coord32(a, q, one_bits), clamped);
}
__device__ __forceinline__ int loc_bits(const Loc32 &l) { return __float_as_int(l.tf); }
__device__ __forceinline__ float lerp(float w, float a, float b) { return fmaf(w, b - a, a); }

__device__ __forceinline__ float4 ldg_f4(const float4 *p)
{
    float4 v;
    asm("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ float4 lds_f4(unsigned addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ float lds_f32(unsigned addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}

// ------------------------------------------------------------------------------------------
// Lookup policies over the T' tables.  corners3 returns c[cr*4 + ce*2 + cb]; every policy feeds the
// same interpolation code, so the software variants agree bit for bit.
// ------------------------------------------------------------------------------------------
struct F32Global {
    static const char *name() { return "F32Global"; }
    static constexpr bool kHw = false, kSmem = false;
    const float *p1; const float4 *p4; int sr, se, si, c3, c4;
    __device__ F32Global(const DevTable &T, const void *) : p1(T.f1), p4(T.f4), sr(T.s_rho), se(T.s_the), si(T.s_thi)
    {
        c3 = (int)(0u - kMagicBits * (unsigned)(sr + se + 1));            // removes the bias of the three index words
        c4 = (int)(0u - kMagicBits * (unsigned)(sr + se + si + 1));
    }
    __device__ __forceinline__ void corners3(const Loc32 &r, const Loc32 &e, const Loc32 &b, float (&c)[8]) const
    {
        const int off = loc_bits(r) * sr + (loc_bits(e) * se + (loc_bits(b) + c3));
        const float *p = elem_addr(p1, off), *q = elem_addr(p1, off + se), *u = elem_addr(p1, off + sr), *v = elem_addr(p1, off + sr + se);
        c[0] = __ldg(p); c[1] = __ldg(p + 1); c[2] = __ldg(q); c[3] = __ldg(q + 1);
        c[4] = __ldg(u); c[5] = __ldg(u + 1); c[6] = __ldg(v); c[7] = __ldg(v + 1);
    }
    // the 16 texels around (r, e, ii, b): q[ce][ci][cr*2 + cb]
    __device__ __forceinline__ void corners4(const Loc32 &r, const Loc32 &e, const Loc32 &ii, const Loc32 &b, float4 (&q)[2][2][4]) const
    {
        const int off = loc_bits(r) * sr + (loc_bits(e) * se + (loc_bits(ii) * si + (loc_bits(b) + c4)));
#pragma unroll
        for (int ce = 0; ce < 2; ++ce)
#pragma unroll
            for (int ci = 0; ci < 2; ++ci) {
                const int o = off + (ce ? se : 0) + (ci ? si : 0);
                const float4 *a = elem_addr(p4, o), *u = elem_addr(p4, o + sr);
                q[ce][ci][0] = ldg_f4(a); q[ce][ci][1] = ldg_f4(a + 1); q[ce][ci][2] = ldg_f4(u); q[ce][ci][3] = ldg_f4(u + 1);
            }
    }
};
// MODE 3 quad layout: q3[r][e][b] = {T'(r,e,b), T'(r,e,b+1), T'(r,e+1,b), T'(r,e+1,b+1)} (same strides as the plain
// layout): a trilinear lookup is two 128-bit gathers, each inside one 32-byte sector.
struct F32GlobalQ {
    static const char *name() { return "F32GlobalQ"; }
    static constexpr bool kHw = false, kSmem = false;
    const float4 *pq; int sr, se, c3;
    __device__ F32GlobalQ(const DevTable &T, const void *) : pq(T.q3), sr(T.s_rho), se(T.s_the)
    {
        c3 = (int)(0u - kMagicBits * (unsigned)(sr + se + 1));
    }
    __device__ __forceinline__ void corners3(const Loc32 &r, const Loc32 &e, const Loc32 &b, float (&c)[8]) const
    {
        const int off = loc_bits(r) * sr + (loc_bits(e) * se + (loc_bits(b) + c3));
        const float4 lo = ldg_f4(elem_addr(pq, off)), hi = ldg_f4(elem_addr(pq, off + sr));
        c[0] = lo.x; c[1] = lo.y; c[2] = lo.z; c[3] = lo.w; c[4] = hi.x; c[5] = hi.y; c[6] = hi.z; c[7] = hi.w;
    }
    __device__ __forceinline__ void corners4(const Loc32 &, const Loc32 &, const Loc32 &, const Loc32 &, float4 (&)[2][2][4]) const {}
};
// MODE 3 oct layout: o3[r][e][b] = the eight corners of table cell (r, e, b) in one 32-byte sector
// {T'(r,e,b), T'(r,e,b+1), T'(r,e+1,b), T'(r,e+1,b+1), T'(r+1,e,b), ...}: a trilinear lookup is ONE 256-bit gather.
struct F32GlobalO {
    static const char *name() { return "F32GlobalO"; }
    static constexpr bool kHw = false, kSmem = false;
    const float4 *po; int sr, se, c3;
    __device__ F32GlobalO(const DevTable &T, const void *) : po(T.o3), sr(T.s_rho), se(T.s_the)
    {
        c3 = (int)(0u - kMagicBits * (unsigned)(sr + se + 1));
    }
    __device__ __forceinline__ void corners3(const Loc32 &r, const Loc32 &e, const Loc32 &b, float (&c)[8]) const
    {
        const int off = loc_bits(r) * sr + (loc_bits(e) * se + (loc_bits(b) + c3));
        const float4 *p = po + 2u * (unsigned)off;
        asm("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
            : "=f"(c[0]), "=f"(c[1]), "=f"(c[2]), "=f"(c[3]), "=f"(c[4]), "=f"(c[5]), "=f"(c[6]), "=f"(c[7]) : "l"(p));
    }
    __device__ __forceinline__ void corners4(const Loc32 &, const Loc32 &, const Loc32 &, const Loc32 &, float4 (&)[2][2][4]) const {}
};
struct F32Smem {
    static const char *name() { return "F32Smem"; }
    static constexpr bool kHw = false, kSmem = true;
    const float *p1; const float4 *p4; int sr, se, si, c3, c4;
    __device__ F32Smem(const DevTable &T, const void *img) : p1((const float *)img), p4((const float4 *)img), sr(T.s_rho), se(T.s_the), si(T.s_thi)
    {
        c3 = (int)(0u - kMagicBits * (unsigned)(sr + se + 1));
        c4 = (int)(0u - kMagicBits * (unsigned)(sr + se + si + 1));
    }
    __device__ __forceinline__ void corners3(const Loc32 &r, const Loc32 &e, const Loc32 &b, float (&c)[8]) const
    {
        const int off = loc_bits(r) * sr + (loc_bits(e) * se + (loc_bits(b) + c3));
        const float *p = p1 + off, *q = p + se, *u = p + sr, *v = u + se;
        c[0] = p[0]; c[1] = p[1]; c[2] = q[0]; c[3] = q[1]; c[4] = u[0]; c[5] = u[1]; c[6] = v[0]; c[7] = v[1];
    }
    __device__ __forceinline__ void corners4(const Loc32 &r, const Loc32 &e, const Loc32 &ii, const Loc32 &b, float4 (&q)[2][2][4]) const
    {
        const int off = loc_bits(r) * sr + (loc_bits(e) * se + (loc_bits(ii) * si + (loc_bits(b) + c4)));
        const float4 *p = p4 + off;
#pragma unroll
        for (int ce = 0; ce < 2; ++ce)
#pragma unroll
            for (int ci = 0; ci < 2; ++ci) {
                const float4 *a = p + (ce ? se : 0) + (ci ? si : 0), *u = a + sr;
                q[ce][ci][0] = a[0]; q[ce][ci][1] = a[1]; q[ce][ci][2] = u[0]; q[ce][ci][3] = u[1];
            }
    }
};
struct F32TexPoint {
    static const char *name() { return "F32TexPoint"; }
    static constexpr bool kHw = false, kSmem = false;
    cudaTextureObject_t tex; float nef;
    __device__ F32TexPoint(const DevTable &T, const void *) : tex(T.ftex_pt), nef((float)T.ax[CAX_THE].n) {}
    // float node indices (Loc32::fi) avoid int->float conversions; texel centres are at +0.5
    __device__ __forceinline__ void corners3(const Loc32 &r, const Loc32 &e, const Loc32 &b, float (&c)[8]) const
    {
        const float x = b.fi + 0.5f, y = e.fi + 0.5f, z = r.fi + 0.5f;
        c[0] = tex3D<float>(tex, x, y, z); c[1] = tex3D<float>(tex, x + 1.f, y, z);
        c[2] = tex3D<float>(tex, x, y + 1.f, z); c[3] = tex3D<float>(tex, x + 1.f, y + 1.f, z);
        c[4] = tex3D<float>(tex, x, y, z + 1.f); c[5] = tex3D<float>(tex, x + 1.f, y, z + 1.f);
        c[6] = tex3D<float>(tex, x, y + 1.f, z + 1.f); c[7] = tex3D<float>(tex, x + 1.f, y + 1.f, z + 1.f);
    }
    // the paper's flattening (L155-L159): z = i_rho * n_the + i_the
    __device__ __forceinline__ void corners4(const Loc32 &r, const Loc32 &e, const Loc32 &ii, const Loc32 &b, float4 (&q)[2][2][4]) const
    {
        const float x = b.fi + 0.5f;
#pragma unroll
        for (int ce = 0; ce < 2; ++ce)
#pragma unroll
            for (int ci = 0; ci < 2; ++ci) {
                const float y = ii.fi + (float)ci + 0.5f, z = fmaf(r.fi, nef, e.fi + (float)ce + 0.5f);
                q[ce][ci][0] = tex3D<float4>(tex, x, y, z); q[ce][ci][1] = tex3D<float4>(tex, x + 1.f, y, z);
                q[ce][ci][2] = tex3D<float4>(tex, x, y, z + nef); q[ce][ci][3] = tex3D<float4>(tex, x + 1.f, y, z + nef);
            }
    }
};
struct F32TexHw {
    static const char *name() { return "F32TexHw"; }
    static constexpr bool kHw = true, kSmem = false;
    cudaTextureObject_t tex; float nef;
    __device__ F32TexHw(const DevTable &T, const void *) : tex(T.ftex_lin), nef((float)T.ax[CAX_THE].n) {}
    // MODE 3: one trilinear fetch.  MODE 4: hardware bilinear on (bsq, theta_i) at the four
    // (rho, theta_e) slices; the flattened dimension is interpolated manually (the paper's scheme).
    __device__ __forceinline__ float hw3(const Loc32 &r, const Loc32 &e, const Loc32 &b) const
    {
        return tex3D<float>(tex, (b.fi + b.w) + 0.5f, (e.fi + e.w) + 0.5f, (r.fi + r.w) + 0.5f);
    }
    __device__ __forceinline__ float4 hw4(const Loc32 &r, const Loc32 &e, const Loc32 &ii, const Loc32 &b) const
    {
        const float x = (b.fi + b.w) + 0.5f, y = (ii.fi + ii.w) + 0.5f, z = fmaf(r.fi, nef, e.fi + 0.5f);
        const float4 v00 = tex3D<float4>(tex, x, y, z), v01 = tex3D<float4>(tex, x, y, z + 1.f);
        const float4 v10 = tex3D<float4>(tex, x, y, z + nef), v11 = tex3D<float4>(tex, x, y, z + nef + 1.f);
        float4 o;
        o.x = lerp(r.w, lerp(e.w, v00.x, v01.x), lerp(e.w, v10.x, v11.x));
        o.y = lerp(r.w, lerp(e.w, v00.y, v01.y), lerp(e.w, v10.y, v11.y));
        o.z = lerp(r.w, lerp(e.w, v00.z, v01.z), lerp(e.w, v10.z, v11.z));
        o.w = lerp(r.w, lerp(e.w, v00.w, v01.w), lerp(e.w, v10.w, v11.w));
        return o;
    }
    __device__ __forceinline__ void corners3(const Loc32 &, const Loc32 &, const Loc32 &, float (&)[8]) const {}
    __device__ __forceinline__ void corners4(const Loc32 &, const Loc32 &, const Loc32 &, const Loc32 &, float4 (&)[2][2][4]) const {}
};

// ------------------------------------------------------------------------------------------
// MODE 3: trilinear interpolation of T' (contract bsq, then Theta_e, then rho)
// ------------------------------------------------------------------------------------------
template <class Fetch>
__device__ __forceinline__ float interp3_f32(const Fetch &F, const Loc32 &r, const Loc32 &e, const Loc32 &b)
{
    if constexpr (Fetch::kHw) {
        return F.hw3(r, e, b);
    } else {
        float c[8];
        F.corners3(r, e, b, c);
        const float a00 = lerp(b.w, c[0], c[1]), a01 = lerp(b.w, c[2], c[3]);
        const float a10 = lerp(b.w, c[4], c[5]), a11 = lerp(b.w, c[6], c[7]);
        return lerp(r.w, lerp(e.w, a00, a01), lerp(e.w, a10, a11));
    }
}

// ------------------------------------------------------------------------------------------
// MODE 4: bilinear patch in (w_e, w_i) of the four channels over one (i_e, i_i) table cell:
//   y_k = c[k][0] + c[k][1] w_e + c[k][2] w_i + c[k][3] w_e w_i     (rho, bsq already contracted)
// ------------------------------------------------------------------------------------------
struct Patch4 { float c[4][4]; int ke, ki; };
template <class Fetch>
__device__ __forceinline__ void build_patch(const Fetch &F, const Loc32 &r, const Loc32 &b, const Loc32 &e, const Loc32 &ii, Patch4 &P)
{
    P.ke = loc_bits(e); P.ki = loc_bits(ii);
    float4 q[2][2][4];
    F.corners4(r, e, ii, b, q);
    float v[2][2][4];
#pragma unroll
    for (int ce = 0; ce < 2; ++ce)
#pragma unroll
        for (int ci = 0; ci < 2; ++ci) {
            const float4 *t = q[ce][ci];
            v[ce][ci][0] = lerp(r.w, lerp(b.w, t[0].x, t[1].x), lerp(b.w, t[2].x, t[3].x));
            v[ce][ci][1] = lerp(r.w, lerp(b.w, t[0].y, t[1].y), lerp(b.w, t[2].y, t[3].y));
            v[ce][ci][2] = lerp(r.w, lerp(b.w, t[0].z, t[1].z), lerp(b.w, t[2].z, t[3].z));
            v[ce][ci][3] = t[0].w;                       // log2 C depends on (i_e, i_i) only
        }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        P.c[k][0] = v[0][0][k];
        P.c[k][1] = v[1][0][k] - v[0][0][k];
        P.c[k][2] = v[0][1][k] - v[0][0][k];
        P.c[k][3] = (v[1][1][k] - v[1][0][k]) - P.c[k][2];
    }
}
__device__ __forceinline__ float patch_eval(const Patch4 &P, int k, float we, float wi)
{
    return fmaf(we, fmaf(wi, P.c[k][3], P.c[k][1]), fmaf(wi, P.c[k][2], P.c[k][0]));
}

// Coulomb coefficient C = 2^(bilinear log2 C) at (a = Theta_i, b = Theta_e) node coordinates.
//   CM = 1, QUAD  : quad layout {C(i,e), C(i,e+1), C(i+1,e), C(i+1,e+1)} staged in shared memory, one LDS.128;
//   CM = 1, !QUAD : plain layout staged in shared memory (SMEM variant: the table image leaves no room for quads);
//   CM = 0        : plain layout in global memory (L1-resident).
template <int CM, bool QUAD>
__device__ __forceinline__ float coulomb_C32(int n1, int qstride, const float *cg, unsigned cs, const Loc32 &a, const Loc32 &b)
{
    const int off = loc_bits(a) * n1 + (loc_bits(b) + (int)(0u - kMagicBits * (unsigned)(n1 + 1)));
    float c00, c01, c10, c11;
    if constexpr (CM >= 1 && QUAD) {
        // quad rows are skewed (row stride = 3 mod 8 quads) so that neighbouring (i, e) quads fall in different bank groups
        const int qoff = loc_bits(a) * qstride + (loc_bits(b) + (int)(0u - kMagicBits * (unsigned)(qstride + 1)));
        const float4 q = lds_f4(cs + 16u * (unsigned)qoff);
        c00 = q.x; c01 = q.y; c10 = q.z; c11 = q.w;
    } else if constexpr (CM >= 1) {
        const unsigned p = cs + 4u * (unsigned)off, q = p + 4u * (unsigned)n1;
        c00 = lds_f32(p); c01 = lds_f32(p + 4); c10 = lds_f32(q); c11 = lds_f32(q + 4);
    } else {
        const float *p = elem_addr(cg, off), *q = elem_addr(cg, off + n1);
        c00 = __ldg(p); c01 = __ldg(p + 1); c10 = __ldg(q); c11 = __ldg(q + 1);
    }
    return ex2_approx(lerp(a.w, lerp(b.w, c00, c01), lerp(b.w, c10, c11)));
}

// Radial profile (eq 25): the warp tile lies in one shell (shell_cells is a multiple of the tile): one warp sum and one
// fp64 atomic per luminosity term, into the warp's replica of this launch's shells.
template <int MODE>
__device__ __forceinline__ void shell_flush(const F32Const &S, const float (&part)[4], unsigned wtile)
{
    double *shell = S.lum_shell + (size_t)((blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) & S.shell_rmask) * S.shell_nloc4
                    + 4u * ((unsigned)(((unsigned long long)(S.tile_offset + wtile) * S.shell_magic) >> 40) - S.shell0);
#pragma unroll
    for (int k = 0; k < (MODE == 4 ? 4 : 1); ++k) {
        float t = part[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if ((threadIdx.x & 31) == 0) atomicAdd(shell + k, (double)t * S.lum_k);
    }
}

// Layout of the Coulomb table in shared memory, chosen by the launcher through CM: CM = 1 quads (64 KiB for 64^2, one
// LDS.128 per cell) — except for the SMEM variant, whose table image leaves no room: plain there too; CM = 2 the plain
// table (16 KiB, four LDS.32), used for small launches with diagnostics (configs[2]-sized: 8 M cells), where it measures
// 13 % faster (0.089 -> 0.077 ms) while at 512^3 the quads win by 6 %.
template <class Fetch, int CM>
__host__ __device__ constexpr bool coul_quads() { return CM == 1 && !Fetch::kSmem; }

struct Ctx32 { const DevTable &T; const F32Const &S; unsigned coul_s; };      // coul_s: shared-memory address of the staged Coulomb quads

// ------------------------------------------------------------------------------------------
// NV cells of one thread through all sub-steps, straight-line (no per-cell branches except the
// MODE-4 patch rebuild), so the compiler interleaves them for ILP.
//   CM: 1 = Coulomb from the coefficient table (shared-memory quads, or the 4th texel channel in
//           MODE 4), 0 = runtime S.coulomb (off / table in global memory / analytic)
// Cells with rho <= 0 pass through and cells with a NaN input give NaN (that cell only): they
// run through the arithmetic like any other cell and are patched at the end.
// ------------------------------------------------------------------------------------------
// Single update of a cell whose INPUT Theta_e lies in the steep band (F32Const::band_*): the only thing fp32 cannot carry
// there is the Theta_e node coordinate (the inputs are exact and no state is carried), so the rate is re-evaluated with
//   * t_e = (log2 Theta_e - lo)/Delta and its interval weight in fp64,
//   * the two Theta_e nodes contracted over (rho, bsq) in fp32, then y = a(e) + w_e (a(e+1) - a(e)) + log2 h + clamp terms in fp64,
//   * 2^y with the integer part exact and the fraction (|f| <= 1/2) by MUFU.EX2.
// Rare (a few cells in ten thousand) and out of line, so the step around it keeps its registers.  Reads the plain T' layout.
static __device__ __noinline__ float precise_rate3(const float *f1, int s_rho, int s_the, int n, double lo10, double inv10,
                                                   int ir, int ib, float wr, float wb, float the, float kcell)      // scalars only: no struct on the stack
{
    const double L10 = 3.321928094887362;
    const double t = (log2((double)the) - lo10 * L10) * (inv10 / L10);
    const double tc = fmin(fmax(t, 0.0), (double)(n - 1));
    int ie = (int)tc;
    if (ie > n - 2) ie = n - 2;
    const double w = tc - (double)ie;
    const float *p = f1 + ((size_t)ir * s_rho + (size_t)ie * s_the + ib), *q = p + s_the, *u = p + s_rho, *v = u + s_the;
    const float a0 = lerp(wr, lerp(wb, __ldg(p), __ldg(p + 1)), lerp(wb, __ldg(u), __ldg(u + 1)));      // node e
    const float a1 = lerp(wr, lerp(wb, __ldg(q), __ldg(q + 1)), lerp(wb, __ldg(v), __ldg(v + 1)));      // node e + 1
    double y = fma(w, (double)a1 - (double)a0, (double)a0) + ((tc - t) * (L10 / inv10) + (double)kcell);
    y = fmin(fmax(y, -1000.0), 1000.0);
    const double yi = rint(y);
    return (float)scalbn((double)ex2_approx((float)(y - yi)), (int)yi);
}

// FIXT: test every cell at every sub-step for the precise pass (F32Const::band_*): two integer subtractions and two unsigned
// compares on values that are live anyway.  (The 4-D step used to test inside its patch-rebuild branch only, with the cells in
// or next to the steep interval re-entering that branch every sub-step: measured 1.5 % slower than the plain test.)
// WF: also form the per-cell event flags (cool_cells::flags).  Compile time, because keeping the three event predicates of
// every cell alive to the end of the step costs the diagnostics kernels registers they do not have (s512f: 11 % with the
// flags merely possible); only tests and callers that pass a flags array get the WF instantiations.
// FLM: 1 = the temperature floor is a run-time switch (S.hfloor2 > 0), 0 = compiled out.  The floor test sits in the sub-step loop
// (the compiler predicates it rather than branching around it: 8 issue slots per sub-step when the floor is off), so the 4-D
// kernels, where the sub-step loop is nearly everything, exist in both forms.
template <int MODE, class Fetch, bool DIAG, int CM, bool NSUB1, int NV, bool FIXT, bool WF, int FLM>
__device__ __forceinline__ void step_cells_f32(const Ctx32 &X, const Fetch &F, const float *rho, const float *bsq, float *the, float *thi,
                                               const float *rr, const float *vol, DiagAcc &acc, float (&tile_part)[4], unsigned wtile,
                                               unsigned &flagword)   // byte j: event flags of cell j (include/cool.h); bit 3 = left to the precise pass
{
    const DevTable &T = X.T; const F32Const &S = X.S;
    const int coulomb = (CM >= 1) ? 1 : S.coulomb;
    const int one_bits = opaque_const(0x3f800000);
    const bool use_floor = FLM != 0 && S.hfloor2 > 0.f;     // warp-uniform
    bool bad[NV], any_bad = false;
    float in_e[NV], in_i[NV], nanq[NV];
    Loc32 lr[NV], lb[NV];
    float kcell[NV], coul_kr[NV], tfloor[NV], lsum[NV][4];
    bool clamped[NV], limited[NV], floored[NV];
    // events of the sub-step loop as running maxima (one instruction each per sub-step, decided once at the end) instead of
    // or-ed predicates, which the compiler keeps as bytes packed into registers: rlim = largest radiated fraction; cmax_* =
    // largest node-coordinate bit pattern of the Theta_e / Theta_i axis (unsigned: negative and too-large t both sort above n-1)
    float rlim[NV]; unsigned cmax_e[NV], cmax_i[NV];
    constexpr bool kMaxEv = DIAG && !NSUB1 && NV == 1;
    Patch4 P[(MODE == 4 && !Fetch::kHw) ? NV : 1];
#pragma unroll
    for (int j = 0; j < NV; ++j) {
        const float chk = (bsq[j] + the[j]) + (thi[j] + rho[j]);      // NaN when any input is NaN (or the sum overflows)
        nanq[j] = chk;
        bad[j] = !(rho[j] > 0.f) || chk != chk;
        any_bad |= bad[j];
        in_e[j] = the[j]; in_i[j] = thi[j];
        clamped[j] = limited[j] = floored[j] = false;
        rlim[j] = 0.f; cmax_e[j] = cmax_i[j] = 0u;
        lr[j] = locate32<DIAG>(T.ax[CAX_RHO], rho[j], clamped[j], one_bits);
        lb[j] = locate32<DIAG>(T.ax[CAX_BSQ], bsq[j], clamped[j], one_bits);
        tfloor[j] = 0.f;
        kcell[j] = fmaf(lr[j].d, T.ax[CAX_RHO].d2f, S.k0);     // log2 h + clamp correction of the rho axis
        coul_kr[j] = S.coul_kh * rho[j];
        lsum[j][0] = lsum[j][1] = lsum[j][2] = lsum[j][3] = 0.f;
        if (MODE == 4 && !Fetch::kHw) { P[j].ke = 0; P[j].ki = 0; }
    }
    if (use_floor) {
#pragma unroll
        for (int j = 0; j < NV; ++j)
            if (rr[j] > 0.f) {
                const float ok = __fdividef(rr[j], fmaf(rr[j], sqrtf(rr[j]), S.spin));     // Omega_K r
                tfloor[j] = S.hfloor2 * ok * ok;
            }
    }

    const int nsub = NSUB1 ? 1 : S.nsub;
    for (int s = 0; s < nsub; ++s) {
        bool changed = false;
        float drad_last[NV], fr[NV][3];
#pragma unroll
        for (int j = 0; j < NV; ++j) {
            const float te = coord32(T.ax[CAX_THE], the[j], one_bits);
            bool cdummy = false;
            const Loc32 le = split32<DIAG && !kMaxEv>(T.ax[CAX_THE], te, kMaxEv ? cdummy : clamped[j]);
            if constexpr (kMaxEv) cmax_e[j] = max(cmax_e[j], __float_as_uint(te));
            const float kk = fmaf(le.d, T.ax[CAX_THE].d2f, kcell[j]);
            float rrad, yc = 0.f, ti = 0.f;
            fr[j][0] = fr[j][1] = fr[j][2] = 0.f;
            Loc32 li{0.f, 0.f, 0.f, 0.f};
            if constexpr (MODE == 3) {
                rrad = ex2_approx(interp3_f32(F, lr[j], le, lb[j]) + kk);
            } else {
                ti = coord32(T.ax[CAX_THI], thi[j], one_bits);
                li = split32<DIAG && !kMaxEv>(T.ax[CAX_THI], ti, kMaxEv ? cdummy : clamped[j]);
                if constexpr (kMaxEv) cmax_i[j] = max(cmax_i[j], __float_as_uint(ti));
                float y0, y1, y2;
                if constexpr (Fetch::kHw) {
                    const float4 v = F.hw4(lr[j], le, li, lb[j]);
                    y0 = v.x; y1 = v.y; y2 = v.z; yc = v.w;
                } else {
                    if (loc_bits(le) != P[j].ke || loc_bits(li) != P[j].ki) build_patch(F, lr[j], lb[j], le, li, P[j]);
                    y0 = patch_eval(P[j], 0, le.w, li.w); y1 = patch_eval(P[j], 1, le.w, li.w);
                    y2 = patch_eval(P[j], 2, le.w, li.w); yc = patch_eval(P[j], 3, le.w, li.w);
                }
                const float rbr = ex2_approx(fminf(y0 + kk, 100.f));
                const float esy = y1 + kk;
                const float rsy = ex2_approx(fminf(esy + y2, 100.f));                              // eta * Q_syn
                const float rthin = rbr + rsy;                                                     // eq 10
                // eqs 13-14 and 11-12 in ratio form: tau_abs = r_thin inv_kB rho c_s / Theta_e^3
                const float num = fmaf(S.ae, the[j], S.ai * thi[j]), den = fmaf(S.be, the[j], fmaf(S.bi, thi[j], 1.f));
                const float rcs = rho[j] * (num * rsqrt_approx(num * den));                       // rho c_s
                const float th3 = fmaxf(the[j] * the[j] * the[j], 1e-30f);
                const float tau_abs = rthin * (S.inv_kB * rcs) * rcp_approx(th3);                 // eq 12
                const float tau_sca = S.ksca * rcs;
                rrad = rthin * rcp_approx(fmaf(tau_abs, fmaf(1.5f, tau_abs + tau_sca, 1.7320508f), 1.f));   // eq 11
                if constexpr (DIAG) {
                    const float inv = rcp_approx(fmaxf(rthin, 1e-37f));
                    const float rs0 = ex2_approx(fminf(esy, 100.f));                               // Q_syn alone
                    fr[j][0] = rbr * inv; fr[j][1] = rs0 * inv; fr[j][2] = (rsy - rs0) * inv;      // shares of Q_thin (reading C-21)
                }
            }
            if (use_floor) {
                if ((the[j] + thi[j]) * S.mr < tfloor[j]) { rrad = 0.f; floored[j] = true; }
            }
            // inside the steep band of the table, radiating a fraction that is neither negligible nor certainly limited: left to
            // the precise pass, passed through here like a cell without matter (the band is empty when no precise pass follows)
            if constexpr (FIXT) {
                if (((__float_as_uint(the[j]) - S.band_lo_bits) < S.band_w) & ((__float_as_uint(rrad) - S.rmin_bits) < S.r_w)) {
                    if constexpr (NSUB1 && !Fetch::kHw) {          // a single update: the precise rate, in place
                        rrad = precise_rate3(T.f1, T.s_rho, T.s_the, T.ax[CAX_THE].n, T.ax[CAX_THE].lo10, T.ax[CAX_THE].inv10,
                                             loc_bits(lr[j]) - (int)kMagicBits, loc_bits(lb[j]) - (int)kMagicBits, lr[j].w, lb[j].w, the[j], kcell[j]);
                        if (use_floor && floored[j]) rrad = 0.f;
                    } else { bad[j] = true; any_bad = true; nanq[j] = -0.f; }          // sub-steps: the precise pass
                }
            }
            if constexpr (DIAG) {
                if constexpr (NSUB1) limited[j] = rrad > S.f_limit;
                else rlim[j] = fmaxf(rlim[j], rrad);            // one FMNMX per sub-step; compared once at the end (NaN: no event, as before)
            }
            rrad = fminf(rrad, S.f_limit);
            // Coulomb exchange (eq 15), capped by f_limit of the donor and by the equalising transfer
            float dthe = 0.f;
            const float D = thi[j] - the[j];
            if (coulomb != 0) {
                float C;
                if (coulomb == 1) {
                    if (MODE == 4 && T.f4_has_coul) {
                        C = ex2_approx(yc);
                    } else {
                        bool dummy = false;
                        Loc32 ca, cb;                                   // Coulomb-table coordinates of Theta_i, Theta_e
                        // branch-free (identical axes give s = 1, o = 0 and the same node coordinate): keeps the NV cells interleaved
                        if (MODE == 4) ca = split32<false>(T.cax[0], fmaf(ti, S.cmi_s, S.cmi_o), dummy);
                        else ca = locate32<false>(T.cax[0], thi[j], dummy, one_bits);
                        cb = split32<false>(T.cax[1], fmaf(te, S.cme_s, S.cme_o), dummy);
                        C = coulomb_C32<CM, coul_quads<Fetch, CM>()>(T.cax[1].n, T.coulq_stride, T.fcoul, X.coul_s, ca, cb);
                    }
                } else {
                    C = (D != 0.f && !bad[j]) ? (float)coolphys::coulomb_C((double)the[j], (double)thi[j] / S.ion_ratio) : 0.f;
                }
                const float raw = coul_kr[j] * C * fabsf(D);
                const float cap1 = (D > 0.f) ? S.cap1i * thi[j] : S.cap1e * the[j];
                const float mag = fminf(raw, fminf(cap1, fabsf(D) * S.eq_frac));
                dthe = copysignf(mag, D);
            }
            // explicit _rn intrinsics: never contracted, so every instantiation rounds identically
            const float drad = __fmul_rn(rrad, the[j]);
            const float the_n = __fadd_rn(__fsub_rn(the[j], drad), dthe);
            const float thi_n = __fmaf_rn(-dthe, S.gi1_over_ge1, thi[j]);
            if constexpr (DIAG) {
                drad_last[j] = drad;
                lsum[j][0] += drad;
                if constexpr (MODE == 4) {                       // per-process split exists only for the three process tables
                    lsum[j][1] = fmaf(drad, fr[j][0], lsum[j][1]);
                    lsum[j][2] = fmaf(drad, fr[j][1], lsum[j][2]); lsum[j][3] = fmaf(drad, fr[j][2], lsum[j][3]);
                }
            }
            if constexpr (!NSUB1) changed |= (the_n != the[j]) | (thi_n != thi[j]);
            the[j] = the_n; thi[j] = thi_n;
        }
        if constexpr (!NSUB1) {
            // exact early exit: a sub-step that leaves every temperature bit-identical repeats itself
            if (!changed) {
                if constexpr (DIAG) {
                    const float rem = (float)(nsub - 1 - s);
#pragma unroll
                    for (int j = 0; j < NV; ++j) {
                        lsum[j][0] = fmaf(rem, drad_last[j], lsum[j][0]);
                        if constexpr (MODE == 4) {
#pragma unroll
                            for (int k = 0; k < 3; ++k) lsum[j][k + 1] = fmaf(rem, drad_last[j] * fr[j][k], lsum[j][k + 1]);
                        }
                    }
                }
                break;
            }
        }
    }
    flagword = 0u;
    if (any_bad) {                       // rare: rho <= 0 and cells of the precise pass pass through, NaN inputs give NaN
#pragma unroll
        for (int j = 0; j < NV; ++j)
            if (bad[j]) {
                const float z = __fsub_rn(nanq[j], nanq[j]);          // 0, or NaN
                the[j] = in_e[j] + z; thi[j] = in_i[j] + z;
                // a cell of the precise pass carries -0 in nanq (the sum of a valid cell's inputs is positive): flag bit 3
                if (__float_as_uint(nanq[j]) == 0x80000000u) flagword |= 8u << (8 * j);
            }
    }
    if constexpr (DIAG) {
        // the NV cells are summed in fp32 first (one fp64 add per sum per call): the fp64 pipe is narrow
        float part[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int j = 0; j < NV; ++j) {
            const float wgt = rho[j] * vol[j];                  // bad cells (possibly NaN) contribute an exact 0
            part[0] += bad[j] ? 0.f : lsum[j][0] * wgt;
            if constexpr (MODE == 4) {
#pragma unroll
                for (int k = 1; k < 4; ++k) part[k] += bad[j] ? 0.f : lsum[j][k] * wgt;
            }
            if constexpr (!NSUB1) limited[j] = rlim[j] > S.f_limit;
            if constexpr (kMaxEv) clamped[j] |= (cmax_e[j] > __float_as_uint(T.ax[CAX_THE].nm1f)) | (MODE == 4 && cmax_i[j] > __float_as_uint(T.ax[CAX_THI].nm1f));
            if (limited[j] && !bad[j]) ++acc.lim;               // predicated increments: the flags stay predicates
            if (floored[j] && !bad[j]) ++acc.flo;
            if (clamped[j] && !bad[j]) ++acc.cla;
        }
        if constexpr (WF) {                                     // per-cell event flags (cool_cells::flags): tests and callers that ask
#pragma unroll
            for (int j = 0; j < NV; ++j)
                if (!bad[j]) flagword |= ((limited[j] ? 1u : 0u) | (floored[j] ? 2u : 0u) | (clamped[j] ? 4u : 0u)) << (8 * j);
        }
        // the caller adds the tile's terms (the NV cells summed in fp32 first: the fp64 pipe is narrow) to its fp64 sums and
        // flushes them to the radial profile once per tile
#pragma unroll
        for (int k = 0; k < 4; ++k) tile_part[k] = part[k];
    }
}

// ------------------------------------------------------------------------------------------
// The kernel.  Dynamic shared memory:
//   [NW*NST mbarriers | NW warps x NST stages x nf arrays x 128 floats | Coulomb quads | table image (SMEM variant)]
// ------------------------------------------------------------------------------------------
constexpr int kF32CellsPerThread = 4;
constexpr int kWarpTile = 32 * kF32CellsPerThread;          // cells per warp tile
constexpr unsigned kWarpArrBytes = kWarpTile * 4u;          // 512 B per array per stage
constexpr unsigned kF32BarBytes = 1024;                     // room for 32 warps x 2 stages of 8-byte mbarriers, 32 list counters, the Coulomb barrier
constexpr unsigned kF32FixCntOff = 768;                     // per-warp count of tiles listed for the precise pass (32 x 4 bytes)

template <int MODE, class Fetch, bool DIAG, int CM, bool NSUB1, int THREADS, int NST, bool WF, int FLM>
__global__ void __launch_bounds__(THREADS, 1)
cool_f32_kernel(const DevTable T, const F32Const S, const CellPtrs C, double *partials, unsigned *ticket, cool_diag *d_diag)
{
    constexpr int NW = THREADS / 32;
    static_assert(NW * NST * 8 <= (int)kF32FixCntOff && NW * 4 <= (int)(kF32BarBytes - 8 - kF32FixCntOff), "mbarrier area too small");
    extern __shared__ __align__(128) unsigned char smem_f32[];
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);           // warp-uniform by construction: TMA operands stay in uniform registers

    // ---- prologue (the only CTA-wide barrier): stage the Coulomb quads / table image, arm the warp's barriers
    // The Coulomb table comes in by TMA bulk copies on a barrier of its own (last slot of the barrier area): the warps
    // arm their cell pipelines meanwhile and wait for it only just before the first tile
    const unsigned cbar = smem_u32(smem_f32) + kF32BarBytes - 8u;
    if (CM >= 1 && S.coul_smem && tid == 0) {
        constexpr bool kQuads = coul_quads<Fetch, CM>();
        const char *src = kQuads ? (const char *)T.fcoulq : (const char *)T.fcoul;  // plain table padded to 16 B at create time
        const unsigned bytes = kQuads ? (unsigned)T.coulq_bytes : (((unsigned)T.coul_bytes + 15u) & ~15u);
        mbar_init(cbar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(cbar, bytes);
        const unsigned dst = smem_u32(smem_f32 + S.coul_off);
        for (unsigned o = 0; o < bytes; o += 16384u) tma_load_1d(dst + o, src + o, min(16384u, bytes - o), cbar);
    }
    if constexpr (Fetch::kSmem) {
        const float4 *src = MODE == 3 ? (const float4 *)T.f1 : T.f4;
        float4 *dst = (float4 *)(smem_f32 + S.table_off);
        const unsigned n16 = T.table_bytes >> 4;                  // table_bytes is padded to 16 B at create time
        for (unsigned k = tid; k < n16; k += THREADS) dst[k] = ldg_f4(src + k);
    }
    const unsigned bar_w = smem_u32(smem_f32) + (unsigned)(warp * NST) * 8u;              // this warp's mbarriers
    const unsigned stg_w = smem_u32(smem_f32 + S.stage_off) + (unsigned)(warp * NST) * S.wstage_bytes;   // this warp's stages
    if (lane == 0) {
        *((unsigned *)(smem_f32 + kF32FixCntOff) + warp) = 0u;
#pragma unroll
        for (int s = 0; s < NST; ++s) mbar_init(bar_w + 8u * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    const Fetch F(T, smem_f32 + S.table_off);
    static_assert(DIAG || !WF, "per-cell flags come with the diagnostics");
    const Ctx32 X{T, S, smem_u32(smem_f32 + S.coul_off)};

    const long long ncell = C.ncell;
    const long long ntiles = (ncell + kWarpTile - 1) / kWarpTile;
    const long long nfull = S.use_tma ? ncell / kWarpTile : 0;                // tiles that go through TMA
    const long long GW = (long long)gridDim.x * NW;
    const int nf = S.nf;

    // lane 0 arms the stage's mbarrier and issues the bulk copies of one full warp tile
    auto issue = [&](long long tile, int s) {
        const unsigned bar = bar_w + 8u * (unsigned)s;
        const unsigned dst = stg_w + (unsigned)s * S.wstage_bytes;
        const size_t goff = (size_t)tile * kWarpArrBytes;
        mbar_expect_tx(bar, kWarpArrBytes * (unsigned)nf);
        tma_load_1d(dst, (const char *)C.rho + goff, kWarpArrBytes, bar);
        tma_load_1d(dst + kWarpArrBytes, (const char *)C.bsq + goff, kWarpArrBytes, bar);
        tma_load_1d(dst + 2 * kWarpArrBytes, (const char *)C.the_in + goff, kWarpArrBytes, bar);
        tma_load_1d(dst + 3 * kWarpArrBytes, (const char *)C.thi_in + goff, kWarpArrBytes, bar);
        unsigned k = 4;
        if (S.has_vol) { tma_load_1d(dst + k * kWarpArrBytes, (const char *)C.vol + goff, kWarpArrBytes, bar); ++k; }
        if (S.has_r) tma_load_1d(dst + k * kWarpArrBytes, (const char *)C.r + goff, kWarpArrBytes, bar);
    };

    constexpr bool kLists = !(MODE == 3 && NSUB1);          // a single 3-D update recomputes its precise cells in place: no lists
    long long tile = (long long)blockIdx.x * NW + warp;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NST; ++s)
            if (tile + s * GW < nfull) issue(tile + s * GW, s);
    }
    __syncwarp();

    if (CM >= 1 && S.coul_smem) mbar_wait(cbar, 0);
    DiagAcc acc;
    // The fp64 luminosity sums are touched once per tile: they live in local memory (L1), not in registers, on purpose.  The
    // diagnostics kernels sit at their register caps, and left to itself the compiler spills either these (harmless) or a
    // value inside the step (s512d: 0.81 vs 0.93 ms), depending on unrelated details of the source.
    constexpr int NLUM = MODE == 4 ? 4 : 1;                 // a 3-D table has no process split
    volatile double lumv[NLUM];
#pragma unroll
    for (int k = 0; k < NLUM; ++k) lumv[k] = 0.0;
    int s = 0; unsigned phase = 0;
    for (; tile < ntiles; tile += GW) {
        const long long c = tile * kWarpTile + (long long)lane * kF32CellsPerThread;
        float4 rho, bsq, the, thi;
        float4 vv = make_float4(1.f, 1.f, 1.f, 1.f), rr = make_float4(0.f, 0.f, 0.f, 0.f);
        const bool full = tile < nfull;
        if (full) {
            mbar_wait(bar_w + 8u * (unsigned)s, phase);
            const unsigned a = stg_w + (unsigned)s * S.wstage_bytes + 16u * (unsigned)lane;
            // vol first: it feeds only the diagnostic sums, and shared-memory loads of a warp return in order, so once
            // the outputs (which depend on every other array) are stored the whole stage has been read
            if (S.has_vol) vv = lds_f4(a + 4 * kWarpArrBytes);
            rho = lds_f4(a); bsq = lds_f4(a + kWarpArrBytes); the = lds_f4(a + 2 * kWarpArrBytes); thi = lds_f4(a + 3 * kWarpArrBytes);
            if (S.has_r) rr = lds_f4(a + (S.has_vol ? 5u : 4u) * kWarpArrBytes);
        } else {
            // ragged last tile, or arrays that are not 16-byte aligned: guarded scalar loads (zeros past the end: rho = 0 passes through)
#pragma unroll
            for (int j = 0; j < kF32CellsPerThread; ++j) {
                const bool in = c + j < ncell;
                (&rho.x)[j] = in ? __ldg((const float *)C.rho + c + j) : 0.f;
                (&bsq.x)[j] = in ? __ldg((const float *)C.bsq + c + j) : 0.f;
                (&the.x)[j] = in ? __ldg((const float *)C.the_in + c + j) : 0.f;
                (&thi.x)[j] = in ? __ldg((const float *)C.thi_in + c + j) : 0.f;
                if (S.has_vol) (&vv.x)[j] = in ? __ldg((const float *)C.vol + c + j) : 1.f;
                if (S.has_r) (&rr.x)[j] = in ? __ldg((const float *)C.r + c + j) : 0.f;
            }
        }
        float tp[4] = {0.f, 0.f, 0.f, 0.f};                 // this thread's luminosity terms of the tile (DIAG)
        unsigned flagword = 0u;                             // byte j: flags of cell j of this lane (bit 3: left to the precise pass)
        if constexpr (MODE == 4) {
            // the 16-register patch allows one cell at a time: one copy of the cell code, run four times with the
            // vectors rotated (a quarter of the instruction footprint of the unrolled form)
            auto rot = [](float4 &v) { const float t = v.x; v.x = v.y; v.y = v.z; v.z = v.w; v.w = t; };
#pragma unroll 1
            for (int j = 0; j < kF32CellsPerThread; ++j) {
                unsigned fw1;
                step_cells_f32<MODE, Fetch, DIAG, CM, NSUB1, 1, true, WF, FLM>(X, F, &rho.x, &bsq.x, &the.x, &thi.x, &rr.x, &vv.x, acc, tp, (unsigned)tile, fw1);
                if (fw1) flagword |= fw1 << (8 * j);        // rare
                // a finished cell's rho, bsq, vol and r slots are dead: they carry its four luminosity terms to the end of the tile
                if constexpr (DIAG) { rho.x = tp[0]; bsq.x = tp[1]; vv.x = tp[2]; rr.x = tp[3]; }
                rot(rho); rot(bsq); rot(the); rot(thi); rot(rr); rot(vv);
            }
            if constexpr (DIAG) {
                tp[0] = (rho.x + rho.y) + (rho.z + rho.w); tp[1] = (bsq.x + bsq.y) + (bsq.z + bsq.w);
                tp[2] = (vv.x + vv.y) + (vv.z + vv.w); tp[3] = (rr.x + rr.y) + (rr.z + rr.w);
            }
        } else {
            // Precise pass: a single update can only put a cell there if its INPUT Theta_e lies in the steep band, so one
            // warp-uniform look at the tile's inputs picks the step without any test (nearly every tile of a coherent field) or
            // the step that tests every cell.  Sub-stepped launches always test (a cell can cool into the band).
            bool tested = !NSUB1;
            if constexpr (NSUB1) {
                const bool inb = ((__float_as_uint(the.x) - S.band_lo_bits) < S.band_w) | ((__float_as_uint(the.y) - S.band_lo_bits) < S.band_w) |
                                 ((__float_as_uint(the.z) - S.band_lo_bits) < S.band_w) | ((__float_as_uint(the.w) - S.band_lo_bits) < S.band_w);
                tested = __any_sync(0xffffffffu, inb);
            }
            if (tested) step_cells_f32<MODE, Fetch, DIAG, CM, NSUB1, kF32CellsPerThread, true, WF, FLM>(X, F, &rho.x, &bsq.x, &the.x, &thi.x, &rr.x, &vv.x, acc, tp, (unsigned)tile, flagword);
            else step_cells_f32<MODE, Fetch, DIAG, CM, NSUB1, kF32CellsPerThread, false, WF, FLM>(X, F, &rho.x, &bsq.x, &the.x, &thi.x, &rr.x, &vv.x, acc, tp, (unsigned)tile, flagword);
        }
        if constexpr (DIAG) {
#pragma unroll
            for (int k = 0; k < NLUM; ++k) lumv[k] = lumv[k] + (double)tp[k];
            if (S.lum_shell) shell_flush<MODE>(S, tp, (unsigned)tile);
        }
        if (full) {
            st_stream((float4 *)C.the_out + (c >> 2), the);
            st_stream((float4 *)C.thi_out + (c >> 2), thi);
            if constexpr (WF) *((unsigned *)(C.flags + c)) = flagword;
            // Re-arm the stage only now: the stores above depend on every value this warp read from it, so its
            // LDS have all returned (read-before-overwrite across the generic and async proxies).  With NST
            // stages the refill is still NST-1 tiles ahead of its use.
            if (elect_one()) {
                const long long nxt = tile + (long long)NST * GW;
                if (nxt < nfull) issue(nxt, s);
            }
            if (++s == NST) { s = 0; phase ^= 1u; }
        } else {
#pragma unroll
            for (int j = 0; j < kF32CellsPerThread; ++j)
                if (c + j < ncell) {
                    ((float *)C.the_out)[c + j] = (&the.x)[j]; ((float *)C.thi_out)[c + j] = (&thi.x)[j];
                    if constexpr (WF) C.flags[c + j] = (unsigned char)(flagword >> (8 * j));
                }
        }
        if constexpr (kLists) if (S.fixmap) {               // cells left to the precise pass: list the tile
            if (__any_sync(0xffffffffu, (flagword & 0x08080808u) != 0u)) {
                const unsigned w0 = __ballot_sync(0xffffffffu, flagword & 0x8u), w1 = __ballot_sync(0xffffffffu, flagword & 0x800u);
                const unsigned w2 = __ballot_sync(0xffffffffu, flagword & 0x80000u), w3 = __ballot_sync(0xffffffffu, flagword & 0x8000000u);
                if (lane == 0) {
                    // this warp's count of listed tiles lives in shared memory (rarely touched; registers are scarce)
                    unsigned *cnt = (unsigned *)(smem_f32 + kF32FixCntOff) + warp;
                    const unsigned k = *cnt;
                    *cnt = k + 1u;
                    const size_t slot = (size_t)(blockIdx.x * NW + warp) * S.fix.cap + k;
                    S.fix.tile[slot] = (unsigned)tile;
                    S.fix.words[slot] = make_uint4(w0, w1, w2, w3);
                }
            }
        }
    }
    if constexpr (kLists) if (S.fixmap && lane == 0) S.fix.count[blockIdx.x * NW + warp] = *((unsigned *)(smem_f32 + kF32FixCntOff) + warp);      // every warp, every launch: no memset needed
    if constexpr (DIAG) {
#pragma unroll
        for (int k = 0; k < NLUM; ++k) acc.lum[k] = lumv[k];
        reduce_diag(acc, S.lum_k, partials, ticket, d_diag);
    }
}

// ------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------
struct LaunchCtx32 { const cool_table *t; F32Const S; const LaunchArgs *a; cudaStream_t st; };

constexpr int kF32Threads3 = 768, kF32Stages3 = 2;          // GLOBAL / texture variants, single-update 3-D step: 24 warps, 2 stages each
// ... with diagnostics: 20 warps x 96 registers.  At 80 registers the luminosity terms and event counters spill inside the step
// (s512d 0.88 -> 0.79 ms, s512f 0.91 -> 0.89 ms).  Thread counts are multiples of 128 so that the four schedulers of an SM hold
// the same number of warps: 608, 672 and 704 threads all measure 4-15 % slower than 640.
constexpr int kF32Threads3Diag = 640;
constexpr int kF32Threads4 = 512, kF32Stages4 = 2;          // GLOBAL / texture variants, sub-stepped or 4-D: 16 warps, 2 stages each
constexpr int kF32SmemThreads = 384, kF32SmemStages = 2;    // SMEM variant: the table image takes most of the shared memory
constexpr int kCoulQuadSmemMax = 73728;                     // Coulomb quads up to 64 x (64 + 2 skew) x 16 B (and a little more) are staged in shared memory

// fills the shared-memory layout fields of S for a launch with `threads` threads; returns the total
inline size_t f32_smem_layout(F32Const &S, int threads, int nst, bool table_in_smem, bool coul_quad, const cool_table *t)
{
    S.wstage_bytes = kWarpArrBytes * (unsigned)S.nf;
    S.stage_off = kF32BarBytes;
    size_t off = kF32BarBytes + (size_t)(threads / 32) * nst * S.wstage_bytes;
    S.coul_off = (unsigned)off;
    if (S.coul_smem) off += coul_quad ? (size_t)t->dev.coulq_bytes : (((size_t)t->dev.coul_bytes + 15) & ~(size_t)15);
    S.table_off = (unsigned)off;
    if (table_in_smem) off += t->dev.table_bytes;
    return off;
}

template <int MODE, class Fetch, bool DIAG, int CM, bool NSUB1, int THREADS, int NST, bool WF, int FLM>
static cudaError_t launch_f32_one(const LaunchCtx32 &L)
{
    F32Const S = L.S;
    const size_t smem = f32_smem_layout(S, THREADS, NST, Fetch::kSmem, coul_quads<Fetch, CM>(), L.t);
    auto kern = cool_f32_kernel<MODE, Fetch, DIAG, CM, NSUB1, THREADS, NST, WF, FLM>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    const LaunchArgs &a = *L.a;
    constexpr long long CTA_TILE = (long long)(THREADS / 32) * kWarpTile;
    const long long need = (a.ncell + CTA_TILE - 1) / CTA_TILE;
    const int grid = (int)(need < L.t->sm_count ? (need < 1 ? 1 : need) : L.t->sm_count);     // one persistent CTA per SM
    if (a.fixmap) {
        const unsigned warps = (unsigned)grid * (THREADS / 32);
        S.fix = fix_layout(a.fixmap, warps, (a.ncell + kWarpTile - 1) / kWarpTile);
        a.fix_warps = warps; a.fix_cap = S.fix.cap;
    }
    CellPtrs C{a.rho, a.bsq, a.the_in, a.thi_in, a.r, a.vol, a.the_out, a.thi_out, a.ncell, a.flags};
    note_kernel("cool_f32_kernel<MODE=%d,%s,DIAG=%d,CM=%d,NSUB1=%d,%dx%d%s%s>", MODE, Fetch::name(), (int)DIAG, CM, (int)NSUB1, THREADS, NST, WF ? ",flags" : "",
                FLM ? "" : ",nofloor");
    kern<<<grid, THREADS, smem, L.st>>>(L.t->dev, S, C, a.partials, a.ticket, a.d_diag);
    return cudaGetLastError();
}

// dispatch over the table variants for fixed <MODE, DIAG, CM, NSUB1>
template <int MODE, bool DIAG, int CM, bool NSUB1, bool WF, int FLM = 1>
static cudaError_t launch_f32_by_variant(const LaunchCtx32 &L, cool_variant v)
{
    // The single-update 3-D step fits 80 registers: 24 warps per SM hide the gather latency (measured best on B200:
    // 768 threads, 2 stages).  Sub-stepping loops and MODE 4 (a 16-register patch per cell) need 128 registers:
    // 16 warps, 2 stages (3 stages measure 1-4 % slower: less L1 under the gathers).
    constexpr bool kWide = MODE == 3 && NSUB1;
    constexpr int TH = kWide ? (DIAG ? kF32Threads3Diag : kF32Threads3) : kF32Threads4, NS = kWide ? kF32Stages3 : kF32Stages4;
    switch (v) {
        case COOL_V_GLOBAL:
            if constexpr (MODE == 3) {
                if (L.t->dev.o3) return launch_f32_one<MODE, F32GlobalO, DIAG, CM, NSUB1, TH, NS, WF, FLM>(L);
                if (L.t->dev.q3) return launch_f32_one<MODE, F32GlobalQ, DIAG, CM, NSUB1, TH, NS, WF, FLM>(L);
            }
            return launch_f32_one<MODE, F32Global, DIAG, CM, NSUB1, TH, NS, WF, FLM>(L);
        case COOL_V_TEX_POINT: return launch_f32_one<MODE, F32TexPoint, DIAG, CM, NSUB1, TH, NS, WF, FLM>(L);
        case COOL_V_TEX_HWFILTER: return launch_f32_one<MODE, F32TexHw, DIAG, CM, NSUB1, TH, NS, WF, FLM>(L);
        case COOL_V_SMEM: return launch_f32_one<MODE, F32Smem, DIAG, CM, NSUB1, kF32SmemThreads, kF32SmemStages, WF, FLM>(L);
        default: return cudaErrorInvalidValue;
    }
}

// one function per translation unit of instantiations (cool_inst_f32_*.cu)
cudaError_t launch_f32_m3(const LaunchCtx32 &L, cool_variant v, bool diag, int cm, bool nsub1);
cudaError_t launch_f32_m4(const LaunchCtx32 &L, cool_variant v, bool diag, int cm);
// the same with per-cell event flags (diagnostics on, LaunchArgs::flags set): translation units of their own
cudaError_t launch_f32_m3_flags(const LaunchCtx32 &L, cool_variant v, int cm, bool nsub1);
cudaError_t launch_f32_m4_flags(const LaunchCtx32 &L, cool_variant v, int cm);
// precise pass over the cells the fp32 launch listed in LaunchArgs::fixmap (cool_fix.cu)
cudaError_t launch_fix(const LaunchCtx &L, int mode, bool diag);

}  // namespace cool
