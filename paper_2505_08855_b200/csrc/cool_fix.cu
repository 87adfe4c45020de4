// cool_fix.cu — the precise pass behind the fp32 kernels of the cooling step (include/cool.h).
//
// Why it exists.  The fp32 path forms a cell's node coordinate along each table axis in fp32 (<= 5e-6 nodes) and carries
// Theta between sub-steps in fp32.  That holds north_star's 1e-5 on the updated energies as long as neighbouring Theta_e
// nodes of the table differ by less than kSteepLog2 (cool_internal.h).  The paper's own tables have one interval that does
// not: the K2(1/theta) -> 2 theta^2 substitution at T_e = 1e8 K (reading C-12) is a 16-19 log2-unit step
// between two nodes — a local power-law index of 60-140, so that a state error of 1e-6 entering the interval moves the
// rate by 1e-4, and the update can amplify it up to 40-fold (dTheta'/dTheta = 1 - r (1 + p)).  Only arithmetic that is
// accurate to fp32 rounding from the cell's first sub-step on survives that, so the cells concerned — inside a steep band
// at the start of a sub-step whose radiated fraction r is neither negligible nor certainly limited (cool_internal.h) — are
// not computed by the fp32 kernels at all: those pass the cells through, list their tiles, and this kernel recomputes them
// from their inputs with the fp64 step of cool_kernels.cuh on the canonical log10 tables (the arithmetic of fp64 cells:
// 1e-12 against the definition), stores them as fp32 and ADDS their luminosity terms and event counts to the cool_diag the
// fp32 kernel has just written.
//
// Work distribution.  Every warp of the fp32 launch has listed its tiles with marked cells (tile index + four 32-bit words,
// cool_internal.h fix_layout); tiles go round-robin over the fp32 warps, so a contiguous block of marked cells (a shell of
// a disc) is already spread over all lists.  One small block here takes one list and compacts its cells into a queue (cool_fix_kernel).
// The processing order is fixed by the lists, and the sums go warp -> block -> fixed-order last block: reproducible bit for bit.
#include "cool_f32.cuh"

namespace cool {

constexpr int kFixThreads = 64, kFixWarps = kFixThreads / 32;      // one small block per list of the fp32 launch: many blocks per SM
constexpr int kFixQueue = 1024;                                    // cells compacted per round (8 listed tiles)

template <int MODE, bool DIAG>
__global__ void __launch_bounds__(kFixThreads)
cool_fix_kernel(const DevTable T, const DevConst K, const StepConst S, const CellPtrs C, const FixLists L, unsigned nlists,
                double *partials, unsigned *ticket, cool_diag *d_diag)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const FetchGlobal F(T, nullptr);
    DiagAcc acc;
    const float *rho = (const float *)C.rho, *bsq = (const float *)C.bsq, *the_in = (const float *)C.the_in, *thi_in = (const float *)C.thi_in;
    const float *rr = (const float *)C.r, *vol = (const float *)C.vol;
    float *the_out = (float *)C.the_out, *thi_out = (float *)C.thi_out;

    auto process = [&](long long c) {
        double the = (double)the_in[c], thi = (double)thi_in[c];
        const double r = S.has_r ? (double)__ldg(rr + c) : 0.0, v = S.has_vol ? (double)__ldg(vol + c) : 1.0;
        int fl = 0;
        step_cell_f64<MODE, FetchGlobal, DIAG>(T, K, S, F, (double)__ldg(rho + c), (double)__ldg(bsq + c), the, thi, r, v, acc, c, &fl);
        the_out[c] = (float)the; thi_out[c] = (float)thi;
        if constexpr (DIAG) {
            if (C.flags) C.flags[c] = (unsigned char)(fl | 8);
        }
    };

    // One block per list.  The set bits of up to 8 listed tiles (32 words) are compacted, in list order, into a queue of cell
    // indices in shared memory (one word per lane of warp 0, an exclusive scan of the popcounts), and the block's warps take
    // the queue 32 cells at a time.  The step is long (fp64, every sub-step) and the marked cells are few, so what counts is
    // the number of passes a warp makes one after the other and how many blocks fit an SM: full warps, small blocks.
    __shared__ unsigned queue[kFixQueue];
    __shared__ unsigned s_total;
    const unsigned v = blockIdx.x;
    const unsigned cnt = __ldg(L.count + v);
    const size_t base = (size_t)v * L.cap;
    for (unsigned u0 = 0; u0 < 4u * cnt; u0 += 32u) {
        if (warp == 0) {
            const unsigned u = u0 + lane;
            unsigned w = 0u, tile = 0u;
            if (u < 4u * cnt) { w = __ldg((const unsigned *)(L.words + base + (u >> 2)) + (u & 3u)); tile = __ldg(L.tile + base + (u >> 2)); }
            unsigned pre = __popc(w);                          // inclusive scan over the lanes
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const unsigned t = __shfl_up_sync(0xffffffffu, pre, o); if (lane >= o) pre += t; }
            unsigned pos = pre - __popc(w);
            while (w) { const int b = __ffs(w) - 1; w &= w - 1u; queue[pos++] = tile * (unsigned)kWarpTile + (unsigned)b * 4u + (u & 3u); }
            if (lane == 31) s_total = pre;
        }
        __syncthreads();
        const unsigned total = s_total;
        for (unsigned q = threadIdx.x; q < total; q += kFixThreads) process((long long)queue[q]);
        __syncthreads();
    }

    if constexpr (DIAG) {
        // warp -> block -> per-block partials -> fixed-order sum by the last block, ADDED to the diagnostics of the fp32 kernel
        __shared__ double sh[kFixWarps][8];
        __shared__ unsigned s_last;
        __shared__ double fin[kFixThreads];
        double v[7] = {acc.lum[0], acc.lum[1], acc.lum[2], acc.lum[3], (double)acc.lim, (double)acc.flo, (double)acc.cla};
#pragma unroll
        for (int k = 0; k < 7; ++k) {
            v[k] = warp_sum(v[k]);
            if (lane == 0) sh[warp][k] = v[k];
        }
        __syncthreads();
        if (threadIdx.x < 7) {
            double s = 0.0;
            for (int w = 0; w < kFixWarps; ++w) s += sh[w][threadIdx.x];
            partials[(size_t)blockIdx.x * 8 + threadIdx.x] = s;
        }
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) s_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
        __syncthreads();
        if (!s_last) return;
        __threadfence();
        for (int k = 0; k < 7; ++k) {
            double s = 0.0;
            for (unsigned b = threadIdx.x; b < gridDim.x; b += kFixThreads) s += ((volatile double *)partials)[(size_t)b * 8 + k];
            fin[threadIdx.x] = s;
            __syncthreads();
            for (int o = kFixThreads / 2; o > 0; o >>= 1) {
                if (threadIdx.x < o) fin[threadIdx.x] += fin[threadIdx.x + o];
                __syncthreads();
            }
            if (threadIdx.x == 0) {
                if (k < 4) (&d_diag->lum_total)[k] += fin[0] * S.lum_k;
                else (&d_diag->n_limited)[k - 4] += (long long)(fin[0] + 0.5);
            }
            __syncthreads();
        }
        if (threadIdx.x == 0) *ticket = 0;
    }
}

cudaError_t launch_fix(const LaunchCtx &L, int mode, bool diag)
{
    const LaunchArgs &a = *L.a;
    const unsigned nlists = a.fix_warps;
    if (nlists == 0) return cudaSuccess;
    const FixLists lists = fix_layout(a.fixmap, nlists, (a.ncell + kWarpTile - 1) / kWarpTile);
    const int grid = (int)nlists;                                    // <= 24 lists per SM, within the diagnostics workspace's 32 blocks per SM
    CellPtrs C{a.rho, a.bsq, a.the_in, a.thi_in, a.r, a.vol, a.the_out, a.thi_out, a.ncell, a.flags};
#define COOL_FIX_LAUNCH(M, D) cool_fix_kernel<M, D><<<grid, kFixThreads, 0, L.st>>>(L.t->dev, L.t->cst, *L.S, C, lists, nlists, a.partials, a.ticket, a.d_diag)
    if (mode == 3) { if (diag) COOL_FIX_LAUNCH(3, true); else COOL_FIX_LAUNCH(3, false); }
    else { if (diag) COOL_FIX_LAUNCH(4, true); else COOL_FIX_LAUNCH(4, false); }
#undef COOL_FIX_LAUNCH
    return cudaGetLastError();
}

}  // namespace cool
