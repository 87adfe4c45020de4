// fp32 cells, MODE 3 tables, diagnostics with per-cell event flags (cool_cells::flags): the instantiations of cool_inst_f32_m3.cu
// with DIAG on, once more with the flags compiled in
#include "cool_f32.cuh"
namespace cool {
template <int CM>
static cudaError_t gof(const LaunchCtx32 &L, cool_variant v, bool nsub1)
{
    return nsub1 ? launch_f32_by_variant<3, true, CM, true, true>(L, v) : launch_f32_by_variant<3, true, CM, false, true>(L, v);
}
cudaError_t launch_f32_m3_flags(const LaunchCtx32 &L, cool_variant v, int cm, bool nsub1)
{
    return cm == 2 ? gof<2>(L, v, nsub1) : cm ? gof<1>(L, v, nsub1) : gof<0>(L, v, nsub1);
}
}  // namespace cool
