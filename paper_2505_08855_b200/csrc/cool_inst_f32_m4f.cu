// fp32 cells, MODE 4 tables, diagnostics with per-cell event flags (cool_cells::flags)
#include "cool_f32.cuh"
namespace cool {
cudaError_t launch_f32_m4_flags(const LaunchCtx32 &L, cool_variant v, int cm)
{
    return cm == 2 ? launch_f32_by_variant<4, true, 2, false, true>(L, v) : cm ? launch_f32_by_variant<4, true, 1, false, true>(L, v) : launch_f32_by_variant<4, true, 0, false, true>(L, v);
}
}  // namespace cool
