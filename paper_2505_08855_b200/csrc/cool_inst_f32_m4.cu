// fp32 cells, MODE 4 tables: {diag off/on} x {Coulomb generic / table fast path} x {floor run-time / compiled out} x 4 lookup variants
#include "cool_f32.cuh"
namespace cool {
template <int FLM>
static cudaError_t go4(const LaunchCtx32 &L, cool_variant v, bool diag, int cm)
{
    if (diag) return cm == 2 ? launch_f32_by_variant<4, true, 2, false, false, FLM>(L, v) : cm ? launch_f32_by_variant<4, true, 1, false, false, FLM>(L, v) : launch_f32_by_variant<4, true, 0, false, false, FLM>(L, v);
    return cm ? launch_f32_by_variant<4, false, 1, false, false, FLM>(L, v) : launch_f32_by_variant<4, false, 0, false, false, FLM>(L, v);
}
cudaError_t launch_f32_m4(const LaunchCtx32 &L, cool_variant v, bool diag, int cm)
{
    if (diag && L.a->flags) return launch_f32_m4_flags(L, v, cm);
    return L.S.hfloor2 > 0.f ? go4<1>(L, v, diag, cm) : go4<0>(L, v, diag, cm);
}
}  // namespace cool
