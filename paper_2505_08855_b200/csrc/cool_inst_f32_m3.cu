// fp32 cells, MODE 3 tables: {diag off/on} x {Coulomb generic / table fast path} x {nsub loop / single update} x 4 lookup variants
#include "cool_f32.cuh"
namespace cool {
template <bool DIAG, int CM>
static cudaError_t go(const LaunchCtx32 &L, cool_variant v, bool nsub1)
{
    return nsub1 ? launch_f32_by_variant<3, DIAG, CM, true, false>(L, v) : launch_f32_by_variant<3, DIAG, CM, false, false>(L, v);
}
cudaError_t launch_f32_m3(const LaunchCtx32 &L, cool_variant v, bool diag, int cm, bool nsub1)
{
    if (diag && L.a->flags) return launch_f32_m3_flags(L, v, cm, nsub1);
    if (diag) return cm == 2 ? go<true, 2>(L, v, nsub1) : cm ? go<true, 1>(L, v, nsub1) : go<true, 0>(L, v, nsub1);
    return cm ? go<false, 1>(L, v, nsub1) : go<false, 0>(L, v, nsub1);
}
}  // namespace cool
