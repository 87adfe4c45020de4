// fp32 cells, MODE 3 tables: {diag off/on} x {Coulomb generic / table fast path} x 4 lookup variants
#include "cool_kernels.cuh"
namespace cool {
cudaError_t launch_f32_m3(const LaunchCtx &L, cool_variant v, bool diag, int cm)
{
    if (diag) return cm ? launch_by_variant<float, 3, true, 1>(L, v) : launch_by_variant<float, 3, true, 0>(L, v);
    return cm ? launch_by_variant<float, 3, false, 1>(L, v) : launch_by_variant<float, 3, false, 0>(L, v);
}
}  // namespace cool
