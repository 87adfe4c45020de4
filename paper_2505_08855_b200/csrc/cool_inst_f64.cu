// fp64 cells: {MODE 3, 4} x {diag off/on} x 4 lookup variants (Coulomb mode is a runtime branch)
#include "cool_kernels.cuh"
namespace cool {
cudaError_t launch_f64(const LaunchCtx &L, int mode, cool_variant v, bool diag)
{
    if (mode == 3) return diag ? launch_by_variant<double, 3, true, 0>(L, v) : launch_by_variant<double, 3, false, 0>(L, v);
    return diag ? launch_by_variant<double, 4, true, 0>(L, v) : launch_by_variant<double, 4, false, 0>(L, v);
}
}  // namespace cool
