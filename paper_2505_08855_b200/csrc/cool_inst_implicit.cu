// COOL_SCHEME_IMPLICIT: {fp32, fp64 cells} x {MODE 3, 4} x {GLOBAL, SMEM, TEX_POINT} lookups (fp64 arithmetic throughout)
#include "cool_implicit.cuh"
namespace cool {
template <class Real, int MODE>
static cudaError_t go(const LaunchCtx &L, cool_variant v)
{
    switch (v) {
        case COOL_V_GLOBAL: return launch_implicit_one<Real, MODE, FetchGlobal>(L, 0);
        case COOL_V_TEX_POINT: return launch_implicit_one<Real, MODE, FetchTexPoint>(L, 0);
        case COOL_V_SMEM: return launch_implicit_one<Real, MODE, FetchSmem>(L, (size_t)L.t->dev.table_bytes);
        default: return cudaErrorInvalidValue;
    }
}
cudaError_t launch_implicit(const LaunchCtx &L, int mode, cool_variant v, cool_dtype dt)
{
    if (dt == COOL_F32) return mode == 3 ? go<float, 3>(L, v) : go<float, 4>(L, v);
    return mode == 3 ? go<double, 3>(L, v) : go<double, 4>(L, v);
}
}  // namespace cool
