// COOL_SCHEME_IMPLICIT: {fp64 cells: fp64 solve, fp32 cells: fp32 solve on the T' tables} x {MODE 3, 4} x {GLOBAL, SMEM, TEX_POINT}
#include "cool_implicit.cuh"
namespace cool {
template <int MODE>
static cudaError_t go64(const LaunchCtx &L, cool_variant v)
{
    switch (v) {
        case COOL_V_GLOBAL: return launch_implicit_one<double, MODE, FetchGlobal>(L, 0);
        case COOL_V_TEX_POINT: return launch_implicit_one<double, MODE, FetchTexPoint>(L, 0);
        case COOL_V_SMEM: return launch_implicit_one<double, MODE, FetchSmem>(L, (size_t)L.t->dev.table_bytes);
        default: return cudaErrorInvalidValue;
    }
}
template <int MODE>
static cudaError_t go32(const LaunchCtx &L, const F32Const &S32, cool_variant v)
{
    switch (v) {
        case COOL_V_GLOBAL: return launch_implicit_f32_one<MODE, FetchGlobal>(L, S32, 0);
        case COOL_V_TEX_POINT: return launch_implicit_f32_one<MODE, FetchTexPoint>(L, S32, 0);
        case COOL_V_SMEM: return launch_implicit_f32_one<MODE, FetchSmem>(L, S32, (size_t)L.t->dev.table_bytes);
        default: return cudaErrorInvalidValue;
    }
}
cudaError_t launch_implicit(const LaunchCtx &L, const F32Const &S32, int mode, cool_variant v, cool_dtype dt)
{
    if (dt == COOL_F32) return mode == 3 ? go32<3>(L, S32, v) : go32<4>(L, S32, v);
    return mode == 3 ? go64<3>(L, v) : go64<4>(L, v);
}
}  // namespace cool
