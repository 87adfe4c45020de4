// COOL_V_ANALYTIC: eqs 1-12 and 15 evaluated per cell in fp64 for either cell dtype
#include "cool_kernels.cuh"
namespace cool {
template <class Real, int MODE>
static cudaError_t go(const LaunchCtx &L, bool diag)
{
    return diag ? launch_one<Real, MODE, FetchNone, true, true, 0, 256, 1>(L, 0) : launch_one<Real, MODE, FetchNone, true, false, 0, 256, 1>(L, 0);
}
cudaError_t launch_analytic(const LaunchCtx &L, int mode, cool_dtype dt, bool diag)
{
    if (dt == COOL_F32) return mode == 3 ? go<float, 3>(L, diag) : go<float, 4>(L, diag);
    return mode == 3 ? go<double, 3>(L, diag) : go<double, 4>(L, diag);
}
}  // namespace cool
