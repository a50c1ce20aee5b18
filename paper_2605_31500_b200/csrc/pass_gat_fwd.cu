#include "dispatch.cuh"
#include "ops_gatv2.cuh"
namespace gnn {
cudaError_t launch_gat_fwd(int dtype, const Shape& sh, const LaunchCtx& c, const GatArgs& a) {
    return dispatch_pass<GatFwd, kGatFwd>(dtype, sh, c, [&](auto& p) {
        p.xl = (decltype(p.xl))a.xl; p.xr = (decltype(p.xr))a.xr; p.a = a.a;
        p.out = (decltype(p.out))a.out; p.lse = a.lse; p.slope = a.slope;
    });
}
}  // namespace gnn
