#include "dispatch.cuh"
#include "ops_gatv2.cuh"
namespace gnn {
cudaError_t launch_gat_bwd_src(int dtype, const Shape& sh, const LaunchCtx& c, const GatArgs& a) {
    return dispatch_pass<GatBwdSrc, kGatBwdSrc>(dtype, sh, c, [&](auto& p) {
        p.xl = (decltype(p.xl))a.xl; p.xr = (decltype(p.xr))a.xr; p.dout = (decltype(p.dout))a.dout;
        p.a = a.a; p.lse = a.lse; p.g = a.g; p.dxr = a.dxr; p.slope = a.slope;
    });
}
}  // namespace gnn
