#include "dispatch.cuh"
#include "ops_gt.cuh"
namespace gnn {
cudaError_t launch_gt_bwd_src(int dtype, const Shape& sh, const LaunchCtx& c, const GtArgs& a) {
    return dispatch_pass<GtBwdSrc, kGtBwdSrc>(dtype, sh, c, [&](auto& p) {
        p.q = (decltype(p.q))a.q; p.k = (decltype(p.k))a.k; p.v = (decltype(p.v))a.v;
        p.dout = (decltype(p.dout))a.dout; p.stat2 = a.stat2; p.dk = a.dk; p.dv = a.dv;
        p.kscale = kLog2e / sqrtf((float)sh.d); p.inv_sqrt_d = 1.f / sqrtf((float)sh.d); p.accumulate = a.accumulate;
    });
}
}  // namespace gnn
