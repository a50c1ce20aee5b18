#include "dispatch.cuh"
#include "ops_gt.cuh"
namespace gnn {
cudaError_t launch_gt_fwd(int dtype, const Shape& sh, const LaunchCtx& c, const GtArgs& a) {
    return dispatch_pass<GtFwd, kGtFwd>(dtype, sh, c, [&](auto& p) {
        p.q = (decltype(p.q))a.q; p.k = (decltype(p.k))a.k; p.v = (decltype(p.v))a.v;
        p.out = (decltype(p.out))a.out; p.lse = a.lse;
        p.qscale = kLog2e / sqrtf((float)sh.d);
    });
}
}  // namespace gnn
