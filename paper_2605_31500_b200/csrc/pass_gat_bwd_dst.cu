#include "dispatch.cuh"
#include "ops_gatv2.cuh"
namespace gnn {
cudaError_t launch_gat_bwd_dst(int dtype, const Shape& sh, const LaunchCtx& c, const GatArgs& a) {
    return dispatch_pass<GatBwdDst, kGatBwdDst>(dtype, sh, c, [&](auto& p) {
        p.xl = (decltype(p.xl))a.xl; p.xr = (decltype(p.xr))a.xr; p.dout = (decltype(p.dout))a.dout;
        p.a = a.a; p.lse = a.lse; p.dxl = a.dxl; p.g = a.g; p.slope = a.slope;
    });
}

// fixed-order fp64 reduction of the per-CTA da partials (row a10): one thread per (h, c) element
__global__ void da_reduce_kernel(const float* __restrict__ part, int slots, int rowe, float* __restrict__ da) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= rowe) return;
    double s = 0.0;
    for (int k = 0; k < slots; ++k) s += (double)part[(size_t)k * rowe + e];
    da[e] = (float)s;
}
cudaError_t launch_da_reduce(const float* da_part, int slots, int rowe, float* da, cudaStream_t st) {
    prof_begin("gatv2_bwd_dst", "da_reduce", st);
    da_reduce_kernel<<<(rowe + 63) / 64, 64, 0, st>>>(da_part, slots, rowe, da);
    prof_end(st);
    ++g_launches;
    return cudaGetLastError();
}
}  // namespace gnn
