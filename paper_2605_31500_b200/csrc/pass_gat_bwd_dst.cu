#include "dispatch.cuh"
#include "ops_gatv2.cuh"
namespace gnn {
cudaError_t launch_gat_bwd_dst(int dtype, const Shape& sh, const LaunchCtx& c, const GatArgs& a) {
    return dispatch_pass<GatBwdDst, kGatBwdDst>(dtype, sh, c, [&](auto& p) {
        p.xl = (decltype(p.xl))a.xl; p.xr = (decltype(p.xr))a.xr; p.dout = (decltype(p.dout))a.dout;
        p.a = a.a; p.lse = a.lse; p.dxl = a.dxl; p.g = a.g; p.slope = a.slope;
    });
}

// fixed-order fp64 reduction of the per-CTA da partials (row a10): one CTA per (h, c) element; thread t sums
// slots t, t+256, ... in fp64, then a fixed-shape shared-memory tree combines the 256 sums (no atomics,
// PAPER.md:498-500 uses atomicAdd here)
__global__ void __launch_bounds__(256) da_reduce_kernel(const float* __restrict__ part, int slots, int rowe,
                                                        float* __restrict__ da) {
    __shared__ double sm[256];
    const int e = blockIdx.x;
    double s = 0.0;
    for (int k = threadIdx.x; k < slots; k += 256) s += (double)part[(size_t)k * rowe + e];
    sm[threadIdx.x] = s;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if (threadIdx.x < w) sm[threadIdx.x] += sm[threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x == 0) da[e] = (float)sm[0];
}
cudaError_t launch_da_reduce(const float* da_part, int slots, int rowe, float* da, cudaStream_t st) {
    prof_begin("gatv2_bwd_dst", "da_reduce", st);
    da_reduce_kernel<<<rowe, 256, 0, st>>>(da_part, slots, rowe, da);
    prof_end(st);
    count_launch();
    return cudaGetLastError();
}
}  // namespace gnn
