#include "dispatch.cuh"
#include "ops_agg.cuh"
namespace gnn {
cudaError_t launch_min_fwd(int dtype, const Shape& sh, const LaunchCtx& c, const AggArgs& a, bool rows_sorted) {
    auto fill = [&](auto& p) {
        p.x = (decltype(p.x))a.x; p.out = (decltype(p.out))a.out; p.arg = a.arg; p.sign = a.sign;
    };
    return rows_sorted ? dispatch_pass<MinFwdSorted, kMinFwd>(dtype, sh, c, fill) : dispatch_pass<MinFwd, kMinFwd>(dtype, sh, c, fill);
}

// Backward of the min / max aggregation: a sparse scatter-add through the saved indices.  One thread
// per 4 consecutive channels of one destination row: 16-byte loads of arg and dout, four fire-and-forget
// red.global.add.f32.  N*C reductions in total (against E*C gathered values in the forward), so the atomic unit is
// not the bound; the order of the additions into one dx element is not fixed (the paper's scheme, stated in DESIGN).
template <typename T>
__global__ void __launch_bounds__(256)
minmax_scatter_kernel(const int32_t* __restrict__ arg, const T* __restrict__ dout, float* __restrict__ dx, long long nquads,
                      int rowe) {
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < nquads; t += (long long)gridDim.x * blockDim.x) {
        const long long e = 4 * t;
        const int c = (int)(e % rowe);
        const int4 j = __ldg(reinterpret_cast<const int4*>(arg + e));
        float g[4];
        if constexpr (sizeof(T) == 4) {
            const float4 v = __ldg(reinterpret_cast<const float4*>(dout + e));
            g[0] = v.x; g[1] = v.y; g[2] = v.z; g[3] = v.w;
        } else {
            const uint2 v = __ldg(reinterpret_cast<const uint2*>(dout + e));
            g[0] = __uint_as_float(v.x << 16); g[1] = __uint_as_float(v.x & 0xffff0000u);
            g[2] = __uint_as_float(v.y << 16); g[3] = __uint_as_float(v.y & 0xffff0000u);
        }
        const int js[4] = {j.x, j.y, j.z, j.w};
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (js[u] >= 0) atomicAdd(dx + (size_t)js[u] * rowe + c + u, g[u]);
    }
}

cudaError_t launch_minmax_scatter(int dtype, long long n, int rowe, const AggArgs& a, int sm_count, cudaStream_t st) {
    const long long nquads = n * rowe / 4;
    if (nquads == 0) return cudaSuccess;
    const int grid = (int)std::min<long long>((nquads + 255) / 256, (long long)sm_count * 32);
    prof_begin("seg_minmax_bwd", "scatter", st);
    if (dtype == GNN_F32)
        minmax_scatter_kernel<float><<<grid, 256, 0, st>>>(a.arg, (const float*)a.dout, a.dx, nquads, rowe);
    else
        minmax_scatter_kernel<__nv_bfloat16><<<grid, 256, 0, st>>>(a.arg, (const __nv_bfloat16*)a.dout, a.dx, nquads, rowe);
    prof_end(st);
    count_launch();
    return cudaGetLastError();
}
}  // namespace gnn
