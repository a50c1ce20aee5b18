// dot_aggr.cu - row f4 (second half): the paper's cache-sensitive `dot-aggr` micro-benchmark:
//   out[i] = sum over the stored in-neighbours j of i of <x_i, x_j>
// as two warp-per-node kernels "that have identical arithmetic but different memory access patterns":
//   feature-parallel   the lanes of the warp span the D features; the neighbours are scanned one after the other, every
//                      neighbour row is read with coalesced loads (scalar: 4 bytes per lane, vec: 16 bytes per lane);
//   neighbour-parallel every lane takes different neighbours (lane l: entries l, l + 32, ... of the row) and walks the D
//                      features of ITS neighbour row alone - gather-like loads, 32 different rows per warp instruction.
// Both accumulate in fp32 and finish with a warp reduction.  bench.py times a second pass over the same inputs (the
// paper's "second-pass to expose cache reuse") for natural, randomly permuted and degree-sorted node ids and reports the
// reordering gap Delta s = s_neighbour - s_feature.  A measurement aid of the locality study, not a layer.
#include <cuda_runtime.h>
#include <stdint.h>

#include "internal.h"

namespace gnn {
void prof_begin(const char* pass, const char* kernel, cudaStream_t st);
void prof_end(cudaStream_t st);
namespace {

__device__ __forceinline__ float wsum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <bool VEC>
__global__ void __launch_bounds__(256)
dot_aggr_feature_kernel(const int32_t* __restrict__ rowptr, const int32_t* __restrict__ colidx, const float* __restrict__ x,
                        int n, int D, float* __restrict__ out) {
    const int lane = threadIdx.x & 31;
    const int nw = gridDim.x * (blockDim.x >> 5);
    for (int i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); i < n; i += nw) {
        const int e0 = __ldg(rowptr + i), e1 = __ldg(rowptr + i + 1);
        const float* xi = x + (size_t)i * D;
        float acc = 0.f;
        for (int e = e0; e < e1; ++e) {
            const float* xj = x + (size_t)__ldg(colidx + e) * D;
            if (VEC) {
                for (int c = lane * 4; c < D; c += 128) {
                    const float4 a = __ldg(reinterpret_cast<const float4*>(xi + c)), b = __ldg(reinterpret_cast<const float4*>(xj + c));
                    acc = fmaf(a.x, b.x, fmaf(a.y, b.y, fmaf(a.z, b.z, fmaf(a.w, b.w, acc))));
                }
            } else {
                for (int c = lane; c < D; c += 32) acc = fmaf(__ldg(xi + c), __ldg(xj + c), acc);
            }
        }
        acc = wsum(acc);
        if (lane == 0) out[i] = acc;
    }
}

template <bool VEC>
__global__ void __launch_bounds__(256)
dot_aggr_neighbor_kernel(const int32_t* __restrict__ rowptr, const int32_t* __restrict__ colidx, const float* __restrict__ x,
                         int n, int D, float* __restrict__ out) {
    const int lane = threadIdx.x & 31;
    const int nw = gridDim.x * (blockDim.x >> 5);
    for (int i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); i < n; i += nw) {
        const int e0 = __ldg(rowptr + i), e1 = __ldg(rowptr + i + 1);
        const float* xi = x + (size_t)i * D;
        float acc = 0.f;
        for (int e = e0 + lane; e < e1; e += 32) {
            const float* xj = x + (size_t)__ldg(colidx + e) * D;
            if (VEC) {
                for (int c = 0; c < D; c += 4) {
                    const float4 a = __ldg(reinterpret_cast<const float4*>(xi + c)), b = __ldg(reinterpret_cast<const float4*>(xj + c));
                    acc = fmaf(a.x, b.x, fmaf(a.y, b.y, fmaf(a.z, b.z, fmaf(a.w, b.w, acc))));
                }
            } else {
                for (int c = 0; c < D; ++c) acc = fmaf(__ldg(xi + c), __ldg(xj + c), acc);
            }
        }
        acc = wsum(acc);
        if (lane == 0) out[i] = acc;
    }
}

}  // namespace
}  // namespace gnn

using namespace gnn;

extern "C" gnn_status_t gnn_dot_aggr(int32_t n, const int32_t* rowptr, const int32_t* colidx, const float* x, int32_t dim,
                                     int32_t mode, int32_t vec, float* out, gnn_stream_t stream) {
    const char* who = "gnn_dot_aggr";
    if (n < 1 || !rowptr || !colidx || !x || !out) { set_error("%s: n < 1 or NULL pointer argument", who); return GNN_EINVAL; }
    if (dim < 4 || dim % 4 != 0 || (mode != 0 && mode != 1) || (((uintptr_t)x) & 15) != 0) {
        set_error("%s: dim must be a positive multiple of 4, mode 0 | 1, x 16-byte aligned", who);
        return GNN_EUNSUPPORTED;
    }
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int grid = (int)(((long long)n + 7) / 8 < (long long)sms * 16 ? ((long long)n + 7) / 8 : (long long)sms * 16);
    cudaStream_t st = (cudaStream_t)stream;
    prof_begin("dot_aggr", mode ? (vec ? "neighbor_vec" : "neighbor") : (vec ? "feature_vec" : "feature"), st);
    if (mode == 0 && !vec) dot_aggr_feature_kernel<false><<<grid, 256, 0, st>>>(rowptr, colidx, x, n, dim, out);
    else if (mode == 0) dot_aggr_feature_kernel<true><<<grid, 256, 0, st>>>(rowptr, colidx, x, n, dim, out);
    else if (!vec) dot_aggr_neighbor_kernel<false><<<grid, 256, 0, st>>>(rowptr, colidx, x, n, dim, out);
    else dot_aggr_neighbor_kernel<true><<<grid, 256, 0, st>>>(rowptr, colidx, x, n, dim, out);
    prof_end(st);
    count_launch();
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_error("%s: CUDA error: %s", who, cudaGetErrorString(e)); return GNN_ECUDA; }
    return GNN_OK;
}
