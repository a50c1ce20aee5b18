// probe.cu - measurement aid behind gnn_probe_gather (include/gnn_attn.h): the achievable rate of uniformly random
// row gathers, i.e. "ceiling 2" of DESIGN.md section 6 (gather ingest) measured in the same process as the layer, on
// an HBM-resident table (>> L2) or an L2-resident one, at the row size of the config.  Two kernels with the same
// consumer arithmetic:
//   mode 0  register gathers: one 256-bit load per lane per row (LDG.E.256), `depth` rows in flight per lane group
//           - what the traversal kernels of kernels.cuh do;
//   mode 1  TMA bulk copies (cp.async.bulk, SASS UBLKCP) into a per-warp shared-memory ring of 2 stages x `depth`
//           rows completing on one mbarrier per stage - bytes in flight hold no registers.
// bench.py times the launch with CUDA events on the caller's stream and prints GB/s next to the kernels' own rates.
#include <cuda_runtime.h>
#include <stdint.h>

#include "internal.h"

namespace gnn {
void prof_begin(const char* pass, const char* kernel, cudaStream_t st);
void prof_end(cudaStream_t st);
namespace {

template <int G, int KU>
__global__ void __launch_bounds__(128)
probe_ldg_kernel(const uint8_t* __restrict__ tab, const int32_t* __restrict__ idx, long long nidx, int row_bytes,
                 float* __restrict__ sink) {
    const int gl = threadIdx.x & (G - 1);
    const long long ngroups = (long long)gridDim.x * blockDim.x / G;
    const long long gid = ((long long)blockIdx.x * blockDim.x + threadIdx.x) / G;
    float acc = 0.f;
    for (long long e = gid * KU; e + KU <= nidx; e += ngroups * KU) {
        Raw<32> r[KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) r[u] = ldg_raw<32>(tab + (size_t)__ldg(idx + e + u) * row_bytes + gl * 32, true);
#pragma unroll
        for (int u = 0; u < KU; ++u)
#pragma unroll
            for (int i = 0; i < 8; ++i) acc += __uint_as_float(r[u].w[i] << 16);
    }
    if (acc == 123.456f) sink[0] = acc;   // keeps the loads alive; never true for the all-ones probe table
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile("{\n .reg .pred p;\n W_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
                 " @p bra D_%=;\n bra W_%=;\n D_%=:\n}" ::"r"(bar), "r"(parity) : "memory");
}

template <int G, int R>
__global__ void __launch_bounds__(128)
probe_bulk_kernel(const uint8_t* __restrict__ tab, const int32_t* __restrict__ idx, long long nidx, int row_bytes,
                  float* __restrict__ sink) {
    constexpr int S = 2, GPW = 32 / G;
    extern __shared__ __align__(128) uint8_t smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const int gl = lane & (G - 1), grp = lane / G;
    uint8_t* ring = smem + (size_t)warp * S * R * row_bytes;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)nwarp * S * R * row_bytes) + warp * S;
    if (lane < S) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(bars + lane)) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncwarp();
    const long long nw = (long long)gridDim.x * nwarp, wid = (long long)blockIdx.x * nwarp + warp;
    const long long nbatch = nidx / R;     // batches of R rows; warp w takes batches w, w + nw, ...
    const long long mine = wid < nbatch ? (nbatch - wid + nw - 1) / nw : 0;
    auto issue = [&](long long t) {
        const int s = (int)(t % S);
        const uint32_t bar = smem_u32(bars + s);
        if (lane == 0)
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(R * row_bytes) : "memory");
        __syncwarp();
        if (lane < R) {
            const int j = __ldg(idx + (wid + t * nw) * R + lane);
            const uint32_t dst = smem_u32(ring + ((size_t)s * R + lane) * row_bytes);
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(dst), "l"(tab + (size_t)j * row_bytes), "r"(row_bytes), "r"(bar) : "memory");
        }
    };
    for (long long t = 0; t < S && t < mine; ++t) issue(t);
    float acc = 0.f;
    for (long long t = 0; t < mine; ++t) {
        const int s = (int)(t % S);
        mbar_wait(smem_u32(bars + s), (uint32_t)((t / S) & 1));
#pragma unroll
        for (int r = grp; r < R; r += GPW) {
            const uint32_t a = smem_u32(ring + ((size_t)s * R + r) * row_bytes + gl * 32);
            uint32_t v[8];
            asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]) : "r"(a));
            asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]) : "r"(a + 16));
#pragma unroll
            for (int i = 0; i < 8; ++i) acc += __uint_as_float(v[i] << 16);
        }
        __syncwarp();                      // every lane has read stage s before it is refilled
        if (t + S < mine) issue(t + S);
    }
    if (acc == 123.456f) sink[0] = acc;
}

template <int G>
cudaError_t launch_probe(int mode, int depth, int grid, const uint8_t* tab, const int32_t* idx, long long nidx,
                         int row_bytes, float* sink, cudaStream_t st) {
    if (mode == 0) {
        if (depth == 1) probe_ldg_kernel<G, 1><<<grid, 128, 0, st>>>(tab, idx, nidx, row_bytes, sink);
        else if (depth == 2) probe_ldg_kernel<G, 2><<<grid, 128, 0, st>>>(tab, idx, nidx, row_bytes, sink);
        else if (depth == 4) probe_ldg_kernel<G, 4><<<grid, 128, 0, st>>>(tab, idx, nidx, row_bytes, sink);
        else if (depth == 8) probe_ldg_kernel<G, 8><<<grid, 128, 0, st>>>(tab, idx, nidx, row_bytes, sink);
        else return cudaErrorInvalidValue;
        return cudaGetLastError();
    }
    auto go = [&](auto kern, int R) -> cudaError_t {
        const size_t smem = (size_t)4 * 2 * R * row_bytes + 4 * 2 * 8;
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        kern<<<grid, 128, smem, st>>>(tab, idx, nidx, row_bytes, sink);
        return cudaGetLastError();
    };
    if (depth == 4) return go(probe_bulk_kernel<G, 4>, 4);
    if (depth == 8) return go(probe_bulk_kernel<G, 8>, 8);
    if (depth == 16) return go(probe_bulk_kernel<G, 16>, 16);
    return cudaErrorInvalidValue;
}

}  // namespace
}  // namespace gnn

using namespace gnn;

extern "C" gnn_status_t gnn_probe_gather(const void* table, int64_t table_rows, int32_t row_bytes, const int32_t* idx,
                                         int64_t n_idx, int32_t mode, int32_t depth, int32_t ctas_per_sm, float* sink,
                                         gnn_stream_t stream) {
    const char* who = "gnn_probe_gather";
    if (!table || !idx || !sink || table_rows < 1 || n_idx < 1 || ctas_per_sm < 1 || ctas_per_sm > 16 ||
        (((uintptr_t)table) & 31) != 0) {
        set_error("%s: NULL / misaligned pointer or bad sizes", who);
        return GNN_EINVAL;
    }
    if (row_bytes != 256 && row_bytes != 512 && row_bytes != 1024) {
        set_error("%s: row_bytes must be 256, 512 or 1024", who);
        return GNN_EUNSUPPORTED;
    }
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int grid = sms * ctas_per_sm;
    cudaStream_t st = (cudaStream_t)stream;
    const uint8_t* tab = (const uint8_t*)table;
    prof_begin("probe", mode == 0 ? "gather_ldg" : "gather_bulk", st);
    cudaError_t e = row_bytes == 256   ? launch_probe<8>(mode, depth, grid, tab, idx, n_idx, row_bytes, sink, st)
                    : row_bytes == 512 ? launch_probe<16>(mode, depth, grid, tab, idx, n_idx, row_bytes, sink, st)
                                       : launch_probe<32>(mode, depth, grid, tab, idx, n_idx, row_bytes, sink, st);
    prof_end(st);
    if (e == cudaErrorInvalidValue) {
        set_error("%s: depth must be 1, 2, 4 or 8 (mode 0) / 4, 8 or 16 (mode 1)", who);
        return GNN_EUNSUPPORTED;
    }
    if (e != cudaSuccess) { set_error("%s: CUDA error: %s", who, cudaGetErrorString(e)); return GNN_ECUDA; }
    count_launch();
    return GNN_OK;
}
