// microbench_gather.cu - measurement aid (not part of libgnn_attn.so): achievable bandwidth of random
// row_bytes-sized row gathers with 256-bit loads, from HBM (table >> L2) and from L2 (table << L2), as a
// function of resident warps per SM and loads in flight per lane group.  This is "ceiling 2" of DESIGN.md
// section 6 (gather ingest).  Build: python -m paper_2605_31500_b200.build --microbench
// Run:   paper_2605_31500_b200/microbench_gather <row_bytes> [table_rows]
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("err %s line %d\n", cudaGetErrorString(e), __LINE__); exit(1);} }while(0)

// each group of G lanes reads one row (G*32 bytes) per edge with a 256-bit load; KU rows in flight per group
template <int G, int KU>
__global__ void gather256(const uint8_t* __restrict__ tab, const int* __restrict__ idx, long long nidx, int row_bytes, float* out) {
    const int lane = threadIdx.x & 31;
    const int gl = lane & (G - 1);
    const long long ngroups = (long long)gridDim.x * blockDim.x / G;
    const long long gid = ((long long)blockIdx.x * blockDim.x + threadIdx.x) / G;
    float acc = 0.f;
    for (long long e = gid * KU; e + KU <= nidx; e += ngroups * KU) {
        uint32_t r[KU][8];
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const int j = __ldg(idx + e + u);
            const uint8_t* p = tab + (size_t)j * row_bytes + gl * 32;
            asm volatile("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                : "=r"(r[u][0]),"=r"(r[u][1]),"=r"(r[u][2]),"=r"(r[u][3]),"=r"(r[u][4]),"=r"(r[u][5]),"=r"(r[u][6]),"=r"(r[u][7]) : "l"(p));
        }
#pragma unroll
        for (int u = 0; u < KU; ++u)
#pragma unroll
            for (int i = 0; i < 8; ++i) acc += __uint_as_float(r[u][i] << 16);
    }
    if (acc == 123.456f) out[0] = acc;
}

// ---- variant: rows fetched by the TMA unit (cp.async.bulk, SASS UBLKCP) into a per-warp shared-memory ring of S
// stages x R rows, completion on one mbarrier per stage; the bytes in flight hold no registers, so the depth is set by
// shared memory (S * R * row_bytes per warp), not by the register file.  The consumer reads its 32-byte slices of the
// landed rows with two LDS.128 and does the same arithmetic as gather256.
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile("{\n .reg .pred p;\n W_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
                 " @p bra D_%=;\n bra W_%=;\n D_%=:\n}" ::"r"(bar), "r"(parity) : "memory");
}
template <int G, int R, int S>
__global__ void gather_bulk(const uint8_t* __restrict__ tab, const int* __restrict__ idx, long long nidx, int row_bytes, float* out) {
    extern __shared__ __align__(128) uint8_t smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const int gl = lane & (G - 1), grp = lane / G;
    constexpr int GPW = 32 / G;
    uint8_t* ring = smem + (size_t)warp * S * R * row_bytes;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)nwarp * S * R * row_bytes) + warp * S;
    if (lane < S) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(bars + lane)) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncwarp();
    const long long nw = (long long)gridDim.x * nwarp, wid = (long long)blockIdx.x * nwarp + warp;
    const long long nbatch = nidx / R;                        // batches of R rows; warp w takes batches w, w + nw, ...
    const long long mine = wid < nbatch ? (nbatch - wid + nw - 1) / nw : 0;
    auto issue = [&](long long t) {                            // batch number t of this warp into stage t % S
        const int s = (int)(t % S);
        const uint32_t bar = smem_u32(bars + s);
        if (lane == 0) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(R * row_bytes) : "memory");
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
        __syncwarp();                                          // every lane has read stage s before it is refilled
        if (t + S < mine) issue(t + S);
    }
    if (acc == 123.456f) out[0] = acc;
}
template <int G, int R, int S> void run_bulk(const char* name, const uint8_t* tab, const int* idx, long long nidx, int row_bytes, float* out, int blocks_per_sm, int threads) {
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    const int grid = 148 * blocks_per_sm, nwarp = threads / 32;
    const size_t smem = (size_t)nwarp * S * R * row_bytes + (size_t)nwarp * S * 8;
    CK(cudaFuncSetAttribute(gather_bulk<G, R, S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    gather_bulk<G, R, S><<<grid, threads, smem>>>(tab, idx, nidx, row_bytes, out);
    CK(cudaDeviceSynchronize());
    cudaEventRecord(a);
    for (int it = 0; it < 3; ++it) gather_bulk<G, R, S><<<grid, threads, smem>>>(tab, idx, nidx, row_bytes, out);
    cudaEventRecord(b); CK(cudaEventSynchronize(b));
    float ms; cudaEventElapsedTime(&ms, a, b); ms /= 3;
    printf("%-12s bulk R=%d S=%d (%3zu KB/CTA) G=%2d warps/SM=%3d : %8.3f ms  %8.1f GB/s (rows) \n", name, R, S, smem >> 10, G,
           blocks_per_sm * threads / 32, ms, (double)nidx * row_bytes / ms * 1e-6);
}

template <int G, int KU> void run(const char* name, const uint8_t* tab, const int* idx, long long nidx, int row_bytes, float* out, int blocks_per_sm, int threads) {
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    int grid = 148 * blocks_per_sm;
    gather256<G, KU><<<grid, threads>>>(tab, idx, nidx, row_bytes, out);
    CK(cudaDeviceSynchronize());
    cudaEventRecord(a);
    for (int it = 0; it < 3; ++it) gather256<G, KU><<<grid, threads>>>(tab, idx, nidx, row_bytes, out);
    cudaEventRecord(b); CK(cudaEventSynchronize(b));
    float ms; cudaEventElapsedTime(&ms, a, b); ms /= 3;
    printf("%-28s G=%2d KU=%d warps/SM=%3d : %8.3f ms  %8.1f GB/s (rows) \n", name, G, KU, blocks_per_sm * threads / 32, ms, (double)nidx * row_bytes / ms * 1e-6);
}

int main(int argc, char** argv) {
    const int row_bytes = argc > 1 ? atoi(argv[1]) : 512;
    const long long nrows = argc > 2 ? atoll(argv[2]) : 4800000;
    const long long nidx = 64000000;
    uint8_t* tab; int* idx; float* out;
    CK(cudaMalloc(&tab, (size_t)nrows * row_bytes)); CK(cudaMemset(tab, 1, (size_t)nrows * row_bytes));
    CK(cudaMalloc(&idx, nidx * 4)); CK(cudaMalloc(&out, 4));
    int* h = (int*)malloc(nidx * 4);
    uint64_t s = 88172645463325252ull;
    for (long long i = 0; i < nidx; ++i) { s ^= s << 13; s ^= s >> 7; s ^= s << 17; h[i] = (int)(s % (uint64_t)nrows); }
    CK(cudaMemcpy(idx, h, nidx * 4, cudaMemcpyHostToDevice));
    printf("row_bytes %d, table %.2f GB, %lld random gathers\n", row_bytes, (double)nrows * row_bytes * 1e-9, nidx);
    if (row_bytes == 512) {
        run<16, 1>("512B", tab, idx, nidx, row_bytes, out, 8, 128);
        run<16, 2>("512B", tab, idx, nidx, row_bytes, out, 8, 128);
        run<16, 4>("512B", tab, idx, nidx, row_bytes, out, 4, 128);
        run<16, 4>("512B", tab, idx, nidx, row_bytes, out, 8, 128);
        run<16, 4>("512B", tab, idx, nidx, row_bytes, out, 16, 128);
        run<16, 8>("512B", tab, idx, nidx, row_bytes, out, 8, 128);
        run<16, 8>("512B", tab, idx, nidx, row_bytes, out, 16, 128);
        run_bulk<16, 8, 2>("512B", tab, idx, nidx, row_bytes, out, 4, 128);   // 32 KB/CTA, 16 warps/SM
        run_bulk<16, 8, 4>("512B", tab, idx, nidx, row_bytes, out, 3, 128);   // 64 KB/CTA, 12 warps/SM
        run_bulk<16, 8, 4>("512B", tab, idx, nidx, row_bytes, out, 2, 128);   //  8 warps/SM
        run_bulk<16, 16, 2>("512B", tab, idx, nidx, row_bytes, out, 3, 128);
        run_bulk<16, 4, 4>("512B", tab, idx, nidx, row_bytes, out, 4, 128);
    } else if (row_bytes == 256) {
        run<8, 2>("256B", tab, idx, nidx, row_bytes, out, 8, 128);
        run<8, 4>("256B", tab, idx, nidx, row_bytes, out, 8, 128);
        run<8, 4>("256B", tab, idx, nidx, row_bytes, out, 16, 128);
        run<8, 8>("256B", tab, idx, nidx, row_bytes, out, 16, 128);
        run_bulk<8, 16, 2>("256B", tab, idx, nidx, row_bytes, out, 4, 128);
        run_bulk<8, 16, 4>("256B", tab, idx, nidx, row_bytes, out, 3, 128);
        run_bulk<8, 8, 4>("256B", tab, idx, nidx, row_bytes, out, 4, 128);
    } else if (row_bytes == 1024) {
        run<32, 2>("1024B", tab, idx, nidx, row_bytes, out, 8, 128);
        run<32, 4>("1024B", tab, idx, nidx, row_bytes, out, 8, 128);
        run<32, 4>("1024B", tab, idx, nidx, row_bytes, out, 16, 128);
    }
    return 0;
}
