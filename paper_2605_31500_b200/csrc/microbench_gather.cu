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
    } else if (row_bytes == 256) {
        run<8, 2>("256B", tab, idx, nidx, row_bytes, out, 8, 128);
        run<8, 4>("256B", tab, idx, nidx, row_bytes, out, 8, 128);
        run<8, 4>("256B", tab, idx, nidx, row_bytes, out, 16, 128);
        run<8, 8>("256B", tab, idx, nidx, row_bytes, out, 16, 128);
    } else if (row_bytes == 1024) {
        run<32, 2>("1024B", tab, idx, nidx, row_bytes, out, 8, 128);
        run<32, 4>("1024B", tab, idx, nidx, row_bytes, out, 8, 128);
        run<32, 4>("1024B", tab, idx, nidx, row_bytes, out, 16, 128);
    }
    return 0;
}
