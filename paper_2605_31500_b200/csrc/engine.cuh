// engine.cuh - traversal engine shared by the six fused CSR attention passes (sm_100a).
//
// One "lane group" of G lanes covers one feature row of a node: every lane owns NV 16-byte vectors
// (VEC = 4 fp32 or 8 bf16 channels each), so a gathered neighbour row is a single coalesced 128-bit
// load per lane ("vectorized float4 loads"; the paper's block-per-(node, head) shape,
// PAPER.md:484, is prior art - here all heads of a row travel together so the gather is one
// contiguous H*d*b-byte burst).  A head's d channels sit in LPH = d/VEC adjacent lanes, so the score
// dot product is a log2(LPH)-step xor-shuffle, and the online-softmax state (running max, sum,
// accumulator) lives in registers.
//
// Three kernels per pass, picked by the plan's degree bins:
//   group_kernel    rows with deg <= warp_max_deg : one lane group per row, 32/G rows per warp,
//                   static round-robin over degree-sorted rows (heaviest first)
//   segment_kernel  CTA rows and hub chunks       : one CTA per segment, groups stride over the
//                   edge list, states merged through shared memory (the paper's cross-warp merge,
//                   PAPER.md:492)
//   hub_merge_kernel                                 : combines the chunk partials of a hub row in
//                   ascending chunk order (log-sum-exp merge for the forward, plain sums backward)
// Control flow is warp-uniform (masked edges instead of divergent trip counts) so full-mask shuffles
// are legal everywhere.  No floating-point atomics: every output element has exactly one writer.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace gnn {

constexpr int kCtaThreads = 256;
constexpr int kWarpsPerCta = kCtaThreads / 32;
constexpr int kU = 4;  // edges gathered per lane group per batch (independent loads in flight)
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

template <typename T> struct Elt;
template <> struct Elt<float> { static constexpr int VEC = 4; };
template <> struct Elt<__nv_bfloat16> { static constexpr int VEC = 8; };

struct Shape {
    int n;        // nodes
    int H;        // heads
    int d;        // head_dim
    int rowe;     // H * d elements per feature row
    int rowv;     // 16-byte vectors per feature row
    int lph;      // lanes per head = d / VEC (power of two, <= 32)
    int lph_log2;
};

struct BinView {
    const int32_t* perm;       // [n] rows sorted by (key, id): hubs, CTA rows, group rows
    const int32_t* chunks;     // [n_chunks][4] (row, e_begin, e_end, hub_slot)
    const int32_t* chunk_ptr;  // [n_hub + 1]
    int n_hub, n_cta, n_group, n_chunks;
};

struct LaunchCtx {
    cudaStream_t stream;
    int sm_count;
    const int32_t* rowptr;
    const int32_t* colidx;
    BinView bins;
    float* partials;  // [n_chunks][TE] hub-chunk partial states
    float* da_part;   // [da_slots][rowe] (ops with HAS_DA) or nullptr
    int da_slot_base; // first slot this pass may use
};

__device__ __forceinline__ float ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float lg2(float x) {
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// 16-byte read-only gather of one lane's vector, converted to fp32.  pred == false -> zeros, no traffic.
__device__ __forceinline__ void load_vec(const float* base, size_t elt, bool pred, float (&o)[4]) {
    float4 r = make_float4(0.f, 0.f, 0.f, 0.f);
    if (pred) r = __ldg(reinterpret_cast<const float4*>(base + elt));
    o[0] = r.x; o[1] = r.y; o[2] = r.z; o[3] = r.w;
}
__device__ __forceinline__ void load_vec(const __nv_bfloat16* base, size_t elt, bool pred, float (&o)[8]) {
    uint4 r = make_uint4(0u, 0u, 0u, 0u);
    if (pred) r = __ldg(reinterpret_cast<const uint4*>(base + elt));
    const uint32_t w[4] = {r.x, r.y, r.z, r.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        o[2 * i] = __uint_as_float(w[i] << 16);
        o[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
    }
}
// fp32 vector (always fp32 in memory: a, gradients)
template <int VEC> __device__ __forceinline__ void load_f32(const float* base, size_t elt, bool pred, float (&o)[VEC]) {
#pragma unroll
    for (int i = 0; i < VEC; i += 4) {
        float4 r = make_float4(0.f, 0.f, 0.f, 0.f);
        if (pred) r = __ldg(reinterpret_cast<const float4*>(base + elt + i));
        o[i] = r.x; o[i + 1] = r.y; o[i + 2] = r.z; o[i + 3] = r.w;
    }
}
template <int VEC> __device__ __forceinline__ void store_f32(float* base, size_t elt, const float (&v)[VEC]) {
#pragma unroll
    for (int i = 0; i < VEC; i += 4)
        *reinterpret_cast<float4*>(base + elt + i) = make_float4(v[i], v[i + 1], v[i + 2], v[i + 3]);
}
// store in the feature dtype (bf16: round-to-nearest-even)
__device__ __forceinline__ void store_vec(float* base, size_t elt, const float (&v)[4]) {
    *reinterpret_cast<float4*>(base + elt) = make_float4(v[0], v[1], v[2], v[3]);
}
__device__ __forceinline__ void store_vec(__nv_bfloat16* base, size_t elt, const float (&v)[8]) {
    uint4 r;
    uint32_t* w = reinterpret_cast<uint32_t*>(&r);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        __nv_bfloat162 b = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]);
        w[i] = *reinterpret_cast<uint32_t*>(&b);
    }
    *reinterpret_cast<uint4*>(base + elt) = r;
}

// lane geometry inside a group
template <int G, int NV, int VEC> struct Geo {
    int eoff[NV];   // element offset of this lane's vector t inside a feature row
    int hd[NV];     // head of vector t
    bool act[NV];   // vector t exists (rowv need not fill the group)
    bool lead[NV];  // first lane of its head (writes per-head scalars)
    int lph;
    __device__ __forceinline__ void init(const Shape& sh, int lane) {
        const int gl = lane & (G - 1);
        lph = sh.lph;
#pragma unroll
        for (int t = 0; t < NV; ++t) {
            const int vi = gl + t * G;
            act[t] = vi < sh.rowv;
            eoff[t] = vi * VEC;
            hd[t] = vi >> sh.lph_log2;
            lead[t] = act[t] && ((vi & (sh.lph - 1)) == 0);
        }
    }
};

// sum x[i] over the LPH lanes of a head (all 32 lanes must call)
template <int N> __device__ __forceinline__ void head_reduce(float (&x)[N], int lph) {
    for (int o = 1; o < lph; o <<= 1) {
#pragma unroll
        for (int i = 0; i < N; ++i) x[i] += __shfl_xor_sync(0xffffffffu, x[i], o);
    }
}

template <int NA, int NS, int NV, int VEC> struct State {
    float acc[NA][NV][VEC];
    float sc[NS > 0 ? NS : 1][NV];
    float m[NV];  // running max in the log2 domain (softmax passes only)
    __device__ __forceinline__ void reset() {
#pragma unroll
        for (int a = 0; a < NA; ++a)
#pragma unroll
            for (int t = 0; t < NV; ++t)
#pragma unroll
                for (int c = 0; c < VEC; ++c) acc[a][t][c] = 0.f;
#pragma unroll
        for (int s = 0; s < (NS > 0 ? NS : 1); ++s)
#pragma unroll
            for (int t = 0; t < NV; ++t) sc[s][t] = 0.f;
#pragma unroll
        for (int t = 0; t < NV; ++t) m[t] = -INFINITY;
    }
};

// number of floats of a serialised state: [NA][rowe] accumulators, [NS][H] scalars, [H] max (softmax)
template <class Op> __host__ __device__ inline int state_floats(const Shape& sh) {
    return Op::NA * sh.rowe + (Op::NS + (Op::SOFTMAX ? 1 : 0)) * sh.H;
}

}  // namespace gnn
