// engine.cuh - traversal engine shared by the six fused CSR attention passes (sm_100a).
//
// One "lane group" of G lanes covers one feature row of a node.  Every lane owns CH = NV * VEC
// CONTIGUOUS channels of ONE head, fetched with NV 128-bit or 256-bit read-only loads
// (LDG.E.128 / LDG.E.256, the latter new on sm_100), so a gathered neighbour row is one contiguous
// H*d*b-byte burst per group ("vectorized float4 loads"; the paper's
// block-per-(node, head) shape, is prior art - here all heads of a row travel
// together).  A head's d channels sit in LPL = d/CH adjacent lanes, so the score dot product ends
// in a log2(LPL)-step xor-shuffle (none at all when a lane holds a whole head), and the
// online-softmax state (running max, sum, accumulator) lives in registers.  Wider CH
// means fewer lanes repeat the same per-(edge, head) scalar work and more edges per warp instruction.
//
// Three kernels per pass, picked by the plan's degree bins:
//   group_kernel    rows with deg <= warp_max_deg : one lane group per row, 32/G rows per warp,
//                   static round-robin over degree-sorted rows (heaviest first)
//   segment_kernel  CTA rows and hub chunks       : one CTA per segment, groups stride over the
//                   edge list, states merged through shared memory (the paper's cross-warp merge,
//                   PAPER.md:492)
//   hub_merge_kernel                                 : combines the chunk partials of a hub row in
//                   a fixed chunk order (log-sum-exp merge for the forward, plain sums backward)
// Control flow is warp-uniform (masked edges instead of divergent trip counts) so full-mask shuffles
// are legal everywhere.  No floating-point atomics: every output element has exactly one writer.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace gnn {

void count_launch(int k = 1);   // host-side launch counter, atomic (api.cu; gnn_launch_count)
bool pdl_enabled();             // run-time switch of the dependent-launch overlap (api.cu; gnn_pdl_enable)

// tuning knobs (profiles/r01_lane_width_sweep.md): resident CTAs per SM the register budget is held to and
// register double-buffering of the gathers, for the forward and the backward passes
#ifndef GNN_FWD_MINB
#define GNN_FWD_MINB 4
#endif
#ifndef GNN_FWD_DB
#define GNN_FWD_DB 0
#endif
#ifndef GNN_BWD_MINB
#define GNN_BWD_MINB 3
#endif
#ifndef GNN_BWD_DB
#define GNN_BWD_DB 0
#endif
#ifndef GNN_GAT_DST_MINB
#define GNN_GAT_DST_MINB 3
#endif
#ifndef GNN_GAT_SRC_MINB
#define GNN_GAT_SRC_MINB 4
#endif
constexpr int kCtaThreads = 128;
constexpr int kWarpsPerCta = kCtaThreads / 32;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

struct Shape {
    int n;          // nodes
    int H;          // heads
    int d;          // head_dim
    int rowe;       // H * d elements per feature row (of the heads this launch processes)
    int ld;         // elements between consecutive rows of the [n, H_total, d] tensors (== rowe unless the call
                    // was split into head groups, api.cu)
    int ldh;        // elements between consecutive rows of the [n, H_total] arrays (lse, Delta, G, stat2)
    int ch;         // channels per lane (CH)
    int lanes;      // active lanes per row = rowe / ch
    int lpl;        // lanes per head = d / ch (power of two)
    int lpl_log2;
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

// ---- mixed-precision arithmetic on packed bf16 pairs (sm_100: FHFMA.BF16 / FHADD.BF16 take the .H0/.H1 half
// of a register directly, so bf16 operands need no unpack instruction; products are exact, sums fp32)
__device__ __forceinline__ void fma_bf16x2(uint32_t a, uint32_t b, float& acc0, float& acc1) {
    asm("{\n .reg .b16 al, ah, bl, bh;\n mov.b32 {al, ah}, %2;\n mov.b32 {bl, bh}, %3;\n"
        " fma.rn.f32.bf16 %0, al, bl, %0;\n fma.rn.f32.bf16 %1, ah, bh, %1;\n}"
        : "+f"(acc0), "+f"(acc1) : "r"(a), "r"(b));
}
// first products of a dot: the accumulator operand is the zero register, so no register pair has to be cleared first
__device__ __forceinline__ void mul_bf16x2(uint32_t a, uint32_t b, float& acc0, float& acc1) {
    asm("{\n .reg .b16 al, ah, bl, bh;\n mov.b32 {al, ah}, %2;\n mov.b32 {bl, bh}, %3;\n"
        " fma.rn.f32.bf16 %0, al, bl, 0f00000000;\n fma.rn.f32.bf16 %1, ah, bh, 0f00000000;\n}"
        : "=f"(acc0), "=f"(acc1) : "r"(a), "r"(b));
}
// ---- packed fp32 pairs (sm_100 FFMA2 / FADD2 / FMUL2: two fp32 lanes of a 64-bit register pair per instruction;
// a scalar operand is broadcast by the instruction itself).  The pairs are named as two floats; ptxas allocates them
// to aligned register pairs, so the mov.b64 packs below cost nothing.
__device__ __forceinline__ void fma2(float& a0, float& a1, float w, float x0, float x1) {            // a += w * x
    asm("{\n .reg .b64 ww, xx, cc;\n mov.b64 ww, {%2, %2};\n mov.b64 xx, {%3, %4};\n mov.b64 cc, {%0, %1};\n"
        " fma.rn.f32x2 cc, ww, xx, cc;\n mov.b64 {%0, %1}, cc;\n}" : "+f"(a0), "+f"(a1) : "f"(w), "f"(x0), "f"(x1));
}
__device__ __forceinline__ void fma2v(float& a0, float& a1, float w0, float w1, float x0, float x1) {  // a += w .* x
    asm("{\n .reg .b64 ww, xx, cc;\n mov.b64 ww, {%2, %3};\n mov.b64 xx, {%4, %5};\n mov.b64 cc, {%0, %1};\n"
        " fma.rn.f32x2 cc, ww, xx, cc;\n mov.b64 {%0, %1}, cc;\n}" : "+f"(a0), "+f"(a1) : "f"(w0), "f"(w1), "f"(x0), "f"(x1));
}
__device__ __forceinline__ void mul2(float& a0, float& a1, float w) {                                 // a *= w
    asm("{\n .reg .b64 ww, cc;\n mov.b64 ww, {%2, %2};\n mov.b64 cc, {%0, %1};\n"
        " mul.rn.f32x2 cc, cc, ww;\n mov.b64 {%0, %1}, cc;\n}" : "+f"(a0), "+f"(a1) : "f"(w));
}
__device__ __forceinline__ void mul2v(float& o0, float& o1, float w0, float w1, float x0, float x1) {  // o = w .* x
    asm("{\n .reg .b64 ww, xx, cc;\n mov.b64 ww, {%2, %3};\n mov.b64 xx, {%4, %5};\n"
        " mul.rn.f32x2 cc, ww, xx;\n mov.b64 {%0, %1}, cc;\n}" : "=f"(o0), "=f"(o1) : "f"(w0), "f"(w1), "f"(x0), "f"(x1));
}
// predicated pair add: (a0, a1) += (x0, x1) if pred (one FADD2 under a predicate)
__device__ __forceinline__ void add2_if(bool pred, float& a0, float& a1, float x0, float x1) {
    asm("{\n .reg .pred q;\n .reg .b64 xx, cc;\n setp.ne.b32 q, %4, 0;\n mov.b64 xx, {%2, %3};\n mov.b64 cc, {%0, %1};\n"
        " @q add.rn.f32x2 cc, cc, xx;\n mov.b64 {%0, %1}, cc;\n}" : "+f"(a0), "+f"(a1) : "f"(x0), "f"(x1), "r"((int)pred));
}
// a[c] += w * x[c] and a[c] *= w over a lane's channels
template <int CH> __device__ __forceinline__ void axpy(float (&a)[CH], float w, const float (&x)[CH]) {
#pragma unroll
    for (int c = 0; c < CH; c += 2) fma2(a[c], a[c + 1], w, x[c], x[c + 1]);
}
template <int CH> __device__ __forceinline__ void scale(float (&a)[CH], float w) {
#pragma unroll
    for (int c = 0; c < CH; c += 2) mul2(a[c], a[c + 1], w);
}

// ---- L2 prefetch of a feature row that a later batch will gather (run_edges): no destination register, so the
// bytes in flight are not bounded by the register file.  GNN_PF_MODE 0: off (default); 1: one prefetch.global.L2 per
// 128-byte line (SASS CCTL.E.PF2); 2: one cp.async.bulk.prefetch.L2 per row (TMA unit).  Measured on B200
// (profiles/r02_csr_experiments.md): both modes are SLOWER than no prefetch (cfg 3 step +8 % / +17 %, cfg 5 +4 % /
// +29 %) - the extra requests cost more in the memory pipeline than the shorter latency returns - so the knob
// stays off; it is kept for the record.
#ifndef GNN_PF_MODE
#define GNN_PF_MODE 0
#endif
__device__ __forceinline__ void prefetch_row_l2(const void* row, int bytes) {
#if GNN_PF_MODE == 1
    for (int o = 0; o < bytes; o += 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char*>(row) + o));
#elif GNN_PF_MODE == 2
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(row), "r"(bytes) : "memory");
#endif
}
// (lo, hi) halves of a packed bf16 pair, each added to an fp32 value: z = bf16 + f32
__device__ __forceinline__ void add_bf16x2(uint32_t a, float x0, float x1, float& z0, float& z1) {
    // volatile: stops the compiler from keeping z alive across the head reduction instead of recomputing it
    asm volatile("{\n .reg .b16 al, ah;\n mov.b32 {al, ah}, %2;\n add.rn.f32.bf16 %0, al, %3;\n add.rn.f32.bf16 %1, ah, %4;\n}"
        : "=f"(z0), "=f"(z1) : "r"(a), "f"(x0), "f"(x1));
}

// ---- raw VB-byte gathers (VB = 16 or 32), kept unconverted until use so in-flight loads stay small
template <int VB> struct Raw { uint32_t w[VB / 4]; };

template <int VB> __device__ __forceinline__ Raw<VB> ldg_raw(const void* p, bool pred);
template <> __device__ __forceinline__ Raw<16> ldg_raw<16>(const void* p, bool pred) {
    Raw<16> r;
    r.w[0] = r.w[1] = r.w[2] = r.w[3] = 0u;
    if (pred)
        asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];"
                     : "=r"(r.w[0]), "=r"(r.w[1]), "=r"(r.w[2]), "=r"(r.w[3]) : "l"(p));
    return r;
}
template <> __device__ __forceinline__ Raw<32> ldg_raw<32>(const void* p, bool pred) {
    Raw<32> r;
#pragma unroll
    for (int i = 0; i < 8; ++i) r.w[i] = 0u;
    if (pred)
        asm volatile("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=r"(r.w[0]), "=r"(r.w[1]), "=r"(r.w[2]), "=r"(r.w[3]), "=r"(r.w[4]), "=r"(r.w[5]),
                       "=r"(r.w[6]), "=r"(r.w[7]) : "l"(p));
    return r;
}

// element i of a raw vector as fp32 (exact up-cast for bf16)
template <typename T, int VB> __device__ __forceinline__ float raw_elt(const Raw<VB>& r, int i);
template <> __device__ __forceinline__ float raw_elt<float, 16>(const Raw<16>& r, int i) { return __uint_as_float(r.w[i]); }
template <> __device__ __forceinline__ float raw_elt<float, 32>(const Raw<32>& r, int i) { return __uint_as_float(r.w[i]); }
template <> __device__ __forceinline__ float raw_elt<__nv_bfloat16, 16>(const Raw<16>& r, int i) {
    return __uint_as_float((i & 1) ? (r.w[i >> 1] & 0xffff0000u) : (r.w[i >> 1] << 16));
}
template <> __device__ __forceinline__ float raw_elt<__nv_bfloat16, 32>(const Raw<32>& r, int i) {
    return __uint_as_float((i & 1) ? (r.w[i >> 1] & 0xffff0000u) : (r.w[i >> 1] << 16));
}

// A lane's CB contiguous bytes (CH = CB / sizeof(T) channels of one head) of a [*, rowe] tensor of T, kept as raw
// 32-bit words.
template <typename T, int CB> struct Chunk {
    static constexpr int CH = CB / (int)sizeof(T), NW = CB / 4, NP = CB / 16;
    uint32_t w[NW];
    __device__ __forceinline__ void load_global(const T* base, size_t elt, bool pred) {
        if constexpr (CB >= 32) {
#pragma unroll
            for (int t = 0; t < CB / 32; ++t) {
                const Raw<32> r = ldg_raw<32>(reinterpret_cast<const char*>(base + elt) + 32 * t, pred);
#pragma unroll
                for (int i = 0; i < 8; ++i) w[8 * t + i] = r.w[i];
            }
        } else {
            const Raw<16> r = ldg_raw<16>(base + elt, pred);
#pragma unroll
            for (int i = 0; i < 4; ++i) w[i] = r.w[i];
        }
    }
    __device__ __forceinline__ float get(int c) const {
        if constexpr (sizeof(T) == 4) return __uint_as_float(w[c]);
        else return __uint_as_float((c & 1) ? (w[c >> 1] & 0xffff0000u) : (w[c >> 1] << 16));
    }
    __device__ __forceinline__ void to_float(float (&o)[CH]) const {
#pragma unroll
        for (int c = 0; c < CH; ++c) o[c] = get(c);
    }
};

// <a, b> over the lane's channels: fp32 accumulation of exact products (bf16: FHFMA on packed halves)
template <typename T, int CB> __device__ __forceinline__ float dot(const Chunk<T, CB>& a, const Chunk<T, CB>& b) {
    float s0, s1;
    if constexpr (sizeof(T) == 4) {
        mul2v(s0, s1, __uint_as_float(a.w[0]), __uint_as_float(a.w[1]), __uint_as_float(b.w[0]), __uint_as_float(b.w[1]));
#pragma unroll
        for (int i = 2; i < CB / 4; i += 2)
            fma2v(s0, s1, __uint_as_float(a.w[i]), __uint_as_float(a.w[i + 1]), __uint_as_float(b.w[i]), __uint_as_float(b.w[i + 1]));
    } else {
        mul_bf16x2(a.w[0], b.w[0], s0, s1);
#pragma unroll
        for (int i = 1; i < CB / 4; ++i) fma_bf16x2(a.w[i], b.w[i], s0, s1);
    }
    return s0 + s1;
}
// z[c] = x[c] + chunk[c]  (bf16: FHADD on packed halves)
template <typename T, int CB> __device__ __forceinline__ void add_chunk(const Chunk<T, CB>& a, const float (&x)[CB / (int)sizeof(T)],
                                                                         float (&z)[CB / (int)sizeof(T)]) {
    if constexpr (sizeof(T) == 4) {
#pragma unroll
        for (int c = 0; c < CB / 4; ++c) z[c] = x[c] + __uint_as_float(a.w[c]);
    } else {
#pragma unroll
        for (int i = 0; i < CB / 4; ++i) add_bf16x2(a.w[i], x[2 * i], x[2 * i + 1], z[2 * i], z[2 * i + 1]);
    }
}

// CH contiguous fp32 values (a, gradients): plain 128-bit accesses
template <int CH> __device__ __forceinline__ void load_f32(const float* base, size_t elt, bool pred, float (&o)[CH]) {
#pragma unroll
    for (int i = 0; i < CH; i += 4) {
        float4 r = make_float4(0.f, 0.f, 0.f, 0.f);
        if (pred) r = __ldg(reinterpret_cast<const float4*>(base + elt + i));
        o[i] = r.x; o[i + 1] = r.y; o[i + 2] = r.z; o[i + 3] = r.w;
    }
}
// 256-bit store (STG.E.256, sm_100): halves the L1 wavefronts of the row-strided output / gradient stores
__device__ __forceinline__ void stg256(void* p, uint32_t a, uint32_t b, uint32_t c, uint32_t d, uint32_t e, uint32_t f,
                                       uint32_t g, uint32_t h) {
    asm volatile("st.global.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(a), "r"(b), "r"(c), "r"(d), "r"(e),
                 "r"(f), "r"(g), "r"(h) : "memory");
}
template <int CH> __device__ __forceinline__ void store_f32(float* base, size_t elt, const float (&v)[CH]) {
    if constexpr (CH % 8 == 0) {
#pragma unroll
        for (int i = 0; i < CH; i += 8)
            stg256(base + elt + i, __float_as_uint(v[i]), __float_as_uint(v[i + 1]), __float_as_uint(v[i + 2]),
                   __float_as_uint(v[i + 3]), __float_as_uint(v[i + 4]), __float_as_uint(v[i + 5]),
                   __float_as_uint(v[i + 6]), __float_as_uint(v[i + 7]));
    } else {
#pragma unroll
        for (int i = 0; i < CH; i += 4)
            *reinterpret_cast<float4*>(base + elt + i) = make_float4(v[i], v[i + 1], v[i + 2], v[i + 3]);
    }
}
// store CH values in the feature dtype (bf16: round-to-nearest-even)
template <int CH> __device__ __forceinline__ void store_feat(float* base, size_t elt, const float (&v)[CH]) {
    store_f32<CH>(base, elt, v);
}
template <int CH> __device__ __forceinline__ void store_feat(__nv_bfloat16* base, size_t elt, const float (&v)[CH]) {
    uint32_t w[CH / 2];
#pragma unroll
    for (int j = 0; j < CH / 2; ++j) {
        __nv_bfloat162 b = __floats2bfloat162_rn(v[2 * j], v[2 * j + 1]);
        w[j] = *reinterpret_cast<uint32_t*>(&b);
    }
    if constexpr (CH % 16 == 0) {
#pragma unroll
        for (int i = 0; i < CH / 2; i += 8)
            stg256(base + elt + 2 * i, w[i], w[i + 1], w[i + 2], w[i + 3], w[i + 4], w[i + 5], w[i + 6], w[i + 7]);
    } else {
#pragma unroll
        for (int i = 0; i < CH / 2; i += 4)
            *reinterpret_cast<uint4*>(base + elt + 2 * i) = make_uint4(w[i], w[i + 1], w[i + 2], w[i + 3]);
    }
}

// lane geometry inside a group
template <int G> struct Geo {
    int eoff;    // element offset of this lane's channels inside a feature row
    int hd;      // head of this lane
    bool act;    // lane holds channels (the row need not fill the group)
    bool lead;   // first lane of its head (writes per-head scalars)
    int lpl;     // lanes per head
    __device__ __forceinline__ void init(const Shape& sh, int lane) {
        const int gl = lane & (G - 1);
        lpl = sh.lpl;
        act = gl < sh.lanes;
        eoff = gl * sh.ch;
        hd = gl >> sh.lpl_log2;
        lead = act && ((gl & (sh.lpl - 1)) == 0);
    }
};

// sum x[i] over the LPL lanes of a head (all 32 lanes must call; lpl is warp-uniform)
template <int N> __device__ __forceinline__ void head_reduce(float (&x)[N], int lpl) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        if (lpl > o) {
#pragma unroll
            for (int i = 0; i < N; ++i) x[i] += __shfl_xor_sync(0xffffffffu, x[i], o);
        }
    }
}

template <int NA, int NS, int CH> struct State {
    float acc[NA][CH];
    float sc[NS > 0 ? NS : 1];
    float m;  // running max in the log2 domain (softmax passes only)
    __device__ __forceinline__ void reset() {
#pragma unroll
        for (int a = 0; a < NA; ++a)
#pragma unroll
            for (int c = 0; c < CH; ++c) acc[a][c] = 0.f;
#pragma unroll
        for (int s = 0; s < (NS > 0 ? NS : 1); ++s) sc[s] = 0.f;
        m = -INFINITY;
    }
};

// number of floats of a serialised state: [NA][rowe] accumulators, [NS][H] scalars, [H] max (softmax)
template <class Op> __host__ __device__ inline int state_floats(const Shape& sh) {
    return Op::NA * sh.rowe + (Op::NS + (Op::SOFTMAX ? 1 : 0)) * sh.H;
}

}  // namespace gnn
