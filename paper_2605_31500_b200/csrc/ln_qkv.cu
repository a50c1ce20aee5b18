// ln_qkv.cu - row f4: the rest of the block the paper timed in front of the Graph Transformer attention
// ("layer normalization, QKV projection, and the attention mechanism itself"): LayerNorm fused into the
// A-operand staging of a tcgen05 GEMM that writes Q, K, V.
//
//   y[i, :] = (x[i, :] - mean_i) / sqrt(var_i + eps) * gamma + beta        (biased variance over the C features)
//   [Q | K | V][i, :] = y[i, :] W^T + bias,   W = [W_Q; W_K; W_V] of shape [3*H*d, C]
//
// The paper runs these as stock PyTorch ops (LayerNorm kernel, cuBLAS GEMM: one write and one read of the normalised
// activations in HBM).  Here a tile of 128 rows is fetched raw by TMA straight into the 128-byte-swizzled K-major
// shared-memory tile the tensor core reads, normalised IN PLACE (two lanes per row keep their half row in registers:
// one shared-memory read and one write per element, no shuffle chains) - the normalised activations never touch HBM -
// and multiplied with the weights, which stream through a TMA ring of 16 KB stages (128 outputs x 64 channels);
// tcgen05.mma 128 x 128 x 16 into 128-column TMEM accumulators; eight epilogue warps (two per TMEM lane quarter, one
// 64-column half each) drain a finished accumulator (tcgen05.ld, + bias, bf16, swizzled staging buffer, TMA store)
// while the MMA warp fills the next one.  Two kernels:
//   C <= 256  ln_qkv_persist_kernel: persistent CTAs (608 threads: 8 epilogue warps, weight-TMA / MMA / x-TMA warps, 8
//             LayerNorm warps) with TWO A tiles, so the x tile of tile t + 1 lands and is normalised while tile t is
//             multiplied and drained; output staging in 128-byte rows (one TMA store per chunk and warp).
//             PAIR form (default when 3 H d is a multiple of 256): clusters of two CTAs on an SM pair; the rank-0 CTA issues
//             tcgen05.mma.cta_group::2 256 x 256 x 16 - each CTA contributes its own 128-row A tile and 128 of the 256
//             weight rows of a stage (TMA .cta_group::2 completing on rank 0's barrier), results land in each CTA's own
//             TMEM (two 256-column accumulators); commits are multicast to both CTAs' barriers and the peer's warps
//             report to rank 0's barriers through the cluster.  Half the operand bytes per flop of the single-CTA form
//             (A and B are read from shared memory once per 256 outputs / 256 rows) - which is what the single-CTA form
//             is bound by - and half the weight bytes per SM.
//   C <= 512  ln_qkv_kernel: one CTA per tile (the 128 KB A tile leaves no room for a second one), two accumulators,
//             output staging in 32-byte rows.
// Measurements and what limits each form: profiles/r02_ncu_ln_qkv.md.
#include <cuda.h>
#include <cuda_bf16.h>

#include "internal.h"
#include "kernels.cuh"
#include "tc_common.cuh"

namespace gnn {
namespace {
using namespace tc;

constexpr int kRows = 128;          // rows per CTA = MMA M
constexpr int kNC = 128;            // output columns per chunk = MMA N
constexpr int kStage = 16384;       // bytes of a weight stage / of a 64-channel half tile of A
constexpr int kWorkWarps = 8;        // warps 0-7: LayerNorm + epilogue (two warps per TMEM lane quarter, one column half each)
constexpr int kThreads = 320;       // + warp 8: TMA, warp 9: MMA
constexpr int kOut = 1024;          // bytes of an output staging buffer: 32 rows x 16 bf16 columns (two per worker warp)
constexpr int kBars = 256;          // mbarriers + TMEM slot, in front of the 1024-byte aligned tiles

struct LnQkvParams {
    const __nv_bfloat16* x;
    const float *gamma, *beta, *bias;
    __nv_bfloat16 *q, *k, *v;
    int n, C, R;                    // rows, input features, H * d
    float eps;
    int n_stages;
};

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void add2(float& a0, float& a1, float x0, float x1) {      // (a0, a1) += (x0, x1), one FADD2
    asm("{\n .reg .b64 xx, cc;\n mov.b64 xx, {%2, %3};\n mov.b64 cc, {%0, %1};\n add.rn.f32x2 cc, cc, xx;\n mov.b64 {%0, %1}, cc;\n}"
        : "+f"(a0), "+f"(a1) : "f"(x0), "f"(x1));
}

// LayerNorm of warp `warp`'s 16 rows of the raw x tile in sA (SWIZZLE_128B half tiles of 64 channels), IN PLACE.
// Two lanes per row: lane l owns row 16 warp + (l & 15), half tiles (l >> 4) KH .. + KH - 1 (KH = 2 for C <= 256, 4 for
// C <= 512), i.e. up to 128 / 256 channels, which it keeps as raw bf16 pairs in registers (one smem read, one smem
// write per element).  No shuffle chains: every lane runs long independent sums and meets its partner (lane ^ 16) twice
// (sum, sum of centred squares).  bf16 halves enter the fp32 sums directly (FHADD), squares / scale / shift are packed
// (FFMA2 / FMUL2); gamma / beta come from L1 as broadcast 16-byte loads.  Rows past n become zeros.
template <int KH>
__device__ __forceinline__ void ln_rows(uint8_t* sA, const LnQkvParams& p, int row0, int warp, int lane) {
    const int KC = p.C / 64;
    const int r = warp * 16 + (lane & 15), kk0 = (lane >> 4) * KH;
    const uint32_t rbase = (uint32_t)((r >> 3) * 1024 + (r & 7) * 128), rx = (uint32_t)(r & 7);
    uint4 raw[KH][8];
    float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
#pragma unroll
    for (int k = 0; k < KH; ++k) {
        const bool on = kk0 + k < KC;
#pragma unroll
        for (int cc = 0; cc < 8; ++cc) {
            raw[k][cc] = make_uint4(0, 0, 0, 0);
            if (on) raw[k][cc] = *reinterpret_cast<const uint4*>(sA + (kk0 + k) * kStage + rbase + (((uint32_t)cc ^ rx) << 4));
            add_bf16x2(raw[k][cc].x, s0, s1, s0, s1);
            add_bf16x2(raw[k][cc].y, s2, s3, s2, s3);
            add_bf16x2(raw[k][cc].z, s0, s1, s0, s1);
            add_bf16x2(raw[k][cc].w, s2, s3, s2, s3);
        }
    }
    float sum = (s0 + s1) + (s2 + s3);
    sum += __shfl_xor_sync(0xffffffffu, sum, 16);
    const float inv_c = 1.f / (float)p.C;
    const float nmean = -sum * inv_c;
    float q0 = 0.f, q1 = 0.f, q2 = 0.f, q3 = 0.f;
#pragma unroll
    for (int k = 0; k < KH; ++k) {
        const float nm = kk0 + k < KC ? nmean : 0.f;          // half tiles past C hold zeros and stay zero
#pragma unroll
        for (int cc = 0; cc < 8; ++cc) {
            const uint32_t w[4] = {raw[k][cc].x, raw[k][cc].y, raw[k][cc].z, raw[k][cc].w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                float a, b;
                add_bf16x2(w[i], nm, nm, a, b);
                if (i & 1) fma2v(q2, q3, a, b, a, b);
                else fma2v(q0, q1, a, b, a, b);
            }
        }
    }
    float ss = (q0 + q1) + (q2 + q3);
    ss += __shfl_xor_sync(0xffffffffu, ss, 16);
    const bool rv = row0 + r < p.n;
    const float rstd = rv ? 1.f / sqrtf(ss * inv_c + p.eps) : 0.f;
#pragma unroll
    for (int k = 0; k < KH; ++k) {
        if (kk0 + k < KC) {
#pragma unroll
            for (int cc = 0; cc < 8; ++cc) {
                const int ch = (kk0 + k) * 64 + cc * 8;
                const float4 g0 = __ldg(reinterpret_cast<const float4*>(p.gamma + ch)), g1 = __ldg(reinterpret_cast<const float4*>(p.gamma + ch + 4));
                float4 b0 = __ldg(reinterpret_cast<const float4*>(p.beta + ch)), b1 = __ldg(reinterpret_cast<const float4*>(p.beta + ch + 4));
                if (!rv) { b0 = make_float4(0.f, 0.f, 0.f, 0.f); b1 = b0; }
                const uint32_t w[4] = {raw[k][cc].x, raw[k][cc].y, raw[k][cc].z, raw[k][cc].w};
                const float gg[8] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w};
                float zz[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
                uint32_t o[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    float y0, y1;
                    add_bf16x2(w[i], nmean, nmean, y0, y1);
                    mul2(y0, y1, rstd);
                    fma2v(zz[2 * i], zz[2 * i + 1], y0, y1, gg[2 * i], gg[2 * i + 1]);
                    const __nv_bfloat162 yb = __floats2bfloat162_rn(zz[2 * i], zz[2 * i + 1]);
                    o[i] = *reinterpret_cast<const uint32_t*>(&yb);
                }
                *reinterpret_cast<uint4*>(sA + (kk0 + k) * kStage + rbase + (((uint32_t)cc ^ rx) << 4)) = make_uint4(o[0], o[1], o[2], o[3]);
            }
        }
    }
}

// The same for rows too wide to keep in registers (C > 256: up to 256 channels per lane): three sweeps over the lane's
// half tiles - sum, centred squares, normalise + write - re-reading shared memory, 8 chunks (one half tile) live at a time.
__device__ __forceinline__ void ln_rows_stream(uint8_t* sA, const LnQkvParams& p, int row0, int warp, int lane) {
    const int KC = p.C / 64, KH = (KC + 1) / 2;
    const int r = warp * 16 + (lane & 15), kk0 = (lane >> 4) * KH, kk1 = min(KC, kk0 + KH);
    const uint32_t rbase = (uint32_t)((r >> 3) * 1024 + (r & 7) * 128), rx = (uint32_t)(r & 7);
    float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
#pragma unroll 1
    for (int kk = kk0; kk < kk1; ++kk) {
#pragma unroll
        for (int cc = 0; cc < 8; ++cc) {
            const uint4 w = *reinterpret_cast<const uint4*>(sA + kk * kStage + rbase + (((uint32_t)cc ^ rx) << 4));
            add_bf16x2(w.x, s0, s1, s0, s1); add_bf16x2(w.y, s2, s3, s2, s3);
            add_bf16x2(w.z, s0, s1, s0, s1); add_bf16x2(w.w, s2, s3, s2, s3);
        }
    }
    float sum = (s0 + s1) + (s2 + s3);
    sum += __shfl_xor_sync(0xffffffffu, sum, 16);
    const float inv_c = 1.f / (float)p.C;
    const float nmean = -sum * inv_c;
    float q0 = 0.f, q1 = 0.f, q2 = 0.f, q3 = 0.f;
#pragma unroll 1
    for (int kk = kk0; kk < kk1; ++kk) {
#pragma unroll
        for (int cc = 0; cc < 8; ++cc) {
            const uint4 w4 = *reinterpret_cast<const uint4*>(sA + kk * kStage + rbase + (((uint32_t)cc ^ rx) << 4));
            const uint32_t w[4] = {w4.x, w4.y, w4.z, w4.w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                float a, b;
                add_bf16x2(w[i], nmean, nmean, a, b);
                if (i & 1) fma2v(q2, q3, a, b, a, b);
                else fma2v(q0, q1, a, b, a, b);
            }
        }
    }
    float ss = (q0 + q1) + (q2 + q3);
    ss += __shfl_xor_sync(0xffffffffu, ss, 16);
    const bool rv = row0 + r < p.n;
    const float rstd = rv ? 1.f / sqrtf(ss * inv_c + p.eps) : 0.f;
#pragma unroll 1
    for (int kk = kk0; kk < kk1; ++kk) {
#pragma unroll
        for (int cc = 0; cc < 8; ++cc) {
            const int ch = kk * 64 + cc * 8;
            uint8_t* at = sA + kk * kStage + rbase + (((uint32_t)cc ^ rx) << 4);
            const uint4 w4 = *reinterpret_cast<const uint4*>(at);
            const float4 g0 = __ldg(reinterpret_cast<const float4*>(p.gamma + ch)), g1 = __ldg(reinterpret_cast<const float4*>(p.gamma + ch + 4));
            float4 b0 = __ldg(reinterpret_cast<const float4*>(p.beta + ch)), b1 = __ldg(reinterpret_cast<const float4*>(p.beta + ch + 4));
            if (!rv) { b0 = make_float4(0.f, 0.f, 0.f, 0.f); b1 = b0; }
            const uint32_t w[4] = {w4.x, w4.y, w4.z, w4.w};
            const float gg[8] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w};
            float zz[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
            uint32_t o[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                float y0, y1;
                add_bf16x2(w[i], nmean, nmean, y0, y1);
                mul2(y0, y1, rstd);
                fma2v(zz[2 * i], zz[2 * i + 1], y0, y1, gg[2 * i], gg[2 * i + 1]);
                const __nv_bfloat162 yb = __floats2bfloat162_rn(zz[2 * i], zz[2 * i + 1]);
                o[i] = *reinterpret_cast<const uint32_t*>(&yb);
            }
            *reinterpret_cast<uint4*>(at) = make_uint4(o[0], o[1], o[2], o[3]);
        }
    }
}

// epilogue state of one worker warp: warp w drains TMEM lanes 32 (w & 3) .. +31 (tile rows) of column half w >> 2 of every
// accumulator: accumulator -> + bias -> bf16 -> 32-row x 16-column staging buffer (the layout TMA's 32-byte swizzle expects)
// -> one TMA store per buffer (rows past n are clipped by the unit); the warp's two staging buffers alternate
template <int W>       // W = 16: two 1 KB buffers per warp, 32-byte rows (SWIZZLE_32B maps), four stores per chunk;
struct Epi {           // W = 64: one 4 KB buffer per warp, 128-byte rows (SWIZZLE_128B maps), one store per chunk
    static constexpr int kBytes = W == 16 ? 2 * kOut : 4096;   // staging bytes per warp
    float4 bb[8];          // bias of the next 32-column pass (prefetched one pass ahead)
    uint8_t* stage;
    uint32_t lane_off, my, sw;
    int q4, hsel, lane, n_st;
    bool to_leader;        // CTA pairs: "drained" is the barrier of the pair's rank-0 CTA (which issues the MMAs)
    __device__ __forceinline__ void init(const LnQkvParams& p, uint8_t* sT, int warp, int lane_, bool to_leader_ = false) {
        q4 = warp & 3; hsel = warp >> 2; lane = lane_; n_st = 0; to_leader = to_leader_;
        lane_off = (uint32_t)(q4 * 32) << 16;
        stage = sT + warp * kBytes;
        if (W == 16) { my = (uint32_t)lane * 32; sw = ((uint32_t)(lane >> 2) & 1u) << 4; }
        else { my = (uint32_t)lane * 128; sw = (uint32_t)lane & 7u; }
        if (p.bias) {
#pragma unroll
            for (int i = 0; i < 8; ++i) bb[i] = __ldg(reinterpret_cast<const float4*>(p.bias + 64 * hsel) + i);
        }
    }
    // output chunk c (columns c * 128 ..) of the tile at row0 from the complete accumulator at TMEM column t_acc; arrives
    // on `drained` after the last TMEM read
    __device__ __forceinline__ void chunk(const LnQkvParams& p, uint32_t t_acc, uint64_t* drained, int c, int n_chunks, int row0,
                                          const CUtensorMap* tmq, const CUtensorMap* tmk, const CUtensorMap* tmv,
                                          bool last = true) {
        const int col0 = c * kNC + 64 * hsel;
        const int t = col0 / p.R, off = col0 - t * p.R;
        const CUtensorMap* tmo = t == 0 ? tmq : (t == 1 ? tmk : tmv);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll 1
        for (int c0 = 0; c0 < 64; c0 += 32) {
            float t32[32];
            if (W == 64 && c0 == 0 && n_st > 0) {
                // the wait for the staging buffer (the previous chunk's TMA store reading it) hides under the TMEM read
                uint32_t r32[32];
                tmem_ld32_issue(t_acc + lane_off + 64 * hsel, r32);
                if (lane == 0) tma_store_wait_read<0>();
                __syncwarp();
                tmem_ld_wait();
#pragma unroll
                for (int i = 0; i < 32; ++i) t32[i] = __uint_as_float(r32[i]);
            } else {
                tmem_ld32(t_acc + lane_off + 64 * hsel + c0, t32);
            }
            if (c0 == 32) {                                 // last read of this accumulator half: hand it back to the MMA warp
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncwarp();
                if (lane == 0 && last) {
                    if (to_leader) mbar_arrive_cluster_relaxed(drained, 0);
                    else mbar_arrive(drained);
                }
            }
            if (p.bias) {
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    add2(t32[4 * i], t32[4 * i + 1], bb[i].x, bb[i].y);
                    add2(t32[4 * i + 2], t32[4 * i + 3], bb[i].z, bb[i].w);
                }
                // the next pass's bias values travel while this pass is packed and stored
                const int nxt = c0 == 0 ? col0 + 32 : ((c + 1) % n_chunks) * kNC + 64 * hsel;
#pragma unroll
                for (int i = 0; i < 8; ++i) bb[i] = __ldg(reinterpret_cast<const float4*>(p.bias + nxt) + i);
            }
            if constexpr (W == 16) {
    #pragma unroll
                for (int g16 = 0; g16 < 2; ++g16, ++n_st) {
                    uint8_t* buf = stage + (n_st & 1) * kOut;
                    if (n_st >= 2) {                            // the store issued from this buffer two groups ago has read it
                        if (lane == 0) tma_store_wait_read<1>();
                        __syncwarp();
                    }
                    uint32_t o[8];
    #pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const __nv_bfloat162 yb = __floats2bfloat162_rn(t32[16 * g16 + 2 * i], t32[16 * g16 + 2 * i + 1]);
                        o[i] = *reinterpret_cast<const uint32_t*>(&yb);
                    }
                    *reinterpret_cast<uint4*>(buf + my + sw) = make_uint4(o[0], o[1], o[2], o[3]);
                    *reinterpret_cast<uint4*>(buf + my + (sw ^ 16u)) = make_uint4(o[4], o[5], o[6], o[7]);
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    __syncwarp();
                    if (lane == 0) {
                        tma_store_2d(tmo, off + c0 + 16 * g16, row0 + 32 * q4, buf);
                        tma_store_commit();
                    }
                }
            } else {
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    uint32_t o[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const __nv_bfloat162 yb = __floats2bfloat162_rn(t32[8 * j + 2 * i], t32[8 * j + 2 * i + 1]);
                        o[i] = *reinterpret_cast<const uint32_t*>(&yb);
                    }
                    *reinterpret_cast<uint4*>(stage + my + ((((uint32_t)(c0 >> 3) + j) ^ sw) << 4)) = make_uint4(o[0], o[1], o[2], o[3]);
                }
                if (c0 == 32) {
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    __syncwarp();
                    if (lane == 0) {
                        tma_store_2d(tmo, off, row0 + 32 * q4, stage);
                        tma_store_commit();
                    }
                    ++n_st;
                }
            }
        }
    }
};

template <int NJ>     // 1: C <= 256 (two CTAs per SM), 2: C <= 512 (one CTA per SM)
__global__ void __launch_bounds__(kThreads, 3 - NJ)
ln_qkv_kernel(const __grid_constant__ CUtensorMap tmx, const __grid_constant__ CUtensorMap tmw,
              const __grid_constant__ CUtensorMap tmq, const __grid_constant__ CUtensorMap tmk,
              const __grid_constant__ CUtensorMap tmv, const LnQkvParams p) {
    extern __shared__ uint8_t smem_raw[];
    // [barriers, kBars bytes][pad to 1024][A: KC half tiles][NS weight stages][16 output staging buffers]
    uint8_t* smem = smem_raw + kBars + ((1024u - ((smem_u32(smem_raw) + kBars) & 1023u)) & 1023u);
    const int KC = p.C / 64, NS = p.n_stages;
    uint8_t* sA = smem;                                   // [KC] half tiles, 128 rows x 128 bytes, SWIZZLE_128B
    uint8_t* sB = sA + KC * kStage;                       // [NS] weight stages
    uint8_t* sT = sB + NS * kStage;                       // [kWorkWarps][2] staging buffers, 32 rows x 32 bytes, SWIZZLE_32B
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw);   // [NS] TMA landed
    uint64_t* empty = full + 8;                           // [NS] stage consumed (tcgen05.commit)
    uint64_t* tfull = empty + 8;                          // [2] accumulator complete
    uint64_t* tempty = tfull + 2;                         // [2] accumulator drained
    uint64_t* xfull = tempty + 2;                         // raw x tile landed
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(xfull + 1);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int row0 = blockIdx.x * kRows;
    {   // the host sizes the allocation for a 1024-byte aligned base (pad + barriers = 1024); refuse anything else loudly
        uint32_t dyn;
        asm("mov.u32 %0, %%dynamic_smem_size;" : "=r"(dyn));
        if ((uint32_t)(sT + kWorkWarps * 2 * kOut - smem_raw) > dyn) __trap();
    }
    const int n_chunks = 3 * p.R / kNC;

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(tfull + b, 1); mbar_init(tempty + b, kWorkWarps); }
        mbar_init(xfull, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 9) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 256;" ::"r"(smem_u32(tmem_slot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;

    if (warp == 8) {
        // ===== TMA producer: weight stage i = (chunk c, channel block kk) -> ring slot i % NS
        // (the first NS stages go out now and overlap the LayerNorm; the rest after the A tile barrier below, because
        // their slots are only released by the MMA warp, which starts behind that barrier)
        if (lane == 0) {
            // the raw x tile lands in the A tile's own layout (TMA applies the 128-byte swizzle); it is normalised in place
            mbar_expect_tx(xfull, KC * kStage);
            for (int kk = 0; kk < KC; ++kk) tma_load_2d(sA + kk * kStage, &tmx, kk * 64, row0, xfull);
            const int items = n_chunks * KC;
            for (int i = 0; i < items && i < NS; ++i) {
                mbar_expect_tx(full + i, kStage);
                tma_load_2d(sB + i * kStage, &tmw, (i % KC) * 64, (i / KC) * kNC, full + i);
            }
        }
    } else if (warp < kWorkWarps) {
        // ===== LayerNorm of this warp's 16 rows, in place in the A tile
        mbar_wait(xfull, 0);
        ln_rows<2 * NJ>(sA, p, row0, warp, lane);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();   // the A tile is complete and visible to the tensor core

    if (warp == 8) {
        if (lane == 0) {
            const int items = n_chunks * KC;
            for (int i = NS; i < items; ++i) {
                const int s = i % NS, c = i / KC, kk = i % KC;
                mbar_wait(empty + s, (uint32_t)((i / NS) & 1) ^ 1u);
                mbar_expect_tx(full + s, kStage);
                tma_load_2d(sB + s * kStage, &tmw, kk * 64, c * kNC, full + s);
            }
        }
    } else if (warp == 9) {
        // ===== MMA issuer
        if (lane == 0) {
            constexpr uint32_t kIdesc = make_idesc(kRows, kNC, false);
            int i = 0;
            for (int c = 0; c < n_chunks; ++c) {
                const int bsel = c & 1;
                mbar_wait(tempty + bsel, (uint32_t)((c >> 1) & 1) ^ 1u);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                for (int kk = 0; kk < KC; ++kk, ++i) {
                    const int s = i % NS;
                    mbar_wait(full + s, (uint32_t)((i / NS) & 1));
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks)
                        umma(tmem + bsel * kNC, make_desc_sw128(smem_u32(sA + kk * kStage) + ks * 32, 1024),
                             make_desc_sw128(smem_u32(sB + s * kStage) + ks * 32, 1024), kIdesc, (kk | ks) > 0);
                    umma_commit(empty + s);
                }
                umma_commit(tfull + bsel);
            }
        }
    } else if (warp < kWorkWarps) {
        // ===== epilogue (Epi)
        Epi<16> ep;
        ep.init(p, sT, warp, lane);
        for (int c = 0; c < n_chunks; ++c) {
            mbar_wait(tfull + (c & 1), (uint32_t)((c >> 1) & 1));
            ep.chunk(p, tmem + (c & 1) * kNC, tempty + (c & 1), c, n_chunks, row0, &tmq, &tmk, &tmv);
        }
        if (lane == 0) tma_store_wait<0>();
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 9) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 256;" ::"r"(tmem) : "memory");
}

// ---- persistent variant for C <= 256: one CTA per SM walks tiles blockIdx.x, + gridDim.x, ... with TWO A tiles, so that
// the raw x tile of tile t + 1 lands and is normalised while the tensor core works on tile t, four TMEM accumulators
// (all 512 columns) so that the MMA warp runs ahead of the epilogue by up to four output chunks, and a weight ring of
// all the shared memory that is left.  Roles: warps 0-7 LayerNorm(t + 1) then epilogue(t); warp 8 weight ring (TMA);
// warp 9 MMA issue; warp 10 x tiles (TMA).  Barriers: xfull[b] (x tile landed in A[b]), aready[b] (A[b] normalised, 8
// warp arrivals), afree[b] (tcgen05.commit after the last product of the tile in A[b]), full / empty (weight ring),
// tfull / tempty (accumulators).
constexpr int kPThreads = 608;       // warps 0-7 epilogue, 8 weight TMA, 9 MMA, 10 x TMA, 11-18 LayerNorm
constexpr int kLnWarp0 = 11;
constexpr int kAcc = 4;
template <bool PAIR, int NBUF>   // NBUF: A tiles per CTA (2 for C <= 256; 1 for C <= 512: no room for a second);
                                 // PAIR: clusters of two CTAs; one tcgen05.mma.cta_group::2 (M = 256) multiplies both CTAs' tiles against
                       // a weight stage of which each CTA loads one half: half the weight bytes per SM, twice the stages
__global__ void __launch_bounds__(kPThreads, 1)
ln_qkv_persist_kernel(const __grid_constant__ CUtensorMap tmx, const __grid_constant__ CUtensorMap tmw,
                      const __grid_constant__ CUtensorMap tmq, const __grid_constant__ CUtensorMap tmk,
                      const __grid_constant__ CUtensorMap tmv, const LnQkvParams p) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + kBars + ((1024u - ((smem_u32(smem_raw) + kBars) & 1023u)) & 1023u);
    const int KC = p.C / 64, NS = p.n_stages;
    uint8_t* sA = smem;                                   // [2][KC] half tiles
    // PAIR: accumulators of 256 columns (MMA 256 x 256 x 16 over the pair): every A byte read from shared memory feeds 256
    // outputs and every CTA loads 128 of a stage's 256 weight rows - half the operand bytes per flop of the single-CTA form
    constexpr int NCc = PAIR ? 256 : kNC;                 // output columns per accumulator / weight stage
    constexpr int NACC = 512 / NCc;                       // accumulators in the 512 TMEM columns
    constexpr int kW = kStage;                            // bytes of this CTA's part of a weight stage (128 rows x 64 channels)
    uint8_t* sB = sA + NBUF * KC * kStage;                // [NS] weight stages
    uint8_t* sT = sB + NS * kW;                           // [kWorkWarps] staging buffers of 32 rows x 128 bytes
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw);
    uint64_t* empty = full + 8;
    uint64_t* tfull = empty + 8;                          // [kAcc]
    uint64_t* tempty = tfull + kAcc;                      // [kAcc]
    uint64_t* xfull = tempty + kAcc;                      // [2]
    uint64_t* aready = xfull + 2;                         // [2]
    uint64_t* afree = aready + 2;                         // [2]
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(afree + 2);
    static_assert((8 + 8 + 2 * kAcc + 6) * 8 + 4 <= kBars, "barrier block");

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    {
        uint32_t dyn;
        asm("mov.u32 %0, %%dynamic_smem_size;" : "=r"(dyn));
        if ((uint32_t)(sT + kWorkWarps * Epi<64>::kBytes - smem_raw) > dyn) __trap();
    }
    const int n_chunks = 3 * p.R / NCc;
    const int tiles = (p.n + kRows - 1) / kRows;
    // walkers: single CTAs over the tiles, or CTA pairs over pairs of consecutive tiles (rank r takes tile 2 * pair + r; both
    // CTAs of a pair run the same number of iterations - a tile past the end is skipped where it touches memory)
    const uint32_t rank = PAIR ? cluster_ctarank() : 0u;
    const int nwalk = PAIR ? (int)gridDim.x / 2 : (int)gridDim.x, me = PAIR ? (int)blockIdx.x / 2 : (int)blockIdx.x;
    const int nunits = PAIR ? (tiles + 1) / 2 : tiles;
    const int nlt = me < nunits ? (nunits - 1 - me) / nwalk + 1 : 0;
    auto tile_row0 = [&](int lt) { return ((me + lt * nwalk) * (PAIR ? 2 : 1) + (int)rank) * kRows; };

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); }
        constexpr int kArr = kWorkWarps * (PAIR ? 2 : 1);   // worker-warp arrivals: both CTAs of a pair report to rank 0
        for (int b = 0; b < NACC; ++b) { mbar_init(tfull + b, 1); mbar_init(tempty + b, kArr); }
        for (int b = 0; b < 2; ++b) { mbar_init(xfull + b, 1); mbar_init(aready + b, kArr); mbar_init(afree + b, 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 9) {
        if (PAIR) {
            asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
        } else {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (PAIR) cluster_sync_all();     // the peer's barriers exist before anything signals them
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;

    if (warp == 10) {
        // ===== x tiles: tile lt -> A[lt & 1] once the products of tile lt - 2 have left it
        if (lane == 0) {
            for (int lt = 0; lt < nlt; ++lt) {
                const int b = lt % NBUF;
                if (tile_row0(lt) >= p.n) continue;          // (pairs) the odd tile past the end: nothing to load
                mbar_wait(afree + b, (uint32_t)((lt / NBUF) & 1) ^ 1u);
                mbar_expect_tx(xfull + b, KC * kStage);
                for (int kk = 0; kk < KC; ++kk) tma_load_2d(sA + (b * KC + kk) * kStage, &tmx, kk * 64, tile_row0(lt), xfull + b);
            }
        }
    } else if (warp == 8) {
        // ===== weight ring: item i = (tile, chunk c, channel block kk) -> slot i % NS
        if (lane == 0) {
            const int per_tile = n_chunks * KC, items = nlt * per_tile;
            for (int i = 0; i < items; ++i) {
                const int s = i % NS, j = i % per_tile;
                mbar_wait(empty + s, (uint32_t)((i / NS) & 1) ^ 1u);
                if (!PAIR) {
                    mbar_expect_tx(full + s, kStage);
                    tma_load_2d(sB + s * kW, &tmw, (j % KC) * 64, (j / KC) * NCc, full + s);
                } else {
                    // this CTA's 128 of the stage's 256 weight rows; both halves complete on rank 0's barrier
                    if (rank == 0) mbar_expect_tx(full + s, 2 * kStage);
                    tma_load_2d_pair(sB + s * kW, &tmw, (j % KC) * 64, (j / KC) * NCc + (int)rank * (NCc / 2), full + s);
                }
            }
        }
    } else if (warp == 9) {
        // ===== MMA issuer (pairs: rank 0 only)
        if (lane == 0 && rank == 0) {
            constexpr uint32_t kIdesc = make_idesc(PAIR ? 2 * kRows : kRows, NCc, false);
            auto commit = [&](uint64_t* bar) {
                if (PAIR) umma2_commit_mc(bar, (uint16_t)3);
                else umma_commit(bar);
            };
            int i = 0, g = 0;
            for (int lt = 0; lt < nlt; ++lt) {
                const int b = lt % NBUF;
                mbar_wait(aready + b, (uint32_t)((lt / NBUF) & 1));
                for (int c = 0; c < n_chunks; ++c, ++g) {
                    const int acc = g % NACC;
                    mbar_wait(tempty + acc, (uint32_t)((g / NACC) & 1) ^ 1u);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    for (int kk = 0; kk < KC; ++kk, ++i) {
                        const int s = i % NS;
                        mbar_wait(full + s, (uint32_t)((i / NS) & 1));
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                        for (int ks = 0; ks < 4; ++ks) {
                            const uint64_t da = make_desc_sw128(smem_u32(sA + (b * KC + kk) * kStage) + ks * 32, 1024);
                            const uint64_t db = make_desc_sw128(smem_u32(sB + s * kW) + ks * 32, 1024);
                            if (PAIR) umma2(tmem + acc * NCc, da, db, kIdesc, (kk | ks) > 0);
                            else umma(tmem + acc * NCc, da, db, kIdesc, (kk | ks) > 0);
                        }
                        commit(empty + s);
                    }
                    commit(tfull + acc);
                }
                commit(afree + b);
            }
        }
    } else if (warp >= kLnWarp0) {
        // ===== LayerNorm warps: tile lt in A[lt & 1] as soon as its x tile has landed (runs ahead of / under the epilogue)
        for (int lt = 0; lt < nlt; ++lt) {
            const int b = lt % NBUF;
            if (tile_row0(lt) < p.n) {
                mbar_wait(xfull + b, (uint32_t)((lt / NBUF) & 1));
                if (NBUF == 2) ln_rows<2>(sA + b * KC * kStage, p, tile_row0(lt), warp - kLnWarp0, lane);
                else ln_rows_stream(sA + b * KC * kStage, p, tile_row0(lt), warp - kLnWarp0, lane);
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            if (lane == 0) {
                if (PAIR) mbar_arrive_cluster(aready + b, 0);
                else mbar_arrive(aready + b);
            }
        }
    } else if (warp < kWorkWarps) {
        // ===== epilogue warps
        Epi<64> ep;
        ep.init(p, sT, warp, lane, PAIR);
        int g = 0;
        for (int lt = 0; lt < nlt; ++lt) {
            for (int c = 0; c < n_chunks; ++c, ++g) {
                const int acc = g % NACC;
                mbar_wait(tfull + acc, (uint32_t)((g / NACC) & 1));
                if (PAIR) {     // a 256-column accumulator leaves as two 128-column output chunks
                    ep.chunk(p, tmem + acc * NCc, tempty + acc, 2 * c, 2 * n_chunks, tile_row0(lt), &tmq, &tmk, &tmv, false);
                    ep.chunk(p, tmem + acc * NCc + kNC, tempty + acc, 2 * c + 1, 2 * n_chunks, tile_row0(lt), &tmq, &tmk, &tmv);
                } else {
                    ep.chunk(p, tmem + acc * NCc, tempty + acc, c, n_chunks, tile_row0(lt), &tmq, &tmk, &tmv);
                }
            }
        }
        if (lane == 0) tma_store_wait<0>();
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (PAIR) cluster_sync_all();     // no CTA leaves (or frees TMEM) while its peer may still signal it / multiply into it
    if (warp == 9) {
        if (PAIR) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
        else asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
    }
}

}  // namespace
}  // namespace gnn

using namespace gnn;

extern "C" gnn_status_t gnn_ln_qkv_fwd(int32_t n, int32_t c_in, int32_t heads, int32_t head_dim, const void* x,
                                       const float* gamma, const float* beta, float eps, const void* w, const float* bias,
                                       void* q, void* k, void* v, gnn_stream_t stream) {
    const char* who = "gnn_ln_qkv_fwd";
    if (n < 1 || !x || !gamma || !beta || !w || !q || !k || !v) { set_error("%s: n < 1 or NULL pointer argument", who); return GNN_EINVAL; }
    if ((((uintptr_t)x | (uintptr_t)w | (uintptr_t)q | (uintptr_t)k | (uintptr_t)v) & 31) != 0) {
        set_error("%s: x, w, q, k, v must be 32-byte aligned", who);
        return GNN_EINVAL;
    }
    if (!(eps >= 0.f)) { set_error("%s: eps must be >= 0", who); return GNN_EINVAL; }
    const long long R = (long long)heads * head_dim;
    if (heads < 1 || head_dim < 1 || c_in < 64 || c_in > 512 || c_in % 64 != 0 || R % kNC != 0 || R > 8192) {
        set_error("%s: unsupported shape c_in=%d heads=%d head_dim=%d (c_in a multiple of 64 in [64, 512], heads*head_dim a multiple of 128)",
                  who, c_in, heads, head_dim);
        return GNN_EUNSUPPORTED;
    }
    CUtensorMap tmx, tmw, tmq, tmk, tmv;
    if (!tc::encode_row_tile_map(&tmx, x, n, c_in, 64, kRows) || !tc::encode_row_tile_map(&tmw, w, (int)(3 * R), c_in, 64, kNC) ||
        !tc::encode_row_tile_map(&tmq, q, n, (int)R, 16, 32, CU_TENSOR_MAP_SWIZZLE_32B) ||
        !tc::encode_row_tile_map(&tmk, k, n, (int)R, 16, 32, CU_TENSOR_MAP_SWIZZLE_32B) ||
        !tc::encode_row_tile_map(&tmv, v, n, (int)R, 16, 32, CU_TENSOR_MAP_SWIZZLE_32B)) {
        set_error("%s: cuTensorMapEncodeTiled unavailable or failed", who);
        return GNN_ECUDA;
    }
    LnQkvParams p = {};
    p.x = (const __nv_bfloat16*)x; p.gamma = gamma; p.beta = beta; p.bias = bias;
    p.q = (__nv_bfloat16*)q; p.k = (__nv_bfloat16*)k; p.v = (__nv_bfloat16*)v;
    p.n = n; p.C = c_in; p.R = (int)R; p.eps = eps;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    const int tiles = (n + kRows - 1) / kRows;
    int dev = 0, sms = 0;
    e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) { set_error("%s: CUDA error: %s", who, cudaGetErrorString(e)); return GNN_ECUDA; }
    // Forms, in order of preference:
    //   CTA pairs (256 x 256 x 16 MMAs over two SMs) whenever the outputs split into 256-column accumulators - persistent,
    //     two A tiles for C <= 256, one for C <= 512;
    //   single persistent CTAs for C <= 256 (also the fallback if the cluster launch is refused, e.g. a partitioned GPU
    //     without free SM pairs);
    //   one CTA per tile for 256 < C <= 512.
    static const bool no_pair = [] { const char* v = getenv("GNN_LNQKV_NO_PAIR"); return v && atoi(v) != 0; }();
    const bool wide = c_in > 256;
    bool pair = !no_pair && (3 * R) % 256 == 0 && tiles > 1 && sms >= 2;
    bool launched = false;
    while (!wide || pair) {
        const int nbuf = wide ? 1 : 2;
        CUtensorMap oq, ok, ov, tmw_k = tmw;
        if (!tc::encode_row_tile_map(&oq, q, n, (int)R, 64, 32) || !tc::encode_row_tile_map(&ok, k, n, (int)R, 64, 32) ||
            !tc::encode_row_tile_map(&ov, v, n, (int)R, 64, 32) ||      // output boxes of 32 rows x 128 bytes, SWIZZLE_128B
            (pair && !tc::encode_row_tile_map(&tmw_k, w, (int)(3 * R), c_in, 64, 128))) {   // a CTA's 128 of a stage's 256 rows
            set_error("%s: cuTensorMapEncodeTiled unavailable or failed", who);
            return GNN_ECUDA;
        }
        const size_t fixed = (size_t)nbuf * (c_in / 64) * kStage + (size_t)kWorkWarps * 4096 + 1024;
        p.n_stages = (int)((226 * 1024 - fixed) / kStage);
        if (p.n_stages > 8) p.n_stages = 8;
        const size_t smem = fixed + (size_t)p.n_stages * kStage;
        auto kern = wide ? ln_qkv_persist_kernel<true, 1> : (pair ? ln_qkv_persist_kernel<true, 2> : ln_qkv_persist_kernel<false, 2>);
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) {
            const int units = pair ? (tiles + 1) / 2 : tiles, walkers = pair ? sms / 2 : sms;
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3((units < walkers ? units : walkers) * (pair ? 2 : 1));
            cfg.blockDim = dim3(kPThreads);
            cfg.dynamicSmemBytes = smem;
            cfg.stream = st;
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeClusterDimension;
            attr[0].val.clusterDim.x = pair ? 2 : 1; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
            cfg.attrs = attr; cfg.numAttrs = 1;
            prof_begin("ln_qkv", "gemm", st);
            e = cudaLaunchKernelEx(&cfg, kern, tmx, tmw_k, oq, ok, ov, p);
            prof_end(st);
            if (e == cudaSuccess) e = cudaGetLastError();
        }
        if (e == cudaSuccess) { launched = true; count_launch(); break; }
        if (!pair) break;                  // the single-CTA form failed: report it
        (void)cudaGetLastError();          // the pair launch was refused: clear the error and take the next form
        pair = false;
        e = cudaSuccess;
    }
    if (!launched && e == cudaSuccess) {
        // one CTA per tile (256 < C <= 512): weight ring = what the 226 KB leave beside the A tile
        const size_t fixed = (size_t)(c_in / 64) * kStage + (size_t)kWorkWarps * 2 * kOut + 1024;   // 1024 = barriers + alignment pad
        const size_t budget = fixed + 2 * kStage <= 113 * 1024 ? 113 * 1024 : 226 * 1024;
        p.n_stages = (int)((budget - fixed) / kStage);
        if (p.n_stages > 8) p.n_stages = 8;
        const size_t smem = fixed + (size_t)p.n_stages * kStage;
        auto kern = ln_qkv_kernel<2>;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) {
            prof_begin("ln_qkv", "gemm", st);
            kern<<<tiles, kThreads, smem, st>>>(tmx, tmw, tmq, tmk, tmv, p);
            prof_end(st);
            count_launch();
            e = cudaGetLastError();
        }
    }
    if (e != cudaSuccess) { set_error("%s: CUDA error: %s", who, cudaGetErrorString(e)); return GNN_ECUDA; }
    return GNN_OK;
}
