// ln_qkv.cu - row f4: the rest of the block the paper timed in front of the Graph Transformer attention
// ("layer normalization, QKV projection, and the attention mechanism itself"): LayerNorm fused into the
// A-operand staging of a tcgen05 GEMM that writes Q, K, V.
//
//   y[i, :] = (x[i, :] - mean_i) / sqrt(var_i + eps) * gamma + beta        (biased variance over the C features)
//   [Q | K | V][i, :] = y[i, :] W^T + bias,   W = [W_Q; W_K; W_V] of shape [3*H*d, C]
//
// (Round-2 layout: 320 threads - eight LayerNorm / epilogue warps, two per TMEM lane quarter - see below.)
// The paper runs these as stock PyTorch ops (LayerNorm kernel, cuBLAS GEMM: one write and one read of the normalised
// activations in HBM).  Here one CTA owns 128 rows: warps 0-3 normalise their rows in registers (a warp per row,
// 16-byte loads, shuffle reductions) and write them as bf16 straight into the 128-byte-swizzled K-major shared-memory
// tile the tensor core reads - the normalised activations never touch HBM.  Then, warp-specialised: warp 4 streams the
// weight tiles (128 outputs x 64 channels, 16 KB) through a TMA ring, warp 5 issues tcgen05.mma (128 x 128 x 16) into
// one of two 128-column TMEM accumulators, and warps 0-3 drain the other one (tcgen05.ld, + bias, bf16, per-warp
// transpose, coalesced stores) - full / empty mbarriers between the three roles, so the epilogue of output chunk c
// overlaps the products of chunk c + 1.
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

template <int NJ>     // 16-byte chunks of a row per lane: 1 for C <= 256, 2 for C <= 512
__global__ void __launch_bounds__(kThreads, 2)
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
        // ===== LayerNorm of this warp's 16 rows, in place in the A tile (lane <-> 16-byte chunks lane [, lane + 32]).
        // bf16 operands enter the fp32 sums directly (FHADD takes a register half: no unpack); squares, scale and shift
        // run as packed fp32 pairs (FFMA2 / FMUL2).
        const int nchunk = p.C / 8;
        float g[NJ][8], b[NJ][8];
        bool on[NJ];
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
            const int cc = lane + 32 * j;
            on[j] = cc < nchunk;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                g[j][i] = on[j] ? __ldg(p.gamma + cc * 8 + i) : 0.f;
                b[j][i] = on[j] ? __ldg(p.beta + cc * 8 + i) : 0.f;
            }
        }
        const float inv_c = 1.f / (float)p.C;
        mbar_wait(xfull, 0);
        constexpr int RB = NJ == 1 ? 4 : 2;   // rows per batch (independent shuffle-reduction chains)
        for (int rl = 0; rl < 16; rl += RB) {
            uint4 raw[RB][NJ];
            uint32_t addr[RB][NJ];
            float s[RB];
#pragma unroll
            for (int u = 0; u < RB; ++u) {
                float s0 = 0.f, s1 = 0.f;
#pragma unroll
                for (int j = 0; j < NJ; ++j) {
                    const int r = warp * 16 + rl + u, cc = lane + 32 * j;
                    addr[u][j] = (uint32_t)((cc >> 3) * kStage + (r >> 3) * 1024 + (r & 7) * 128 + (((cc & 7) ^ (r & 7)) << 4));
                    raw[u][j] = make_uint4(0, 0, 0, 0);
                    if (on[j]) raw[u][j] = *reinterpret_cast<const uint4*>(sA + addr[u][j]);
                    add_bf16x2(raw[u][j].x, s0, s1, s0, s1);
                    add_bf16x2(raw[u][j].y, s0, s1, s0, s1);
                    add_bf16x2(raw[u][j].z, s0, s1, s0, s1);
                    add_bf16x2(raw[u][j].w, s0, s1, s0, s1);
                }
                s[u] = s0 + s1;
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                for (int u = 0; u < RB; ++u) s[u] += __shfl_xor_sync(0xffffffffu, s[u], o);
            float v[RB][NJ][8], ss[RB];
#pragma unroll
            for (int u = 0; u < RB; ++u) {
                const float nmean = -s[u] * inv_c;
                float q0 = 0.f, q1 = 0.f;
#pragma unroll
                for (int j = 0; j < NJ; ++j) {
                    const uint32_t w[4] = {raw[u][j].x, raw[u][j].y, raw[u][j].z, raw[u][j].w};
                    const float nm = on[j] ? nmean : 0.f;     // lanes past the row's last chunk hold zeros and stay zero
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        add_bf16x2(w[i], nm, nm, v[u][j][2 * i], v[u][j][2 * i + 1]);
                        fma2v(q0, q1, v[u][j][2 * i], v[u][j][2 * i + 1], v[u][j][2 * i], v[u][j][2 * i + 1]);
                    }
                }
                ss[u] = q0 + q1;
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                for (int u = 0; u < RB; ++u) ss[u] += __shfl_xor_sync(0xffffffffu, ss[u], o);
#pragma unroll
            for (int u = 0; u < RB; ++u) {
                const int r = warp * 16 + rl + u;
                const float rstd = row0 + r < p.n ? 1.f / sqrtf(ss[u] * inv_c + p.eps) : 0.f;
                const bool rv = row0 + r < p.n;
#pragma unroll
                for (int j = 0; j < NJ; ++j) {
                    if (on[j]) {
                        uint32_t o[4];
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            float y0 = v[u][j][2 * i], y1 = v[u][j][2 * i + 1];
                            mul2(y0, y1, rstd);
                            float z0 = rv ? b[j][2 * i] : 0.f, z1 = rv ? b[j][2 * i + 1] : 0.f;
                            fma2v(z0, z1, y0, y1, g[j][2 * i], g[j][2 * i + 1]);
                            const __nv_bfloat162 yb = __floats2bfloat162_rn(z0, z1);
                            o[i] = *reinterpret_cast<const uint32_t*>(&yb);
                        }
                        *reinterpret_cast<uint4*>(sA + addr[u][j]) = make_uint4(o[0], o[1], o[2], o[3]);
                    }
                }
            }
        }
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
        // ===== epilogue: warp w drains TMEM lanes 32 (w & 3) .. +31 (tile rows) of column half w >> 2 of every chunk:
        // accumulator -> + bias -> bf16 -> 32-row x 16-column staging buffer (the layout TMA's 32-byte swizzle expects)
        // -> one TMA store per buffer (rows past n are clipped by the unit); two buffers per warp alternate
        const int q4 = warp & 3, hsel = warp >> 2;
        const uint32_t t_lane = tmem + ((uint32_t)(q4 * 32) << 16);
        uint8_t* stage = sT + warp * 2 * kOut;
        const uint32_t my = (uint32_t)lane * 32, sw = ((uint32_t)(lane >> 2) & 1u) << 4;
        int n_st = 0;
        float4 bb[8];
        if (p.bias) {
#pragma unroll
            for (int i = 0; i < 8; ++i) bb[i] = __ldg(reinterpret_cast<const float4*>(p.bias + 64 * hsel) + i);
        }
        for (int c = 0; c < n_chunks; ++c) {
            const int bsel = c & 1;
            const int col0 = c * kNC + 64 * hsel;
            const int t = col0 / p.R, off = col0 - t * p.R;
            const CUtensorMap* tmo = t == 0 ? &tmq : (t == 1 ? &tmk : &tmv);
            mbar_wait(tfull + bsel, (uint32_t)((c >> 1) & 1));
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll 1
            for (int c0 = 0; c0 < 64; c0 += 32) {
                float t32[32];
                tmem_ld32(t_lane + bsel * kNC + 64 * hsel + c0, t32);
                if (c0 == 32) {                                 // last read of this accumulator half: hand it back to the MMA warp
                    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                    __syncwarp();
                    if (lane == 0) mbar_arrive(tempty + bsel);
                }
                if (p.bias) {
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        add2(t32[4 * i], t32[4 * i + 1], bb[i].x, bb[i].y);
                        add2(t32[4 * i + 2], t32[4 * i + 3], bb[i].z, bb[i].w);
                    }
                    // the next pass's bias values travel while this pass is packed and stored
                    const int nxt = c0 == 0 ? col0 + 32 : (c + 1 < n_chunks ? (c + 1) * kNC + 64 * hsel : col0);
#pragma unroll
                    for (int i = 0; i < 8; ++i) bb[i] = __ldg(reinterpret_cast<const float4*>(p.bias + nxt) + i);
                }
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
            }
        }
        if (lane == 0) tma_store_wait<0>();
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 9) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 256;" ::"r"(tmem) : "memory");
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
    // weight ring: as many 16 KB stages as keep two CTAs per SM (113 KB each) when the A tile allows it, else one CTA
    const size_t fixed = (size_t)(c_in / 64) * kStage + (size_t)kWorkWarps * 2 * kOut + 1024;   // 1024 = barriers + alignment pad
    const size_t budget = fixed + 2 * kStage <= 113 * 1024 ? 113 * 1024 : 226 * 1024;
    p.n_stages = (int)((budget - fixed) / kStage);
    if (p.n_stages > 8) p.n_stages = 8;
    const size_t smem = fixed + (size_t)p.n_stages * kStage;
    auto kern = c_in <= 256 ? ln_qkv_kernel<1> : ln_qkv_kernel<2>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) {
        cudaStream_t st = (cudaStream_t)stream;
        prof_begin("ln_qkv", "gemm", st);
        kern<<<(n + kRows - 1) / kRows, kThreads, smem, st>>>(tmx, tmw, tmq, tmk, tmv, p);
        prof_end(st);
        count_launch();
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) { set_error("%s: CUDA error: %s", who, cudaGetErrorString(e)); return GNN_ECUDA; }
    return GNN_OK;
}
