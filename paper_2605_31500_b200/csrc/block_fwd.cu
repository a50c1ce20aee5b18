// block_fwd.cu - row a12: block-sparse Graph Transformer forward on the 5th-generation tensor cores
// (tcgen05.mma, accumulators in TMEM) for locally dense graphs, merged with the CSR remainder.
//
// Paper's version: per 16-row window and head, WMMA 16x16x16 on A100: S = Q_win K_blk^T,
// bitmap mask, FlashAttention-style online softmax, acc += P V_blk.  tcgen05.mma has M in {64, 128}, so here one
// CTA owns a tile of 128 destination rows = 8 windows and, per head, issues ONE 128x128xd product
// S = Q_tile K_tile^T (bf16 in, fp32 in TMEM); thread t owns row t (TMEM lane t), reads back only the 32 columns
// that hold its window's diagonal block, masks its 16 scores with the plan's 16-bit row bitmap (row a11), forms
// p = 2^(s - m) in registers, writes P (bf16, zero off the diagonal blocks) over the dead Q/K staging area and a
// second product O = P V_tile (128x128 by 128xd) leaves the block part in the same TMEM columns.  The off-diagonal
// blocks are wasted tensor work (8x) - far below the memory time of the tile.
//
// The block part is then handed to a cooperative layout through a shared-memory transpose (row slots of 272 bytes):
// 8 lanes per row, each owning 8 channels, gather the row's remainder sources (sources outside the window: the
// long-range in-edges) as coalesced 128-byte slices, run the same online softmax, merge it with the block part by
// log-sum-exp and store O coalesced - so the result equals the plain CSR forward.  Per-thread row-wise
// gathers and stores (32 L1 wavefronts per instruction) made the first version LSU-bound; this layout needs 4.
//
// Operand staging: the head slices of Q, K (K-major operands) and V (MN-major B operand, no transpose) of the 128
// tile rows are 128 x 128-byte boxes of the [n, H*d] tensors: one elected thread fetches them with three TMA tile
// loads (cp.async.bulk.tensor.2d, 128-byte swizzle, rows past n zero-filled) that complete on an mbarrier, kStages
// heads ahead of the consumers; the tensor core reads them through 64-bit shared-memory matrix descriptors
// (SWIZZLE_128B: 8-row groups 1024 bytes apart).  P is written by the threads in the canonical no-swizzle
// core-matrix layout (8 x 16-byte core matrices; LBO / SBO = byte distance between core matrices along K / along M).
// MMA completion is signalled with tcgen05.commit on an mbarrier.  48 KB of shared memory per stage and 128 TMEM
// columns per CTA.
#include <cuda.h>
#include <cuda_bf16.h>

#include "internal.h"
#include "kernels.cuh"
#include "tc_common.cuh"

namespace gnn {
namespace {

#ifndef GNN_BLOCK_STAGES
#define GNN_BLOCK_STAGES 1
#endif
#ifndef GNN_BLOCK_MINB
#define GNN_BLOCK_MINB 3
#endif
constexpr int kStages = GNN_BLOCK_STAGES;   // heads of Q/K/V in flight per CTA (1: 3 CTAs/SM, 2: 2 CTAs/SM)
constexpr int kTile = 128;  // destination rows per CTA = MMA M = TMEM lanes
constexpr int kTS = 68;     // floats per row slot of the transpose buffer (64 + m, l, lx + pad): 272 B

using namespace tc;

template <int D>
__global__ void __launch_bounds__(kTile, kStages == 1 ? GNN_BLOCK_MINB : 2)
gt_fwd_block_kernel(const __grid_constant__ CUtensorMap tmq, const __grid_constant__ CUtensorMap tmk,
                    const __grid_constant__ CUtensorMap tmv, const __nv_bfloat16* __restrict__ q,
                    const __nv_bfloat16* __restrict__ k, const __nv_bfloat16* __restrict__ v,
                    __nv_bfloat16* __restrict__ out, float* __restrict__ lse, const uint16_t* __restrict__ bitmap,
                    const int32_t* __restrict__ rem_rowptr, const int32_t* __restrict__ rem_colidx, int n, int H,
                    float sscale) {
    static_assert(D == 64, "a head slice must be one 128-byte swizzle row");
    constexpr int SBO_P = (kTile / 8) * 128;
    constexpr int kBytesQK = kTile * D * 2, kBytesP = kTile * kTile * 2, kStageBytes = 3 * kBytesQK;
    static_assert(kBytesP <= 2 * kBytesQK, "P aliases the Q and K staging buffers");
    static_assert(kTile * kTS * 4 <= kStageBytes, "the transpose buffer aliases one stage");
    extern __shared__ uint8_t smem_raw[];
    // 128-byte swizzle atoms (8 rows x 128 bytes) must sit on 1024-byte boundaries
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + kStages * kStageBytes);   // TMA completion, one per stage
    uint64_t* bar = full + kStages;                                               // tcgen05.commit
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar + 1);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int row0 = blockIdx.x * kTile, row = row0 + tid;
    const bool rvalid = row < n;
    const size_t rowe = (size_t)H * D;

    // ---- one-time setup: barrier, TMEM (128 columns: S, later overwritten by O)
    // one head's Q, K, V boxes into stage hh % kStages (rows past n arrive as zeros and count as full bytes)
    auto issue_head = [&](int hh) {
        uint8_t* st = smem + (hh % kStages) * kStageBytes;
        uint64_t* fb = full + (hh % kStages);
        mbar_expect_tx(fb, 3 * kBytesQK);
        tma_load_2d(st, &tmq, hh * D, row0, fb);
        tma_load_2d(st + kBytesQK, &tmk, hh * D, row0, fb);
        tma_load_2d(st + 2 * kBytesQK, &tmv, hh * D, row0, fb);
    };
    if (tid == 0) {
        mbar_init(bar, 1);
#pragma unroll
        for (int s = 0; s < kStages; ++s) mbar_init(full + s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        for (int hh = 0; hh < kStages - 1 && hh < H; ++hh) issue_head(hh);
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 128;" ::"r"(smem_u32(tmem_slot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;
    const uint32_t t_lane = tmem + ((uint32_t)(warp * 32) << 16);
    uint32_t phase = 0;

    const uint32_t bits = rvalid ? (uint32_t)__ldg(bitmap + row) : 0u;
    const int rb = rvalid ? __ldg(rem_rowptr + row) : 0, re = rvalid ? __ldg(rem_rowptr + row + 1) : 0;
    const int wl = tid >> 4;  // window of this row inside the tile
    constexpr uint32_t kIdescS = make_idesc(kTile, kTile, false), kIdescO = make_idesc(kTile, D, true);

    // cooperative role (8 lanes per row, group g4 of the warp takes rows g4 + 4 i): the remainder sources of the
    // group's 8 rows are head-invariant - the first two per row stay in registers
    const int g4 = lane >> 3, gl = lane & 7;
    int cj0[8], cj1[8], ccnt[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int rowc = row0 + warp * 32 + g4 + 4 * i;
        const bool cv = rowc < n;
        const int rbc = cv ? __ldg(rem_rowptr + rowc) : 0;
        ccnt[i] = cv ? __ldg(rem_rowptr + rowc + 1) - rbc : 0;
        cj0[i] = ccnt[i] > 0 ? __ldg(rem_colidx + rbc) : -1;
        cj1[i] = ccnt[i] > 1 ? __ldg(rem_colidx + rbc + 1) : -1;
    }

    for (int h = 0; h < H; ++h) {
        // ---- operands of this head: issue the TMA loads of the head kStages - 1 ahead (its stage was released by
        // the barrier that ended the previous head), then wait for this head's boxes
        uint8_t* sQ = smem + (h % kStages) * kStageBytes;
        uint8_t* sK = sQ + kBytesQK;
        uint8_t* sP = sQ;                    // P overwrites Q and K once S = Q K^T has completed
        uint8_t* sV = sQ + 2 * kBytesQK;
        if (tid == 0 && h + kStages - 1 < H) issue_head(h + kStages - 1);
        mbar_wait(full + (h % kStages), (uint32_t)(h / kStages) & 1u);
        // ---- S = Q K^T on the tensor cores (one elected thread issues)
        if (tid == 0) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
            for (int s = 0; s < D / 16; ++s)
                umma(tmem, make_desc_sw128(smem_u32(sQ) + s * 32, 1024), make_desc_sw128(smem_u32(sK) + s * 32, 1024),
                     kIdescS, s > 0);   // K step = 16 channels = 32 bytes inside the 128-byte swizzle row
            umma_commit(bar);
        }
        mbar_wait(bar, phase);
        phase ^= 1;
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        // ---- this row's 16 scores of its own window's diagonal block; mask; block-local softmax
        float m = -INFINITY, l = 0.f, lx = 0.f;   // l: sum of the bf16-rounded weights (normalises O); lx: exact (for L)
        {
            float sv[32];
            tmem_ld32(t_lane + warp * 32, sv);
            float s16[16];
#pragma unroll
            for (int c = 0; c < 16; ++c) {
                const float x = (lane >= 16) ? sv[16 + c] : sv[c];
                s16[c] = ((bits >> c) & 1u) ? x * sscale : -INFINITY;
                m = fmaxf(m, s16[c]);
            }
            const float ms = (m == -INFINITY) ? 0.f : m;
            uint32_t pk[8];
#pragma unroll
            for (int c = 0; c < 16; c += 2) {
                const float p0 = ex2(s16[c] - ms), p1 = ex2(s16[c + 1] - ms);
                const __nv_bfloat162 pb = __floats2bfloat162_rn(p0, p1);
                l += __low2float(pb) + __high2float(pb);   // normalise with the rounded weights the MMA will use
                lx += p0 + p1;
                pk[c >> 1] = *reinterpret_cast<const uint32_t*>(&pb);
            }
            // P aliases Q/K.  The rows of warp w occupy the contiguous 8 KB [w * 8192, +8192) of the canonical layout:
            // the warp clears its own region with conflict-free stores, then every lane writes its diagonal block
#pragma unroll
            for (int it = 0; it < 16; ++it)
                *reinterpret_cast<uint4*>(sP + warp * 8192 + (it * 32 + lane) * 16) = make_uint4(0, 0, 0, 0);
            __syncwarp();
            uint8_t* prow = sP + canon(tid, 16 * wl, SBO_P);
            *reinterpret_cast<uint4*>(prow) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
            *reinterpret_cast<uint4*>(prow + 128) = make_uint4(pk[4], pk[5], pk[6], pk[7]);
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        // ---- O_block = P V on the tensor cores
        if (tid == 0) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
            for (int s = 0; s < kTile / 16; ++s)
                umma(tmem, make_desc(smem_u32(sP) + s * 256, 128, SBO_P), make_desc_sw128(smem_u32(sV) + s * 2048, 1024),
                     kIdescO, s > 0);   // V: [source][channel] rows of 128 bytes = MN-major, K step = 16 sources
            umma_commit(bar);
        }
        mbar_wait(bar, phase);
        phase ^= 1;
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        // ---- hand the block part over to the cooperative layout: thread t (owner of row t) writes its unnormalised
        // O row and (m, l, lx) into the warp's transpose buffer (aliases the dead Q/K/P/V staging area; 272-byte row
        // slots keep 16-byte accesses conflict-free)
        float* sT = reinterpret_cast<float*>(sQ) + warp * (32 * kTS);
        {
            float* slot = sT + lane * kTS;
#pragma unroll
            for (int c0 = 0; c0 < D; c0 += 32) {
                float t32[32];
                tmem_ld32(t_lane + c0, t32);
#pragma unroll
                for (int i = 0; i < 32; i += 4)
                    *reinterpret_cast<float4*>(slot + c0 + i) = make_float4(t32[i], t32[i + 1], t32[i + 2], t32[i + 3]);
            }
            slot[D] = m; slot[D + 1] = l; slot[D + 2] = lx;
        }
        __syncwarp();
        // ---- remainder edges (sources outside the window) and the final merge, 8 lanes per row: every gather is a
        // coalesced 128-byte row slice and the O row is stored coalesced (a lane owns 8 channels of the head).
        // Rows are handled four at a time so that 20 independent 16-byte gathers are in flight per lane.
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            uint4 Lq[4], Lk0[4], Lk1[4], Lv0[4], Lv1[4];
#pragma unroll
            for (int ii = 0; ii < 4; ++ii) {
                const int i = 4 * half + ii;
                const int rowc = row0 + warp * 32 + g4 + 4 * i;
                const uint4 z = make_uint4(0, 0, 0, 0);
                Lq[ii] = Lk0[ii] = Lk1[ii] = Lv0[ii] = Lv1[ii] = z;
                if (cj0[i] >= 0) {
                    const size_t off = (size_t)cj0[i] * rowe + (size_t)h * D;
                    Lq[ii] = __ldg(reinterpret_cast<const uint4*>(q + (size_t)rowc * rowe + (size_t)h * D) + gl);
                    Lk0[ii] = __ldg(reinterpret_cast<const uint4*>(k + off) + gl);
                    Lv0[ii] = __ldg(reinterpret_cast<const uint4*>(v + off) + gl);
                }
                if (cj1[i] >= 0) {
                    const size_t off = (size_t)cj1[i] * rowe + (size_t)h * D;
                    Lk1[ii] = __ldg(reinterpret_cast<const uint4*>(k + off) + gl);
                    Lv1[ii] = __ldg(reinterpret_cast<const uint4*>(v + off) + gl);
                }
            }
#pragma unroll
            for (int ii = 0; ii < 4; ++ii) {
                const int i = 4 * half + ii;
                const int rl = g4 + 4 * i;
                const int rowc = row0 + warp * 32 + rl;
                const bool cv = rowc < n;
                float mr = -INFINITY, lr = 0.f, a[8];
#pragma unroll
                for (int c = 0; c < 8; ++c) a[c] = 0.f;
                // one step of the online softmax over two gathered sources (masked when the id is negative)
                auto pair_step = [&](int j0, int j1, const uint4& qv, const uint4& k0, const uint4& k1, const uint4& v0,
                                     const uint4& v1) {
                    float d0 = 0.f, d0b = 0.f, d1 = 0.f, d1b = 0.f;
                    fma_bf16x2(qv.x, k0.x, d0, d0b); fma_bf16x2(qv.y, k0.y, d0, d0b);
                    fma_bf16x2(qv.z, k0.z, d0, d0b); fma_bf16x2(qv.w, k0.w, d0, d0b);
                    fma_bf16x2(qv.x, k1.x, d1, d1b); fma_bf16x2(qv.y, k1.y, d1, d1b);
                    fma_bf16x2(qv.z, k1.z, d1, d1b); fma_bf16x2(qv.w, k1.w, d1, d1b);
                    d0 += d0b; d1 += d1b;
#pragma unroll
                    for (int o = 1; o < 8; o <<= 1) {
                        d0 += __shfl_xor_sync(0xffffffffu, d0, o);
                        d1 += __shfl_xor_sync(0xffffffffu, d1, o);
                    }
                    const float s0 = j0 < 0 ? -INFINITY : d0 * sscale, s1 = j1 < 0 ? -INFINITY : d1 * sscale;
                    const float mx = fmaxf(mr, fmaxf(s0, s1));
                    const float ms = (mx == -INFINITY) ? 0.f : mx;
                    const float corr = ex2(mr - ms), p0 = ex2(s0 - ms), p1 = ex2(s1 - ms);
                    lr = lr * corr + p0 + p1;
                    mr = mx;
                    const uint32_t w0[4] = {v0.x, v0.y, v0.z, v0.w}, w1[4] = {v1.x, v1.y, v1.z, v1.w};
#pragma unroll
                    for (int jj = 0; jj < 4; ++jj) {
                        float x = a[2 * jj] * corr, y = a[2 * jj + 1] * corr;
                        x = fmaf(p0, __uint_as_float(w0[jj] << 16), x);
                        y = fmaf(p0, __uint_as_float(w0[jj] & 0xffff0000u), y);
                        a[2 * jj] = fmaf(p1, __uint_as_float(w1[jj] << 16), x);
                        a[2 * jj + 1] = fmaf(p1, __uint_as_float(w1[jj] & 0xffff0000u), y);
                    }
                };
                pair_step(cj0[i], cj1[i], Lq[ii], Lk0[ii], Lk1[ii], Lv0[ii], Lv1[ii]);
                // rows with more than two remainder sources: further pairs, gathered directly (warp-uniform trip count)
                int maxcnt = ccnt[i];
                maxcnt = max(maxcnt, __shfl_xor_sync(0xffffffffu, maxcnt, 8));
                maxcnt = max(maxcnt, __shfl_xor_sync(0xffffffffu, maxcnt, 16));
                if (maxcnt > 2) {
                    const int rbc = cv ? __ldg(rem_rowptr + rowc) : 0;
                    for (int eb = 2; eb < maxcnt; eb += 2) {
                        const int j0 = eb < ccnt[i] ? __ldg(rem_colidx + rbc + eb) : -1;
                        const int j1 = eb + 1 < ccnt[i] ? __ldg(rem_colidx + rbc + eb + 1) : -1;
                        uint4 k0 = make_uint4(0, 0, 0, 0), k1 = k0, v0 = k0, v1 = k0;
                        if (j0 >= 0) {
                            const size_t off = (size_t)j0 * rowe + (size_t)h * D;
                            k0 = __ldg(reinterpret_cast<const uint4*>(k + off) + gl);
                            v0 = __ldg(reinterpret_cast<const uint4*>(v + off) + gl);
                        }
                        if (j1 >= 0) {
                            const size_t off = (size_t)j1 * rowe + (size_t)h * D;
                            k1 = __ldg(reinterpret_cast<const uint4*>(k + off) + gl);
                            v1 = __ldg(reinterpret_cast<const uint4*>(v + off) + gl);
                        }
                        pair_step(j0, j1, Lq[ii], k0, k1, v0, v1);
                    }
                }
                // block part of this row from the transpose buffer, log-sum-exp merge, normalise, store
                const float* slot = sT + rl * kTS;
                const float4 b0 = *reinterpret_cast<const float4*>(slot + gl * 8);
                const float4 b1 = *reinterpret_cast<const float4*>(slot + gl * 8 + 4);
                const float mb = slot[D], lb = slot[D + 1], lxb = slot[D + 2];
                const float mm = fmaxf(mb, mr);
                const float ms = (mm == -INFINITY) ? 0.f : mm;
                const float cb = ex2(mb - ms), cr = ex2(mr - ms);
                const float lsum = lb * cb + lr * cr, lxsum = lxb * cb + lr * cr;
                const float inv = lsum > 0.f ? 1.f / lsum : 0.f;
                if (cv) {
                    const float ob[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
                    uint32_t w[4];
#pragma unroll
                    for (int jj = 0; jj < 4; ++jj) {
                        const __nv_bfloat162 b2 = __floats2bfloat162_rn((ob[2 * jj] * cb + a[2 * jj] * cr) * inv,
                                                                        (ob[2 * jj + 1] * cb + a[2 * jj + 1] * cr) * inv);
                        w[jj] = *reinterpret_cast<const uint32_t*>(&b2);
                    }
                    reinterpret_cast<uint4*>(out + (size_t)rowc * rowe + (size_t)h * D)[gl] = make_uint4(w[0], w[1], w[2], w[3]);
                    if (gl == 0) lse[(size_t)rowc * H + h] = lxsum > 0.f ? (mm + lg2(lxsum)) * kLn2 : -INFINITY;
                }
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic writes (P, transpose) before the next TMA
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();   // this stage and TMEM are reused by a later head
    }
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 128;" ::"r"(tmem) : "memory");
}

}  // namespace
}  // namespace gnn

using namespace gnn;

extern "C" gnn_status_t gnn_gt_attn_fwd_block(const gnn_plan_t* P, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                              const void* q, const void* k, const void* v, int32_t heads, int32_t head_dim,
                                              gnn_dtype_t dtype, void* out, float* lse, gnn_stream_t stream) {
    const char* who = "gnn_gt_attn_fwd_block";
    if (!P || rowptr != P->rowptr || colidx != P->colidx || n != P->n) {
        set_error("%s: NULL plan, or rowptr/colidx/n differ from the arrays the plan was built from", who);
        return GNN_EINVAL;
    }
    if (!P->blk_bitmap) { set_error("%s: plan was built without build_blocks", who); return GNN_EINVAL; }
    if (!q || !k || !v || !out || !lse) { set_error("%s: NULL pointer argument", who); return GNN_EINVAL; }
    if ((((uintptr_t)q | (uintptr_t)k | (uintptr_t)v | (uintptr_t)out) & 31) != 0) {
        set_error("%s: feature pointers must be 32-byte aligned", who);
        return GNN_EINVAL;
    }
    if (dtype != GNN_BF16 || head_dim != 64 || heads < 1) {
        set_error("%s: unsupported shape heads=%d head_dim=%d dtype=%d (bf16, head_dim 64 only)", who, heads, head_dim, dtype);
        return GNN_EUNSUPPORTED;
    }
    constexpr int D = 64;
    CUtensorMap tmq, tmk, tmv;
    if (!tc::encode_row_tile_map(&tmq, q, n, heads * D, D, kTile) || !tc::encode_row_tile_map(&tmk, k, n, heads * D, D, kTile) ||
        !tc::encode_row_tile_map(&tmv, v, n, heads * D, D, kTile)) {
        set_error("%s: cuTensorMapEncodeTiled unavailable or failed", who);
        return GNN_ECUDA;
    }
    // kStages x (Q, K (aliased by P), V), barriers, TMEM slot, slack for the 1024-byte alignment
    const size_t smem = (size_t)kStages * 3 * kTile * D * 2 + 64 + 1024;
    cudaError_t e = cudaFuncSetAttribute(gt_fwd_block_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) {
        const int grid = (n + kTile - 1) / kTile;
        prof_begin("gt_fwd_block", "tile", (cudaStream_t)stream);
        gt_fwd_block_kernel<D><<<grid, kTile, smem, (cudaStream_t)stream>>>(
            tmq, tmk, tmv, (const __nv_bfloat16*)q, (const __nv_bfloat16*)k, (const __nv_bfloat16*)v, (__nv_bfloat16*)out, lse, P->blk_bitmap,
            P->blk_rem_rowptr, P->blk_rem_colidx, n, heads, kLog2e / sqrtf((float)D));
        prof_end((cudaStream_t)stream);
        count_launch();
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) { set_error("%s: CUDA error: %s", who, cudaGetErrorString(e)); return GNN_ECUDA; }
    return GNN_OK;
}
