// block_bwd.cu - tensor-core backward for the diagonal 16-row block layout (rows a11 / a12 + the backward half of f2):
// the in-window ("diagonal block") edges of a tile of 128 rows are TILE-LOCAL - dQ, dK and dV of the tile's rows get
// their in-window contributions from the tile's own Q, K, V, dO rows only - so they run as dense products on the 5th
// generation tensor cores without any atomics (P = exp(S - L), dV = P^T dO, dP = dO V^T,
// dS = P o (dP - Delta), dQ = dS K, dK = dS^T Q; the paper needs atomicAdd because its tiles share source columns).
// The out-of-window edges (the remainder CSR of the plan: the ~2 long-range in-edges per node of cfg 4, duplicates):
//   dst side  inside this kernel: 8 lanes per row gather k_j, v_j of the row's remainder sources as coalesced 128-byte
//             slices (as the forward does, block_fwd.cu), first for Delta - which must be complete (block part +
//             remainder part, fp32) before any dS is formed - then for their dQ terms;
//   src side  afterwards through the CSR src pass (ops_gt.cuh::GtBwdSrc) restricted to the TRANSPOSED remainder CSR the
//             plan holds, adding to the tile-local dK / dV this kernel stored (one writer per element, fixed order).
// Per (tile, head): TMA loads the Q, K, V, dO head slices (128 rows x 128 bytes, SWIZZLE_128B); ONE commit covers
// S = Q K^T and dP = dO V^T (two 128-column TMEM accumulators); thread t = tile row t reads its window's 16 + 16 values,
// forms P and dS in registers and stages dS, dS^T and P^T one after the other as the block-diagonal bf16 A operand of
// dQ = dS K, dK = dS^T Q, dV = P^T dO (B operands = the resident K, Q, dO tiles, MN-major).  In-window sums have at most
// 16 terms, so one bf16 rounding of the weights stays far inside the tolerance.  96 KB of shared memory and 256 TMEM
// columns per CTA: two CTAs per SM.
#include <cuda.h>
#include <cuda_bf16.h>

#include "internal.h"
#include "kernels.cuh"
#include "tc_common.cuh"

namespace gnn {
namespace {
using namespace tc;

constexpr int kTile = 128;
constexpr int kHT = 16384;      // one operand tile: 128 rows x 64 channels bf16
constexpr int kWBytes = 32768;  // block-diagonal 128 x 128 bf16 weight tile
constexpr int kTS = 68;         // floats per transpose slot

struct BlockBwdParams {
    const __nv_bfloat16 *q, *k, *v, *dout;
    const float* lse;
    const uint16_t* bitmap;
    const int32_t *rem_rowptr, *rem_colidx;
    float *dq, *dk, *dv, *delta;
    float2* stat2;               // [n, H] (L log2e, Delta) for the remainder src pass
    int n, H;
    float sscale, inv_sqrt_d;
};

// <a, b> over this lane's 8 bf16 channels, partial (to be reduced over the 8 lanes of the row)
__device__ __forceinline__ float dot8(const uint4& a, const uint4& b) {
    float d0 = 0.f, d1 = 0.f;
    fma_bf16x2(a.x, b.x, d0, d1); fma_bf16x2(a.y, b.y, d0, d1);
    fma_bf16x2(a.z, b.z, d0, d1); fma_bf16x2(a.w, b.w, d0, d1);
    return d0 + d1;
}
__device__ __forceinline__ float red8(float x) {
#pragma unroll
    for (int o = 1; o < 8; o <<= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}
// acc[0..8) += w * (8 bf16 channels of r)
__device__ __forceinline__ void axpy8(float (&acc)[8], float w, const uint4& r) {
    const uint32_t x[4] = {r.x, r.y, r.z, r.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        acc[2 * j] = fmaf(w, __uint_as_float(x[j] << 16), acc[2 * j]);
        acc[2 * j + 1] = fmaf(w, __uint_as_float(x[j] & 0xffff0000u), acc[2 * j + 1]);
    }
}

template <int D>
__global__ void __launch_bounds__(kTile, 2)
gt_bwd_block_kernel(const __grid_constant__ CUtensorMap tmq, const __grid_constant__ CUtensorMap tmk,
                    const __grid_constant__ CUtensorMap tmv, const __grid_constant__ CUtensorMap tmdo,
                    const BlockBwdParams p) {
    static_assert(D == 64, "a head slice must be one 128-byte swizzle row");
    constexpr int SBO_W = (kTile / 8) * 128;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint8_t *sQ = smem, *sK = smem + kHT, *sV = smem + 2 * kHT, *sdO = smem + 3 * kHT, *sW = smem + 4 * kHT;
    uint64_t* full = reinterpret_cast<uint64_t*>(sW + kWBytes);
    uint64_t* bar = full + 1;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar + 1);
    float* s_drem = reinterpret_cast<float*>(sW + kWBytes + 32);   // [128] remainder part of Delta per row
    float* s_delta = s_drem + kTile;                               // [128] Delta per row
    float* sT = reinterpret_cast<float*>(smem);                    // transpose slots over the dead operand tiles

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int row0 = blockIdx.x * kTile, row = row0 + tid;
    const bool rvalid = row < p.n;
    const int wl = tid >> 4;
    const size_t rowe = (size_t)p.H * D;

    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_init(full, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 256;" ::"r"(smem_u32(tmem_slot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
#pragma unroll
    for (int it = 0; it < kWBytes / (kTile * 16); ++it)   // off-diagonal blocks of the weight tile stay zero
        *reinterpret_cast<uint4*>(sW + (it * kTile + tid) * 16) = make_uint4(0, 0, 0, 0);
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;
    const uint32_t t_lane = tmem + ((uint32_t)(warp * 32) << 16);
    uint32_t phase = 0;
    const uint32_t bits = rvalid ? (uint32_t)__ldg(p.bitmap + row) : 0u;
    constexpr uint32_t kIdescS = make_idesc(kTile, kTile, false), kIdescO = make_idesc(kTile, D, true);

    // cooperative role (8 lanes per row; lane group g4 of the warp takes rows g4 + 4 i): remainder sources are
    // head-invariant, the first two per row stay in registers
    const int g4 = lane >> 3, gl = lane & 7;
    int cj0[8], cj1[8], ccnt[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int rowc = row0 + warp * 32 + g4 + 4 * i;
        const bool cv = rowc < p.n;
        const int rbc = cv ? __ldg(p.rem_rowptr + rowc) : 0;
        ccnt[i] = cv ? __ldg(p.rem_rowptr + rowc + 1) - rbc : 0;
        cj0[i] = ccnt[i] > 0 ? __ldg(p.rem_colidx + rbc) : -1;
        cj1[i] = ccnt[i] > 1 ? __ldg(p.rem_colidx + rbc + 1) : -1;
    }

    for (int h = 0; h < p.H; ++h) {
        const size_t hoff = (size_t)h * D;
        if (tid == 0) {
            mbar_expect_tx(full, 4 * kHT);
            tma_load_2d(sQ, &tmq, h * D, row0, full);
            tma_load_2d(sK, &tmk, h * D, row0, full);
            tma_load_2d(sV, &tmv, h * D, row0, full);
            tma_load_2d(sdO, &tmdo, h * D, row0, full);
        }
        // ---- remainder, pass 1 (overlaps the TMA loads and the first products): p_r, dP_r of the first two remainder
        // edges of every row (kept in registers) and the remainder part of Delta
        float pr[8][2], dpr[8][2];
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            uint4 Lq[4], Ld[4], Lk0[4], Lk1[4], Lv0[4], Lv1[4];
#pragma unroll
            for (int ii = 0; ii < 4; ++ii) {
                const int i = 4 * half + ii;
                const int rowc = row0 + warp * 32 + g4 + 4 * i;
                const uint4 z = make_uint4(0, 0, 0, 0);
                Lq[ii] = Ld[ii] = Lk0[ii] = Lk1[ii] = Lv0[ii] = Lv1[ii] = z;
                if (cj0[i] >= 0) {
                    Lq[ii] = __ldg(reinterpret_cast<const uint4*>(p.q + (size_t)rowc * rowe + hoff) + gl);
                    Ld[ii] = __ldg(reinterpret_cast<const uint4*>(p.dout + (size_t)rowc * rowe + hoff) + gl);
                    Lk0[ii] = __ldg(reinterpret_cast<const uint4*>(p.k + (size_t)cj0[i] * rowe + hoff) + gl);
                    Lv0[ii] = __ldg(reinterpret_cast<const uint4*>(p.v + (size_t)cj0[i] * rowe + hoff) + gl);
                }
                if (cj1[i] >= 0) {
                    Lk1[ii] = __ldg(reinterpret_cast<const uint4*>(p.k + (size_t)cj1[i] * rowe + hoff) + gl);
                    Lv1[ii] = __ldg(reinterpret_cast<const uint4*>(p.v + (size_t)cj1[i] * rowe + hoff) + gl);
                }
            }
#pragma unroll
            for (int ii = 0; ii < 4; ++ii) {
                const int i = 4 * half + ii;
                const int rl = g4 + 4 * i;
                const int rowc = row0 + warp * 32 + rl;
                const bool cv = rowc < p.n;
                const float lr = (cv && ccnt[i] > 0) ? __ldg(p.lse + (size_t)rowc * p.H + h) * kLog2e : 0.f;
                const float s0 = red8(dot8(Lq[ii], Lk0[ii])), s1 = red8(dot8(Lq[ii], Lk1[ii]));
                dpr[i][0] = red8(dot8(Ld[ii], Lv0[ii]));
                dpr[i][1] = red8(dot8(Ld[ii], Lv1[ii]));
                pr[i][0] = cj0[i] >= 0 ? ex2(fmaf(s0, p.sscale, -lr)) : 0.f;
                pr[i][1] = cj1[i] >= 0 ? ex2(fmaf(s1, p.sscale, -lr)) : 0.f;
                float drem = pr[i][0] * dpr[i][0] + pr[i][1] * dpr[i][1];
                int maxcnt = ccnt[i];
                maxcnt = max(maxcnt, __shfl_xor_sync(0xffffffffu, maxcnt, 8));
                maxcnt = max(maxcnt, __shfl_xor_sync(0xffffffffu, maxcnt, 16));
                if (maxcnt > 2) {      // rows with more than two remainder sources (warp-uniform trip count)
                    const int rbc = cv ? __ldg(p.rem_rowptr + rowc) : 0;
                    for (int eb = 2; eb < maxcnt; ++eb) {
                        const int j = eb < ccnt[i] ? __ldg(p.rem_colidx + rbc + eb) : -1;
                        uint4 kk = make_uint4(0, 0, 0, 0), vv = kk;
                        if (j >= 0) {
                            kk = __ldg(reinterpret_cast<const uint4*>(p.k + (size_t)j * rowe + hoff) + gl);
                            vv = __ldg(reinterpret_cast<const uint4*>(p.v + (size_t)j * rowe + hoff) + gl);
                        }
                        const float s = red8(dot8(Lq[ii], kk)), dp = red8(dot8(Ld[ii], vv));
                        drem += j >= 0 ? ex2(fmaf(s, p.sscale, -lr)) * dp : 0.f;
                    }
                }
                if (gl == 0) s_drem[warp * 32 + rl] = drem;
            }
        }
        // ---- S = Q K^T and dP = dO V^T on the tensor cores, one commit
        mbar_wait(full, (uint32_t)h & 1u);
        if (tid == 0) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
            for (int s = 0; s < D / 16; ++s)
                umma(tmem, make_desc_sw128(smem_u32(sQ) + s * 32, 1024), make_desc_sw128(smem_u32(sK) + s * 32, 1024), kIdescS, s > 0);
#pragma unroll
            for (int s = 0; s < D / 16; ++s)
                umma(tmem + 128, make_desc_sw128(smem_u32(sdO) + s * 32, 1024), make_desc_sw128(smem_u32(sV) + s * 32, 1024), kIdescS, s > 0);
            umma_commit(bar);
        }
        mbar_wait(bar, phase);
        phase ^= 1;
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        // ---- this row's diagonal block: P, the block part of Delta, then dS once Delta is complete
        float p16[16], w16[16];
        float ddiag = 0.f;
        const float lrow = rvalid ? __ldg(p.lse + (size_t)row * p.H + h) * kLog2e : 0.f;
        {
            float sv[32], tv[32];
            tmem_ld32(t_lane + warp * 32, sv);
            tmem_ld32(t_lane + 128 + warp * 32, tv);
#pragma unroll
            for (int c = 0; c < 16; ++c) {
                const float sc = (lane >= 16) ? sv[16 + c] : sv[c];
                const float tc_ = (lane >= 16) ? tv[16 + c] : tv[c];
                p16[c] = ((bits >> c) & 1u) ? ex2(fmaf(sc, p.sscale, -lrow)) : 0.f;
                w16[c] = tc_;
                ddiag = fmaf(p16[c], tc_, ddiag);
            }
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();                       // remainder parts of Delta are visible; every thread holds its S / dP values
        const float dl = ddiag + s_drem[tid];
        s_delta[tid] = dl;
        if (rvalid) {
            p.delta[(size_t)row * p.H + h] = dl;
            p.stat2[(size_t)row * p.H + h] = make_float2(lrow, dl);
        }
#pragma unroll
        for (int c = 0; c < 16; ++c) w16[c] = p16[c] * (w16[c] - dl);
        // one accumulating product with the staged block-diagonal A operand: TMEM[col0 ..] = W B
        auto mma2 = [&](uint8_t* sB, int col0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncthreads();
            if (tid == 0) {
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                for (int ks = 0; ks < kTile / 16; ++ks)
                    umma(tmem + col0, make_desc(smem_u32(sW) + ks * 256, 128, SBO_W),
                         make_desc_sw128(smem_u32(sB) + ks * 2048, 1024), kIdescO, ks > 0);
                umma_commit(bar);
            }
            mbar_wait(bar, phase);
            phase ^= 1;
        };
        // dQ_block = dS K: this row's 16 weights as a row of the tile
        {
            uint32_t pk[8];
#pragma unroll
            for (int c = 0; c < 16; c += 2) {
                const __nv_bfloat162 b2 = __floats2bfloat162_rn(w16[c], w16[c + 1]);
                pk[c >> 1] = *reinterpret_cast<const uint32_t*>(&b2);
            }
            uint8_t* prow = sW + canon(tid, 16 * wl, SBO_W);
            *reinterpret_cast<uint4*>(prow) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
            *reinterpret_cast<uint4*>(prow + 128) = make_uint4(pk[4], pk[5], pk[6], pk[7]);
        }
        mma2(sK, 0);
        // dK_block = dS^T Q and dV_block = P^T dO: this row's weights as a COLUMN of the window's block
#pragma unroll
        for (int c = 0; c < 16; ++c)
            *reinterpret_cast<__nv_bfloat16*>(sW + canon(16 * wl + c, tid, SBO_W)) = __float2bfloat16_rn(w16[c]);
        mma2(sQ, 64);
#pragma unroll
        for (int c = 0; c < 16; ++c)
            *reinterpret_cast<__nv_bfloat16*>(sW + canon(16 * wl + c, tid, SBO_W)) = __float2bfloat16_rn(p16[c]);
        mma2(sdO, 128);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");

        // ---- dQ: block part through the transpose slots, remainder terms and the store by 8 lanes per row
        float* sTw = sT + warp * 32 * kTS;
        float* slot = sTw + lane * kTS;
        const int row0w = row0 + warp * 32;
#pragma unroll
        for (int c0 = 0; c0 < D; c0 += 32) {
            float t32[32];
            tmem_ld32(t_lane + c0, t32);
            slot_write32(slot, c0, t32);
        }
        __syncwarp();
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            uint4 Lk0[4], Lk1[4];
#pragma unroll
            for (int ii = 0; ii < 4; ++ii) {
                const int i = 4 * half + ii;
                Lk0[ii] = Lk1[ii] = make_uint4(0, 0, 0, 0);
                if (cj0[i] >= 0) Lk0[ii] = __ldg(reinterpret_cast<const uint4*>(p.k + (size_t)cj0[i] * rowe + hoff) + gl);
                if (cj1[i] >= 0) Lk1[ii] = __ldg(reinterpret_cast<const uint4*>(p.k + (size_t)cj1[i] * rowe + hoff) + gl);
            }
#pragma unroll
            for (int ii = 0; ii < 4; ++ii) {
                const int i = 4 * half + ii;
                const int rl = g4 + 4 * i;
                const int rowc = row0w + rl;
                const bool cv = rowc < p.n;
                const float dlr = s_delta[warp * 32 + rl];
                const float4 b0 = *reinterpret_cast<const float4*>(sTw + rl * kTS + gl * 8);
                const float4 b1 = *reinterpret_cast<const float4*>(sTw + rl * kTS + gl * 8 + 4);
                float a[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
                axpy8(a, pr[i][0] * (dpr[i][0] - dlr), Lk0[ii]);
                axpy8(a, pr[i][1] * (dpr[i][1] - dlr), Lk1[ii]);
                int maxcnt = ccnt[i];
                maxcnt = max(maxcnt, __shfl_xor_sync(0xffffffffu, maxcnt, 8));
                maxcnt = max(maxcnt, __shfl_xor_sync(0xffffffffu, maxcnt, 16));
                if (maxcnt > 2) {
                    const int rbc = cv ? __ldg(p.rem_rowptr + rowc) : 0;
                    uint4 qq = make_uint4(0, 0, 0, 0), dd = qq;
                    float lr = 0.f;
                    if (ccnt[i] > 2) {
                        qq = __ldg(reinterpret_cast<const uint4*>(p.q + (size_t)rowc * rowe + hoff) + gl);
                        dd = __ldg(reinterpret_cast<const uint4*>(p.dout + (size_t)rowc * rowe + hoff) + gl);
                        lr = __ldg(p.lse + (size_t)rowc * p.H + h) * kLog2e;
                    }
                    for (int eb = 2; eb < maxcnt; ++eb) {
                        const int j = eb < ccnt[i] ? __ldg(p.rem_colidx + rbc + eb) : -1;
                        uint4 kk = make_uint4(0, 0, 0, 0), vv = kk;
                        if (j >= 0) {
                            kk = __ldg(reinterpret_cast<const uint4*>(p.k + (size_t)j * rowe + hoff) + gl);
                            vv = __ldg(reinterpret_cast<const uint4*>(p.v + (size_t)j * rowe + hoff) + gl);
                        }
                        const float s = red8(dot8(qq, kk)), dp = red8(dot8(dd, vv));
                        const float pe = j >= 0 ? ex2(fmaf(s, p.sscale, -lr)) : 0.f;
                        axpy8(a, pe * (dp - dlr), kk);
                    }
                }
                if (cv) {
                    float* dst = p.dq + (size_t)rowc * rowe + hoff + gl * 8;
                    *reinterpret_cast<float4*>(dst) = make_float4(a[0] * p.inv_sqrt_d, a[1] * p.inv_sqrt_d, a[2] * p.inv_sqrt_d, a[3] * p.inv_sqrt_d);
                    *reinterpret_cast<float4*>(dst + 4) = make_float4(a[4] * p.inv_sqrt_d, a[5] * p.inv_sqrt_d, a[6] * p.inv_sqrt_d, a[7] * p.inv_sqrt_d);
                }
            }
        }
        __syncwarp();
        // ---- tile-local dK, dV (the remainder src pass adds the out-of-window terms afterwards)
#pragma unroll
        for (int which = 0; which < 2; ++which) {
#pragma unroll
            for (int c0 = 0; c0 < D; c0 += 32) {
                float t32[32];
                tmem_ld32(t_lane + 64 + 64 * which + c0, t32);
                if (which == 0) {
#pragma unroll
                    for (int i = 0; i < 32; ++i) t32[i] *= p.inv_sqrt_d;
                }
                slot_write32(slot, c0, t32);
            }
            flush_rows<D, float>(sTw, (which ? p.dv : p.dk) + hoff, rowe, row0w, p.n, lane);
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic writes (slots, weights) before the next TMA
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
    }
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 256;" ::"r"(tmem) : "memory");
}

}  // namespace

cudaError_t launch_gt_bwd_block(const gnn_plan* P, const GtArgs& a, int heads, cudaStream_t st) {
    constexpr int D = 64;
    const int n = P->n;
    CUtensorMap tmq, tmk, tmv, tmdo;
    if (!tc::encode_row_tile_map(&tmq, a.q, n, heads * D, D, kTile) || !tc::encode_row_tile_map(&tmk, a.k, n, heads * D, D, kTile) ||
        !tc::encode_row_tile_map(&tmv, a.v, n, heads * D, D, kTile) || !tc::encode_row_tile_map(&tmdo, a.dout, n, heads * D, D, kTile))
        return cudaErrorNotSupported;
    BlockBwdParams p = {};
    p.q = (const __nv_bfloat16*)a.q; p.k = (const __nv_bfloat16*)a.k; p.v = (const __nv_bfloat16*)a.v;
    p.dout = (const __nv_bfloat16*)a.dout; p.lse = a.lse; p.bitmap = P->blk_bitmap;
    p.rem_rowptr = P->blk_rem_rowptr; p.rem_colidx = P->blk_rem_colidx;
    p.dq = a.dq; p.dk = a.dk; p.dv = a.dv; p.delta = a.delta; p.stat2 = a.stat2;
    p.n = n; p.H = heads; p.sscale = kLog2e / sqrtf((float)D); p.inv_sqrt_d = 1.f / sqrtf((float)D);
    const size_t smem = 4 * (size_t)kHT + kWBytes + 32 + 2 * kTile * 4 + 1024;
    cudaError_t e = cudaFuncSetAttribute(gt_bwd_block_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    prof_begin("gt_bwd_block", "tile", st);
    gt_bwd_block_kernel<D><<<(n + kTile - 1) / kTile, kTile, smem, st>>>(tmq, tmk, tmv, tmdo, p);
    prof_end(st);
    count_launch();
    return cudaGetLastError();
}

}  // namespace gnn
