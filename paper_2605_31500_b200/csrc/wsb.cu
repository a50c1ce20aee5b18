// wsb.cu - row f2: Graph Transformer attention on the paper's general WSB block-sparse layout,
// forward AND backward on the 5th-generation tensor cores (tcgen05.mma, accumulators in TMEM), atomics-free.
//
// Paper (A100, WMMA 16x16x16): one program per (16-row window, head) walks the window's TCB pairs, S = Q_win K_blk^T,
// bitmap mask, online softmax, acc += P V_blk; the backward reconstructs P = exp(S - L), dV = P^T dO,
// dP = dO V^T, dS = P o (dP - Delta), dQ = dS K, dK = dS^T Q with ATOMIC accumulation of dK / dV "because the same
// source columns can appear in multiple row windows", which is why the paper falls back to SpMM there.
//
// Here (B200): tcgen05.mma has M in {64, 128}, so one CTA of 128 threads owns a TILE of 128 rows = 8 row windows and
// walks the windows' TCB pairs in lock step: step s gathers, for every window, the 16 columns of its TCBs 2s and 2s+1
// (128 column slots per step; windows that have run out of TCBs contribute zero rows) into shared memory in the
// 128-byte-swizzled K-major layout the tensor core reads, and issues ONE 128x128xD product per operand pair; thread t
// owns tile row t (TMEM lane t) and reads back only the 16 columns of its own window (the other 7/8 of the product is
// masked waste, far below the gather time).  Three kernels share that skeleton:
//   forward            own Q tile (TMA), gathered K_c, V_c:  S = Q K_c^T -> online softmax -> P (bf16, block diagonal)
//                      -> O_step = P V_c -> acc = acc * corr + O_step in registers.
//   backward, dst side the SAME layout, own Q and dO tiles, gathered K_c, V_c: S = Q K_c^T, dP = dO V_c^T,
//                      P = exp(S - L_i); B += P K_c, A += [P o (dP - Delta~_i)] K_c in TMEM, Delta_i = sum P dP in fp32
//                      registers; dQ_i = (A - (Delta_i - Delta~_i) B) / sqrt(d).  Delta~_i = <O_i, dO_i> from the stored
//                      bf16 forward output is only a centring value (PAPER.md:494 uses it as Delta itself): it removes the
//                      cancellation between the two bf16-staged products, and the fp32 correction term makes the result
//                      independent of its rounding.  Row-local: no atomics.
//   backward, src side the layout of the TRANSPOSED graph (source windows x destination columns, built by the plan; the
//                      same arrays on an undirected graph), own K and V tiles, gathered Q_c, dO_c and the
//                      per-column (L_c, Delta_c): S^T = K Q_c^T, dP^T = V dO_c^T, P^T = exp(S^T - L_c);
//                      dV += P^T dO_c, dK += [P^T o (dP^T - Delta_c)] Q_c in TMEM.  Source rows own their gradients: no
//                      atomics and a fixed summation order, where the paper needs atomicAdd.
// Operands: own tiles arrive by TMA (cp.async.bulk.tensor.2d, SWIZZLE_128B); gathered tiles are written by the threads
// (8 lanes per 128-byte row slice, coalesced 16-byte loads, the same XOR swizzle); P / dS are staged as bf16 in the
// canonical no-swizzle K-major layout; V_c / K_c / Q_c / dO_c double as MN-major B operands of the second products.
// head_dim 32, 64 or 128 (128 = two 64-channel half tiles per operand; 32 = one half tile whose upper 32 channels are
// zeros, own rows placed by the threads instead of TMA); bf16 features; outputs leave through a per-warp
// shared-memory transpose so global stores are coalesced 16-byte pieces.
#include <cuda.h>
#include <cuda_bf16.h>

#include "internal.h"
#include "kernels.cuh"
#include "tc_common.cuh"

namespace gnn {
namespace {
using namespace tc;

#ifndef GNN_WSB_PF
#define GNN_WSB_PF 1
#endif
constexpr int kTile = 128;      // rows per CTA = MMA M = TMEM lanes
constexpr int kHT = 16384;      // bytes of a half tile: 128 rows x 64 channels bf16, 128-byte swizzled rows
constexpr int kWBytes = 32768;  // bytes of the block-diagonal 128 x 128 bf16 weight tile (P / dS)
enum { kFwd = 0, kBwdDst = 1, kBwdSrc = 2 };

struct WsbParams {
    const int32_t* row_offset;       // WSB of the graph the kernel walks (CSR for fwd / dst side, CSR^T for src side)
    const int32_t* cols;
    const uint8_t* bitmap;
    int n_win, n, H;
    const __nv_bfloat16 *ox, *oy;    // own operands of the two products (what tmx / tmy map; read directly when head_dim = 32)
    const __nv_bfloat16* gx;         // gathered operand of the first product  (fwd / dst: K, src: Q)
    const __nv_bfloat16* gy;         // gathered operand of the second product (fwd / dst: V, src: dO)
    const __nv_bfloat16* o;          // dst: stored forward output; dout for the Delta~ estimate comes from gdo
    const __nv_bfloat16* gdo;        // dst: dO (row-wise reads for Delta~)
    const float* lse;                // [n, H] natural-log L of the forward
    const float* delta_in;           // src: Delta [n, H] from the dst side
    __nv_bfloat16* out;              // fwd: O
    float* lse_out;                  // fwd: L
    float* o1;                       // dst: dQ, src: dV
    float* o2;                       // src: dK
    float* delta_out;                // dst: Delta
    float sscale;                    // log2(e) / sqrt(d)
    float inv_sqrt_d;
};

// one 128-row tile of `g` (rows s_col[0..128), -1 = zero row) -> NH half tiles at sT, 128-byte swizzled K-major
// (NCH = valid 16-byte chunks of a row slice: 8, or 4 for head_dim 32, whose upper 32 channels of the tile are zeros)
template <int NH, int NCH>
__device__ __forceinline__ void gather_tile(uint8_t* sT, const __nv_bfloat16* __restrict__ g, const int* s_col, size_t rowe,
                                            int hoff, int tid) {
    const int c = tid & 7, rb = tid >> 3;
    uint4 v[8 * NH];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int col = s_col[rb + 16 * i];
#pragma unroll
        for (int hf = 0; hf < NH; ++hf) {
            v[i * NH + hf] = make_uint4(0, 0, 0, 0);
            if (col >= 0 && c < NCH) v[i * NH + hf] = __ldg(reinterpret_cast<const uint4*>(g + (size_t)col * rowe + hoff + hf * 64) + c);
        }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int row = rb + 16 * i;
#pragma unroll
        for (int hf = 0; hf < NH; ++hf)
            *reinterpret_cast<uint4*>(sT + hf * kHT + (row >> 3) * 1024 + (row & 7) * 128 + ((c ^ (row & 7)) << 4)) = v[i * NH + hf];
    }
}

// this row's 16 weights (window columns 16*wl .. +15) into the block-diagonal canonical K-major tile
__device__ __forceinline__ void write_block(uint8_t* sW, int tid, int wl, const uint32_t (&pk)[8]) {
    constexpr int SBO = (kTile / 8) * 128;
    uint8_t* prow = sW + canon(tid, 16 * wl, SBO);
    *reinterpret_cast<uint4*>(prow) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
    *reinterpret_cast<uint4*>(prow + 128) = make_uint4(pk[4], pk[5], pk[6], pk[7]);
}

template <int MODE, int D>
__global__ void __launch_bounds__(kTile, (MODE == kFwd && D <= 64) ? 3 : (D <= 64 ? 2 : 1))
wsb_kernel(const __grid_constant__ CUtensorMap tmx, const __grid_constant__ CUtensorMap tmy, const WsbParams p) {
    constexpr int NH = D >= 64 ? D / 64 : 1;      // half tiles per operand; head_dim 32 = one half tile, upper channels zero
    constexpr int DP = NH * 64;                   // tile width in channels
    constexpr int NCH = D >= 64 ? 8 : D / 8;      // valid 16-byte chunks per row slice
    constexpr bool BWD = MODE != kFwd;
    constexpr int kOwnBytes = (BWD ? 2 : 1) * NH * kHT;
    constexpr int kPadBytes = (!BWD && NH * kHT < kWBytes) ? kWBytes - NH * kHT : 0;   // fwd: P aliases K (+ pad)
    constexpr int kTmemCols = BWD ? (DP == 64 ? 256 : 512) : 128;
    constexpr int kColAcc1 = 128, kColAcc2 = 128 + DP;
    constexpr int SBO_W = (kTile / 8) * 128;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint8_t* sX = smem;                                   // own tile of the first product (Q | K)
    uint8_t* sY = sX + NH * kHT;                          // own tile of the second product (bwd: dO | V)
    uint8_t* sGx = smem + kOwnBytes;                      // gathered tile of the first product
    uint8_t* sGy = sGx + NH * kHT + kPadBytes;            // gathered tile of the second product
    uint8_t* sW = BWD ? sGy + NH * kHT : sGx;             // block-diagonal weights (fwd: over the dead K tile)
    uint8_t* tail = BWD ? sW + kWBytes : sGy + NH * kHT;
    uint64_t* full = reinterpret_cast<uint64_t*>(tail);   // TMA completion
    uint64_t* bar = full + 1;                             // tcgen05.commit
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar + 1);
    int* s_col = reinterpret_cast<int*>(tail + 32);       // [128] column id of every slot of the step (-1: none)
    float2* s_stat = reinterpret_cast<float2*>(s_col + kTile);   // src side: (L_c log2e, Delta_c) per slot
    int* s_red = reinterpret_cast<int*>(s_stat + kTile);  // [4]
    float* s_dt = reinterpret_cast<float*>(s_red + 4);    // dst side: Delta~ per row [128]
    float* sT = reinterpret_cast<float*>(smem);           // transpose slots (over the dead operand tiles)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int row0 = blockIdx.x * kTile, row = row0 + tid;
    const bool rvalid = row < p.n;
    const int wl = tid >> 4, rr = tid & 15;
    const size_t rowe = (size_t)p.H * D;

    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_init(full, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(kTmemCols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (BWD) {   // the off-diagonal blocks of the weight tile stay zero for the whole kernel
#pragma unroll
        for (int it = 0; it < kWBytes / (kTile * 16); ++it)
            *reinterpret_cast<uint4*>(sW + (it * kTile + tid) * 16) = make_uint4(0, 0, 0, 0);
    }
    // TCB range of this thread's window, and the number of steps of the tile
    const int gw = blockIdx.x * (kTile / 16) + wl;
    const int t0 = gw < p.n_win ? __ldg(p.row_offset + gw) : 0;
    const int t1 = gw < p.n_win ? __ldg(p.row_offset + gw + 1) : 0;
    int nst = (t1 - t0 + 1) >> 1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) nst = max(nst, __shfl_xor_sync(0xffffffffu, nst, o));
    if (lane == 0) s_red[warp] = nst;
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const int n_steps = max(max(s_red[0], s_red[1]), max(s_red[2], s_red[3]));
    const uint32_t tmem = *tmem_slot;
    const uint32_t t_lane = tmem + ((uint32_t)(warp * 32) << 16);
    uint32_t phase = 0;
    constexpr uint32_t kIdescS = make_idesc(kTile, kTile, false), kIdescO = make_idesc(kTile, 64, true);

    for (int h = 0; h < p.H; ++h) {
        const int hoff = h * D;
        // ---- own tiles of this head by TMA (rows past n arrive as zeros)
        if (D >= 64 && tid == 0) {
            mbar_expect_tx(full, kOwnBytes);
#pragma unroll
            for (int hf = 0; hf < NH; ++hf) {
                tma_load_2d(sX + hf * kHT, &tmx, hoff + hf * 64, row0, full);
                if (BWD) tma_load_2d(sY + hf * kHT, &tmy, hoff + hf * 64, row0, full);
            }
        }
        // ---- per-row statistics
        float m = -INFINITY, l = 0.f, lx = 0.f;      // fwd: running max (log2 domain), sum of rounded / exact weights
        float acc[MODE == kFwd ? D : 1];
#pragma unroll
        for (int c = 0; c < (MODE == kFwd ? D : 1); ++c) acc[c] = 0.f;
        float lrow = 0.f, dtil = 0.f, dacc = 0.f;    // dst: L_i log2e, Delta~_i, Delta_i
        if (MODE == kBwdDst) {
            lrow = rvalid ? __ldg(p.lse + (size_t)row * p.H + h) * kLog2e : 0.f;
            // Delta~ = <O_i, dO_i> from the stored bf16 rows, 8 lanes per row (coalesced 128-byte slices)
            const int c8 = lane & 7;
#pragma unroll
            for (int it = 0; it < 8; ++it) {
                const int rl = it * 4 + (lane >> 3);
                const int rg = row0 + warp * 32 + rl;
                float d0 = 0.f, d1 = 0.f;
                if (rg < p.n) {
#pragma unroll
                    for (int hf = 0; hf < NH; ++hf) {
                        if (c8 >= NCH) continue;
                        const uint4 a = __ldg(reinterpret_cast<const uint4*>(p.o + (size_t)rg * rowe + hoff + hf * 64) + c8);
                        const uint4 b = __ldg(reinterpret_cast<const uint4*>(p.gdo + (size_t)rg * rowe + hoff + hf * 64) + c8);
                        fma_bf16x2(a.x, b.x, d0, d1); fma_bf16x2(a.y, b.y, d0, d1);
                        fma_bf16x2(a.z, b.z, d0, d1); fma_bf16x2(a.w, b.w, d0, d1);
                    }
                }
                d0 += d1;
#pragma unroll
                for (int o = 1; o < 8; o <<= 1) d0 += __shfl_xor_sync(0xffffffffu, d0, o);
                if (c8 == 0) s_dt[warp * 32 + rl] = d0;
            }
            __syncwarp();
            dtil = s_dt[tid];
        }
        if constexpr (D >= 64) {
            mbar_wait(full, (uint32_t)h & 1u);
        } else {
            // head_dim 32: a 64-byte head slice is no TMA box of the 128-byte-swizzled tile; the threads place the own
            // rows themselves, upper 32 channels zero (made visible to the tensor core by the fence of the first step)
            s_col[tid] = rvalid ? row : -1;
            __syncthreads();
            gather_tile<NH, NCH>(sX, p.ox, s_col, rowe, hoff, tid);
            if (BWD) gather_tile<NH, NCH>(sY, p.oy, s_col, rowe, hoff, tid);
            __syncthreads();
        }

        for (int s = 0; s < n_steps; ++s) {
            // ---- column of this thread's slot (window wl, position rr of the TCB pair) and this row's 16 mask bits
            const int ta = t0 + 2 * s;
            int col = -1;
            {
                const int tcb = ta + (rr >> 3);
                if (tcb < t1) col = __ldg(p.cols + (size_t)tcb * 8 + (rr & 7));
            }
            s_col[tid] = col;
            if (MODE == kBwdSrc) {
                float2 st = make_float2(0.f, 0.f);
                if (col >= 0) {
                    st.x = __ldg(p.lse + (size_t)col * p.H + h) * kLog2e;
                    st.y = __ldg(p.delta_in + (size_t)col * p.H + h);
                }
                s_stat[tid] = st;
            }
            uint32_t bits = 0;
            if (ta < t1) bits = __ldg(p.bitmap + (size_t)ta * 16 + rr);
            if (ta + 1 < t1) bits |= (uint32_t)__ldg(p.bitmap + (size_t)(ta + 1) * 16 + rr) << 8;
            if (!rvalid) bits = 0;
            __syncthreads();
            // ---- the row slices the NEXT step (or the next head's first step) will gather: into L2 now, so that its
            // gathers do not pay the DRAM latency inside the serial phase chain (every gathered line is a DRAM miss:
            // each (row, head) slice is one 128-byte line used by one window; GNN_WSB_PF=0 switches this off)
            if (GNN_WSB_PF) {
                const bool nh = s + 1 >= n_steps;               // wraps to the next head
                const int sn = nh ? 0 : s + 1, hn = nh ? hoff + D : hoff;
                const int tcb = t0 + 2 * sn + (rr >> 3);
                if (tcb < t1 && (!nh || h + 1 < p.H)) {
                    const size_t off = (size_t)__ldg(p.cols + (size_t)tcb * 8 + (rr & 7)) * rowe + hn;
#pragma unroll
                    for (int hf = 0; hf < NH; ++hf) {
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(p.gx + off + hf * 64));
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(p.gy + off + hf * 64));
                    }
                }
            }
            // ---- gathered tiles
            gather_tile<NH, NCH>(sGx, p.gx, s_col, rowe, hoff, tid);
            gather_tile<NH, NCH>(sGy, p.gy, s_col, rowe, hoff, tid);
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncthreads();
            // ---- S = X_own Xc^T
            if (tid == 0) {
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                for (int hf = 0; hf < NH; ++hf)
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks)
                        umma(tmem, make_desc_sw128(smem_u32(sX + hf * kHT) + ks * 32, 1024),
                             make_desc_sw128(smem_u32(sGx + hf * kHT) + ks * 32, 1024), kIdescS, (hf | ks) > 0);
                umma_commit(bar);
            }
            mbar_wait(bar, phase);
            phase ^= 1;
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            float s16[16];
            {
                float sv[32];
                tmem_ld32(t_lane + warp * 32, sv);
#pragma unroll
                for (int c = 0; c < 16; ++c) s16[c] = (lane >= 16) ? sv[16 + c] : sv[c];
            }
            uint32_t pk[8];
            if constexpr (MODE == kFwd) {
                float mx = m;
#pragma unroll
                for (int c = 0; c < 16; ++c) {
                    s16[c] = ((bits >> c) & 1u) ? s16[c] * p.sscale : -INFINITY;
                    mx = fmaxf(mx, s16[c]);
                }
                const float ms = (mx == -INFINITY) ? 0.f : mx;
                const float corr = ex2(m - ms);
                float ls = 0.f, lxs = 0.f;
#pragma unroll
                for (int c = 0; c < 16; c += 2) {
                    const float p0 = ex2(s16[c] - ms), p1 = ex2(s16[c + 1] - ms);
                    const __nv_bfloat162 pb = __floats2bfloat162_rn(p0, p1);
                    ls += __low2float(pb) + __high2float(pb);   // O is normalised with the rounded weights the MMA uses
                    lxs += p0 + p1;
                    pk[c >> 1] = *reinterpret_cast<const uint32_t*>(&pb);
                }
                l = l * corr + ls;
                lx = lx * corr + lxs;
                m = mx;
                // P overwrites the dead K tile: the warp clears its own 8 KB, then every lane writes its diagonal block
#pragma unroll
                for (int it = 0; it < 16; ++it)
                    *reinterpret_cast<uint4*>(sW + warp * 8192 + (it * 32 + lane) * 16) = make_uint4(0, 0, 0, 0);
                __syncwarp();
                write_block(sW, tid, wl, pk);
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncthreads();
                // ---- O_step = P V_c (overwrites the S columns: every thread has read its scores)
                if (tid == 0) {
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                    for (int hf = 0; hf < NH; ++hf)
#pragma unroll
                        for (int ks = 0; ks < kTile / 16; ++ks)
                            umma(tmem + hf * 64, make_desc(smem_u32(sW) + ks * 256, 128, SBO_W),
                                 make_desc_sw128(smem_u32(sGy + hf * kHT) + ks * 2048, 1024), kIdescO, ks > 0);
                    umma_commit(bar);
                }
                mbar_wait(bar, phase);
                phase ^= 1;
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                for (int c0 = 0; c0 < D; c0 += 32) {
                    float t32[32];
                    tmem_ld32(t_lane + c0, t32);
#pragma unroll
                    for (int i = 0; i < 32; ++i) acc[c0 + i] = fmaf(acc[c0 + i], corr, t32[i]);
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncthreads();
            } else {
                // ---- T = Y_own Yc^T into the same TMEM columns once every thread holds its scores
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncthreads();
                if (tid == 0) {
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                    for (int hf = 0; hf < NH; ++hf)
#pragma unroll
                        for (int ks = 0; ks < 4; ++ks)
                            umma(tmem, make_desc_sw128(smem_u32(sY + hf * kHT) + ks * 32, 1024),
                                 make_desc_sw128(smem_u32(sGy + hf * kHT) + ks * 32, 1024), kIdescS, (hf | ks) > 0);
                    umma_commit(bar);
                }
                mbar_wait(bar, phase);
                phase ^= 1;
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                float t16[16];
                {
                    float sv[32];
                    tmem_ld32(t_lane + warp * 32, sv);
#pragma unroll
                    for (int c = 0; c < 16; ++c) t16[c] = (lane >= 16) ? sv[16 + c] : sv[c];
                }
                // weights of the two accumulating products, staged as bf16 (tcgen05 wants A and B in one format).  The
                // src side sums over the destinations of a SOURCE - unbounded for a hub, unlike the convex row sums of
                // the dst side - so there every weight is staged as hi + lo bf16 parts (16 significant bits): the sums
                // stay inside the tolerance at any degree (a single bf16 rounding of P cost 2.6e-2 on a 700-edge hub).
                uint32_t pk2[8], pkl[MODE == kBwdSrc ? 8 : 1], pk2l[MODE == kBwdSrc ? 8 : 1];
#pragma unroll
                for (int c = 0; c < 16; c += 2) {
                    float pw[2], w2[2];
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
                        const bool on = (bits >> (c + u)) & 1u;
                        float lref = lrow, dref = dtil;
                        if (MODE == kBwdSrc) {
                            const float2 st = s_stat[16 * wl + c + u];
                            lref = st.x;
                            dref = st.y;
                        }
                        pw[u] = on ? ex2(fmaf(s16[c + u], p.sscale, -lref)) : 0.f;
                        if (MODE == kBwdDst) dacc = fmaf(pw[u], t16[c + u], dacc);
                        w2[u] = pw[u] * (t16[c + u] - dref);
                    }
                    const __nv_bfloat162 a = __floats2bfloat162_rn(pw[0], pw[1]), b = __floats2bfloat162_rn(w2[0], w2[1]);
                    pk[c >> 1] = *reinterpret_cast<const uint32_t*>(&a);
                    pk2[c >> 1] = *reinterpret_cast<const uint32_t*>(&b);
                    if constexpr (MODE == kBwdSrc) {
                        const __nv_bfloat162 al = __floats2bfloat162_rn(pw[0] - __low2float(a), pw[1] - __high2float(a));
                        const __nv_bfloat162 bl = __floats2bfloat162_rn(w2[0] - __low2float(b), w2[1] - __high2float(b));
                        pkl[c >> 1] = *reinterpret_cast<const uint32_t*>(&al);
                        pk2l[c >> 1] = *reinterpret_cast<const uint32_t*>(&bl);
                    }
                }
                // one accumulating product: stage this row's block, Acc[col0 ..] (+)= W Z, wait until the tile is free again
                auto stage2 = [&](const uint32_t (&blk)[8], uint8_t* sZ, int col0, bool first) {
                    write_block(sW, tid, wl, blk);
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                    __syncthreads();
                    if (tid == 0) {
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                        for (int hf = 0; hf < NH; ++hf)
#pragma unroll
                            for (int ks = 0; ks < kTile / 16; ++ks)
                                umma(tmem + col0 + hf * 64, make_desc(smem_u32(sW) + ks * 256, 128, SBO_W),
                                     make_desc_sw128(smem_u32(sZ + hf * kHT) + ks * 2048, 1024), kIdescO, !first || (ks > 0));
                        umma_commit(bar);
                    }
                    mbar_wait(bar, phase);
                    phase ^= 1;
                };
                // Acc1 += P Z1 (dst: B = sum P K_c; src: dV = sum P^T dO_c); Acc2 += W2 Xc (dst: A = sum P (dP - Delta~) K_c;
                // src: dK = sum dS^T Q_c)
                stage2(pk, MODE == kBwdSrc ? sGy : sGx, kColAcc1, s == 0);
                if constexpr (MODE == kBwdSrc) stage2(pkl, sGy, kColAcc1, false);
                stage2(pk2, sGx, kColAcc2, s == 0);
                if constexpr (MODE == kBwdSrc) stage2(pk2l, sGx, kColAcc2, false);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            }
        }
        // ---- results of this head: thread-row values -> per-warp transpose slots -> coalesced stores
        float* sTw = sT + warp * 32 * (D + 4);
        float* slot = sTw + lane * (D + 4);
        const int row0w = row0 + warp * 32;
        if constexpr (MODE == kFwd) {
            const float inv = l > 0.f ? 1.f / l : 0.f;
#pragma unroll
            for (int c0 = 0; c0 < D; c0 += 32) {
                float t32[32];
#pragma unroll
                for (int i = 0; i < 32; ++i) t32[i] = acc[c0 + i] * inv;
                slot_write32(slot, c0, t32);
            }
            flush_rows<D, __nv_bfloat16>(sTw, p.out + hoff, rowe, row0w, p.n, lane);
            if (rvalid) p.lse_out[(size_t)row * p.H + h] = lx > 0.f ? (m + lg2(lx)) * kLn2 : -INFINITY;
        } else if constexpr (MODE == kBwdDst) {
            const float corr = dacc - dtil;      // exact Delta minus the centring value
#pragma unroll
            for (int c0 = 0; c0 < D; c0 += 32) {
                float a1[32], a2[32];
                if (n_steps > 0) {
                    tmem_ld32(t_lane + kColAcc1 + c0, a1);
                    tmem_ld32(t_lane + kColAcc2 + c0, a2);
                }
#pragma unroll
                for (int i = 0; i < 32; ++i) a2[i] = n_steps > 0 ? (a2[i] - corr * a1[i]) * p.inv_sqrt_d : 0.f;
                slot_write32(slot, c0, a2);
            }
            flush_rows<D, float>(sTw, p.o1 + hoff, rowe, row0w, p.n, lane);
            if (rvalid) p.delta_out[(size_t)row * p.H + h] = dacc;
        } else {
#pragma unroll
            for (int which = 0; which < 2; ++which) {
#pragma unroll
                for (int c0 = 0; c0 < D; c0 += 32) {
                    float a[32];
                    if (n_steps > 0) tmem_ld32(t_lane + (which ? kColAcc2 : kColAcc1) + c0, a);
#pragma unroll
                    for (int i = 0; i < 32; ++i) a[i] = n_steps > 0 ? a[i] * (which ? p.inv_sqrt_d : 1.f) : 0.f;
                    slot_write32(slot, c0, a);
                }
                flush_rows<D, float>(sTw, (which ? p.o2 : p.o1) + hoff, rowe, row0w, p.n, lane);
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic writes (transpose slots) before the next TMA
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
    }
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kTmemCols) : "memory");
}

template <int MODE, int D> size_t wsb_smem_bytes() {
    constexpr int NH = D >= 64 ? D / 64 : 1;
    constexpr bool BWD = MODE != kFwd;
    const size_t own = (size_t)(BWD ? 2 : 1) * NH * kHT;
    const size_t pad = (!BWD && NH * kHT < kWBytes) ? kWBytes - NH * kHT : 0;
    const size_t tiles = own + 2 * (size_t)NH * kHT + pad + (BWD ? kWBytes : 0);
    const size_t tail = 32 + kTile * 4 + kTile * 8 + 16 + kTile * 4;
    const size_t tr = (size_t)kTile * (D + 4) * 4;       // transpose slots alias the operand tiles
    return (tiles > tr ? tiles : tr) + tail + 1024;
}

template <int MODE, int D>
cudaError_t launch_wsb(const CUtensorMap& tmx, const CUtensorMap& tmy, const WsbParams& p, const char* name, cudaStream_t st) {
    const size_t smem = wsb_smem_bytes<MODE, D>();
    cudaError_t e = cudaFuncSetAttribute(wsb_kernel<MODE, D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int grid = (p.n + kTile - 1) / kTile;
    prof_begin(name, "tile", st);
    wsb_kernel<MODE, D><<<grid, kTile, smem, st>>>(tmx, tmy, p);
    prof_end(st);
    count_launch();
    return cudaGetLastError();
}

bool wsb_check(const gnn_plan* P, const int32_t* rowptr, const int32_t* colidx, int32_t n, int32_t heads, int32_t head_dim,
               int dtype, bool backward, const char* who, gnn_status_t& rc) {
    rc = GNN_EINVAL;
    if (!P || rowptr != P->rowptr || colidx != P->colidx || n != P->n) {
        set_error("%s: NULL plan, or rowptr/colidx/n differ from the arrays the plan was built from", who);
        return false;
    }
    if (!P->has_wsb) { set_error("%s: plan was built without GNN_BLOCKS_WSB", who); return false; }
    if (backward && !P->opts.build_transpose) { set_error("%s: plan was built without build_transpose", who); return false; }
    rc = GNN_EUNSUPPORTED;
    if (P->wsb.n_dup > 0 || (backward && P->wsb_t.n_dup > 0)) {
        set_error("%s: the CSR holds %d duplicate entries; a WSB bitmap stores each (dst, src) pair once - use the CSR entry points", who,
                  P->wsb.n_dup);
        return false;
    }
    if (dtype != GNN_BF16 || (head_dim != 32 && head_dim != 64 && head_dim != 128) || heads < 1) {
        set_error("%s: unsupported shape heads=%d head_dim=%d dtype=%d (bf16, head_dim 32, 64 or 128)", who, heads, head_dim, dtype);
        return false;
    }
    rc = GNN_OK;
    return true;
}

}  // namespace
}  // namespace gnn

using namespace gnn;

extern "C" gnn_status_t gnn_gt_attn_fwd_wsb(const gnn_plan_t* P, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                            const void* q, const void* k, const void* v, int32_t heads, int32_t head_dim,
                                            gnn_dtype_t dtype, void* out, float* lse, gnn_stream_t stream) {
    const char* who = "gnn_gt_attn_fwd_wsb";
    gnn_status_t rc;
    if (!wsb_check(P, rowptr, colidx, n, heads, head_dim, dtype, false, who, rc)) return rc;
    if (!q || !k || !v || !out || !lse) { set_error("%s: NULL pointer argument", who); return GNN_EINVAL; }
    if ((((uintptr_t)q | (uintptr_t)k | (uintptr_t)v | (uintptr_t)out) & 31) != 0) {
        set_error("%s: feature pointers must be 32-byte aligned", who);
        return GNN_EINVAL;
    }
    CUtensorMap tmq;
    if (!tc::encode_row_tile_map(&tmq, q, n, heads * head_dim, head_dim < 64 ? head_dim : 64, kTile)) {
        set_error("%s: cuTensorMapEncodeTiled unavailable or failed", who);
        return GNN_ECUDA;
    }
    WsbParams p = {};
    p.row_offset = P->wsb.row_offset; p.cols = P->wsb.cols; p.bitmap = P->wsb.bitmap;
    p.n_win = (n + 15) / 16; p.n = n; p.H = heads;
    p.gx = (const __nv_bfloat16*)k; p.gy = (const __nv_bfloat16*)v;
    p.ox = (const __nv_bfloat16*)q; p.oy = nullptr;
    p.out = (__nv_bfloat16*)out; p.lse_out = lse;
    p.sscale = kLog2e / sqrtf((float)head_dim); p.inv_sqrt_d = 1.f / sqrtf((float)head_dim);
    cudaError_t e = head_dim == 64   ? launch_wsb<kFwd, 64>(tmq, tmq, p, "gt_fwd_wsb", (cudaStream_t)stream)
                    : head_dim == 128 ? launch_wsb<kFwd, 128>(tmq, tmq, p, "gt_fwd_wsb", (cudaStream_t)stream)
                                      : launch_wsb<kFwd, 32>(tmq, tmq, p, "gt_fwd_wsb", (cudaStream_t)stream);
    if (e != cudaSuccess) { set_error("%s: CUDA error: %s", who, cudaGetErrorString(e)); return GNN_ECUDA; }
    return GNN_OK;
}

extern "C" gnn_status_t gnn_gt_attn_bwd_wsb(const gnn_plan_t* P, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                            const void* q, const void* k, const void* v, const void* out, const float* lse,
                                            const void* dout, int32_t heads, int32_t head_dim, gnn_dtype_t dtype,
                                            float* delta, float* dq, float* dk, float* dv, gnn_stream_t stream) {
    const char* who = "gnn_gt_attn_bwd_wsb";
    gnn_status_t rc;
    if (!wsb_check(P, rowptr, colidx, n, heads, head_dim, dtype, true, who, rc)) return rc;
    if (!q || !k || !v || !out || !lse || !dout || !delta || !dq || !dk || !dv) {
        set_error("%s: NULL pointer argument", who);
        return GNN_EINVAL;
    }
    if ((((uintptr_t)q | (uintptr_t)k | (uintptr_t)v | (uintptr_t)out | (uintptr_t)dout | (uintptr_t)dq | (uintptr_t)dk |
          (uintptr_t)dv) & 31) != 0) {
        set_error("%s: feature / gradient pointers must be 32-byte aligned", who);
        return GNN_EINVAL;
    }
    const int R = heads * head_dim, bc = head_dim < 64 ? head_dim : 64;
    CUtensorMap tmq, tmdo, tmk, tmv;
    if (!tc::encode_row_tile_map(&tmq, q, n, R, bc, kTile) || !tc::encode_row_tile_map(&tmdo, dout, n, R, bc, kTile) ||
        !tc::encode_row_tile_map(&tmk, k, n, R, bc, kTile) || !tc::encode_row_tile_map(&tmv, v, n, R, bc, kTile)) {
        set_error("%s: cuTensorMapEncodeTiled unavailable or failed", who);
        return GNN_ECUDA;
    }
    cudaStream_t st = (cudaStream_t)stream;
    WsbParams p = {};
    p.n_win = (n + 15) / 16; p.n = n; p.H = heads;
    p.lse = lse;
    p.sscale = kLog2e / sqrtf((float)head_dim); p.inv_sqrt_d = 1.f / sqrtf((float)head_dim);
    // dst side over the WSB of the CSR: Delta, dQ
    p.row_offset = P->wsb.row_offset; p.cols = P->wsb.cols; p.bitmap = P->wsb.bitmap;
    p.gx = (const __nv_bfloat16*)k; p.gy = (const __nv_bfloat16*)v;
    p.o = (const __nv_bfloat16*)out; p.gdo = (const __nv_bfloat16*)dout;
    p.ox = (const __nv_bfloat16*)q; p.oy = (const __nv_bfloat16*)dout;
    p.o1 = dq; p.delta_out = delta;
    cudaError_t e = head_dim == 64   ? launch_wsb<kBwdDst, 64>(tmq, tmdo, p, "gt_bwd_wsb_dst", st)
                    : head_dim == 128 ? launch_wsb<kBwdDst, 128>(tmq, tmdo, p, "gt_bwd_wsb_dst", st)
                                      : launch_wsb<kBwdDst, 32>(tmq, tmdo, p, "gt_bwd_wsb_dst", st);
    // src side over the WSB of CSR^T: dK, dV
    if (e == cudaSuccess) {
        p.row_offset = P->wsb_t.row_offset; p.cols = P->wsb_t.cols; p.bitmap = P->wsb_t.bitmap;
        p.gx = (const __nv_bfloat16*)q; p.gy = (const __nv_bfloat16*)dout;
        p.ox = (const __nv_bfloat16*)k; p.oy = (const __nv_bfloat16*)v;
        p.delta_in = delta; p.o1 = dv; p.o2 = dk;
        e = head_dim == 64   ? launch_wsb<kBwdSrc, 64>(tmk, tmv, p, "gt_bwd_wsb_src", st)
            : head_dim == 128 ? launch_wsb<kBwdSrc, 128>(tmk, tmv, p, "gt_bwd_wsb_src", st)
                              : launch_wsb<kBwdSrc, 32>(tmk, tmv, p, "gt_bwd_wsb_src", st);
    }
    if (e != cudaSuccess) { set_error("%s: CUDA error: %s", who, cudaGetErrorString(e)); return GNN_ECUDA; }
    return GNN_OK;
}
