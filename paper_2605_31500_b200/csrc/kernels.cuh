// kernels.cuh - the three traversal kernels + launcher, generic over an Op (see ops.cuh).
#pragma once
#include "engine.cuh"

namespace gnn {

// optional per-launch CUDA-event timing (gnn_profile_enable); no-ops when disabled
void prof_begin(const char* pass, const char* kernel, cudaStream_t st);
void prof_end(cudaStream_t st);
bool prof_enabled();
// programmatic dependent launch of a pass's group kernel behind its segment kernel (tuning knob, on by default)
#ifndef GNN_PDL
#define GNN_PDL 1
#endif

// lexicographic (value, index) order of the MINARG states; index < 0 marks "no candidate yet"
__device__ __forceinline__ bool minarg_better(float v, int j, float bv, int bj) {
    return j >= 0 && (bj < 0 || v < bv || (v == bv && j < bj));
}

// ------------------------------------------------------------------------------------------------
// state <-> shared memory (serialised layout of state_floats<Op>)
template <class Op> __device__ __forceinline__ void state_to_smem(const typename Op::St& st, float* dst,
                                                                  const typename Op::GeoT& g, const Shape& sh) {
    constexpr int CH = Op::kCH;
    if (g.act) {
#pragma unroll
        for (int a = 0; a < Op::NA; ++a)
#pragma unroll
            for (int c = 0; c < CH; c += 4)
                *reinterpret_cast<float4*>(dst + a * sh.rowe + g.eoff + c) =
                    make_float4(st.acc[a][c], st.acc[a][c + 1], st.acc[a][c + 2], st.acc[a][c + 3]);
    }
    if (g.lead) {
#pragma unroll
        for (int s = 0; s < Op::NS; ++s) dst[Op::NA * sh.rowe + s * sh.H + g.hd] = st.sc[s];
    }
}

template <class Op> __device__ __forceinline__ void state_from_smem(typename Op::St& st, const float* src,
                                                                    const typename Op::GeoT& g, const Shape& sh) {
    constexpr int CH = Op::kCH;
#pragma unroll
    for (int a = 0; a < Op::NA; ++a)
#pragma unroll
        for (int c = 0; c < CH; ++c) st.acc[a][c] = g.act ? src[a * sh.rowe + g.eoff + c] : 0.f;
#pragma unroll
    for (int s = 0; s < Op::NS; ++s) st.sc[s] = g.act ? src[Op::NA * sh.rowe + s * sh.H + g.hd] : 0.f;
    if (Op::SOFTMAX) st.m = g.act ? src[Op::NA * sh.rowe + Op::NS * sh.H + g.hd] : -INFINITY;
}

// per-CTA reduction of the per-thread `da` accumulators (GATv2 dst pass) -> da_part[slot][rowe],
// fixed order over groups.  smem: NG * rowe floats.
template <class Op>
__device__ __forceinline__ void cta_write_da(const float (&da)[Op::kCH], float* smem, float* da_part, int slot,
                                             const typename Op::GeoT& g, const Shape& sh, int gi, int ng) {
    constexpr int CH = Op::kCH;
    __syncthreads();
    if (g.act) {
#pragma unroll
        for (int c = 0; c < CH; ++c) smem[gi * sh.rowe + g.eoff + c] = da[c];
    }
    __syncthreads();
    for (int e = threadIdx.x; e < sh.rowe; e += blockDim.x) {
        float s = 0.f;
        for (int k = 0; k < ng; ++k) s += smem[k * sh.rowe + e];
        da_part[(size_t)slot * sh.rowe + e] = s;
    }
}

// ------------------------------------------------------------------------------------------------
// The edge loop of one lane group: blocks of G edges (block k = [ebeg + k*stride, +G), clipped to eend), cut
// into batches of KU edges.  The gathers of batch t+1 are issued (into a second register set) before batch t
// is computed, and the colidx words of the next block are fetched one block ahead.  nblk and cnt_last (edges to
// cover in the last block) are warp-uniform; groups with fewer edges see masked (-1) neighbours.
template <class Op>
__device__ __forceinline__ void run_edges(typename Op::St& st, const typename Op::Own& own, const typename Op::Params& p,
                                          const Shape& sh, const typename Op::GeoT& g,
                                          const int32_t* __restrict__ colidx, int ebeg, int eend, int stride, int nblk,
                                          int cnt_last) {
    constexpr int G = Op::kG, KU = Op::kU, BPB = G / KU;
    static_assert(G % KU == 0, "KU must divide G");
    if (nblk <= 0) return;
    const int gl = threadIdx.x & (G - 1);
    const int T = (nblk - 1) * BPB + (cnt_last + KU - 1) / KU;
    auto ldidx = [&](int k) -> int {
        const int e = ebeg + k * stride + gl;
        return (k < nblk && e < eend) ? __ldg(colidx + e) : -1;
    };
    int my_cur = ldidx(0), my_next = ldidx(1);
    auto nbrs = [&](int t, int kc, int (&nbr)[KU]) {
        const int k = t / BPB, u0 = (t % BPB) * KU;
        const int src = (k == kc) ? my_cur : my_next;
#pragma unroll
        for (int u = 0; u < KU; ++u) nbr[u] = __shfl_sync(0xffffffffu, src, u0 + u, G);
    };
    if constexpr (!Op::kDoubleBuffer) {
        // single register set: gather batch t, then compute it (passes whose accumulators leave no room for two sets)
        for (int t = 0; t < T; ++t) {
            const int kc = t / BPB;
            int na[KU];
            nbrs(t, kc, na);
            typename Op::Src sa;
            Op::gather(p, sh, na, g, sa);
            // while the first batch of block kc is in flight: this lane's neighbour of block kc + 1 (my_next, loaded one
            // block ago) -> its rows into L2, so the gathers of that block find them there instead of in DRAM
            if (GNN_PF_MODE != 0 && (t % BPB) == 0 && kc + 1 < nblk && my_next >= 0) Op::prefetch(p, sh, my_next);
            Op::compute(st, own, p, sh, na, g, sa);
            if ((t % BPB) == BPB - 1) { my_cur = my_next; my_next = ldidx(kc + 2); }
        }
        return;
    } else {
    typename Op::Src sa, sb;
    int na[KU], nb[KU];
    nbrs(0, 0, na);
    Op::gather(p, sh, na, g, sa);
    for (int t = 0; t < T; t += 2) {
        const int kc = t / BPB;
        // batch t+1 -> set b (masked when past the end), then compute batch t from set a
        if (t + 1 < T) nbrs(t + 1, kc, nb);
        else {
#pragma unroll
            for (int u = 0; u < KU; ++u) nb[u] = -1;
        }
        Op::gather(p, sh, nb, g, sb);
        Op::compute(st, own, p, sh, na, g, sa);
        if ((t % BPB) == BPB - 1) { my_cur = my_next; my_next = ldidx(kc + 2); }
        if (t + 1 >= T) break;
        const int kc1 = (t + 1) / BPB;
        if (t + 2 < T) nbrs(t + 2, kc1, na);
        else {
#pragma unroll
            for (int u = 0; u < KU; ++u) na[u] = -1;
        }
        Op::gather(p, sh, na, g, sa);
        Op::compute(st, own, p, sh, nb, g, sb);
        if (((t + 1) % BPB) == BPB - 1) { my_cur = my_next; my_next = ldidx(kc1 + 2); }
    }
    }
}

// ------------------------------------------------------------------------------------------------
// group rows: one lane group per row, rows perm[first .. first+count), static round-robin over warps.
// The (row, rowptr) chain of the next tile is fetched while the current tile is processed.
// smem: NG * rowe floats for the da reduction (GATv2 dst pass only)
template <class Op>
__global__ void __launch_bounds__(kCtaThreads, Op::kMinBlocks)
group_kernel(typename Op::Params p, Shape sh, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ colidx,
             const int32_t* __restrict__ perm, int first, int count, float* da_part, int da_slot) {
    constexpr int G = Op::kG, CH = Op::kCH;
    constexpr int GPW = 32 / G;
    extern __shared__ float4 smem4[];
    float* smem = reinterpret_cast<float*>(smem4);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    typename Op::GeoT g;
    g.init(sh, lane);
    float da[CH];
#pragma unroll
    for (int c = 0; c < CH; ++c) da[c] = 0.f;

    const int ntiles = (count + GPW - 1) / GPW;
    const int total_warps = gridDim.x * kWarpsPerCta;
    const int sub = lane / G;
    auto ld_row = [&](int tile) -> int {
        const int idx = tile * GPW + sub;
        return (tile < ntiles && idx < count) ? __ldg(perm + first + idx) : -1;
    };
    int tile = blockIdx.x * kWarpsPerCta + warp;
    int row = ld_row(tile);
    int e0 = row >= 0 ? __ldg(rowptr + row) : 0;
    int e1 = row >= 0 ? __ldg(rowptr + row + 1) : 0;
    int row_n = ld_row(tile + total_warps);
    for (; tile < ntiles; tile += total_warps) {
        // next tile's row pointers and the row id of the tile after it: consumed at the bottom of the loop
        const int e0_n = row_n >= 0 ? __ldg(rowptr + row_n) : 0;
        const int e1_n = row_n >= 0 ? __ldg(rowptr + row_n + 1) : 0;
        const int row_nn = ld_row(tile + 2 * total_warps);
        const bool valid = row >= 0;
        const int len = e1 - e0;
        typename Op::Own own;
        Op::load_own(own, p, sh, valid ? row : 0, valid, g);
        typename Op::St st;
        st.reset();
        if constexpr (Op::MINARG) Op::init_state(st);
        int maxlen = len;
#pragma unroll
        for (int o = G; o < 32; o <<= 1) maxlen = max(maxlen, __shfl_xor_sync(0xffffffffu, maxlen, o));
        const int nblk = (maxlen + G - 1) / G;
        run_edges<Op>(st, own, p, sh, g, colidx, e0, e1, G, nblk, maxlen - (nblk - 1) * G);
        if (valid) Op::finalize(st, p, sh, row, g, da);
        row = row_n; e0 = e0_n; e1 = e1_n; row_n = row_nn;
    }
    if (Op::HAS_DA)
        cta_write_da<Op>(da, smem, da_part, da_slot + blockIdx.x, g, sh, warp * GPW + sub, kWarpsPerCta * GPW);
    // This grid may have been launched programmatically behind the pass's segment grid (run_op).  It reads nothing
    // from that grid, so the wait sits at its very end: the PTX ISA requires a dependent of a grid that executes
    // griddepcontrol.launch_dependents to execute griddepcontrol.wait, and with it "this grid has completed" implies
    // "the segment grid has completed and its writes (partials, stat2, Delta / G, da slots) are visible" - which is
    // what the ordinary launches that follow in the stream (hub merge, next pass, the caller's kernels) rely on.
    // A no-op when the launch carried no programmatic dependency.
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// ------------------------------------------------------------------------------------------------
// CTA rows + hub chunks: one CTA per segment; seg < n_chunks is hub chunk `seg` (partial state ->
// partials[seg]), otherwise the full row perm[n_hub + seg - n_chunks] (finalised in place).
// smem: NG * TEs + state_floats + NG * H floats for the merge.
template <class Op>
__global__ void __launch_bounds__(kCtaThreads, Op::kMinBlocks)
segment_kernel(typename Op::Params p, Shape sh, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ colidx,
               BinView bins, float* __restrict__ partials, float* da_part, int da_slot) {
    constexpr int G = Op::kG, CH = Op::kCH;
    constexpr int GPW = 32 / G, NG = kWarpsPerCta * GPW;
    // programmatic dependent launch: once every CTA of this grid is resident (or done), the group kernel of the same
    // pass - which touches disjoint rows and needs nothing from here - may start filling the SMs this grid's
    // last, partial wave leaves idle (run_op launches it with programmatic stream serialization; the group kernel
    // ends with griddepcontrol.wait, which restores full stream order for everything launched after it)
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    extern __shared__ float4 smem4[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float* smem = reinterpret_cast<float*>(smem4);
    const int gi = warp * GPW + lane / G;
    typename Op::GeoT g;
    g.init(sh, lane);
    const int TEp = Op::NA * sh.rowe + Op::NS * sh.H;  // floats per group partial (without max)
    const int TE = state_floats<Op>(sh);
    const int TEs = (TEp + 3) & ~3;     // group stride in smem, keeps float4 stores aligned
    float* s_part = smem;               // [NG][TEs]
    float* s_merged = smem + NG * TEs;  // [TE]
    float* s_max = s_merged + TE;       // [NG][H]
    float da[CH];
#pragma unroll
    for (int c = 0; c < CH; ++c) da[c] = 0.f;

    const int nseg = bins.n_chunks + bins.n_cta;
    for (int seg = blockIdx.x; seg < nseg; seg += gridDim.x) {
        int row, e0, e1;
        const bool partial = seg < bins.n_chunks;
        if (partial) {
            const int4 ch = __ldg(reinterpret_cast<const int4*>(bins.chunks) + seg);
            row = ch.x; e0 = ch.y; e1 = ch.z;
        } else {
            row = __ldg(bins.perm + bins.n_hub + (seg - bins.n_chunks));
            e0 = __ldg(rowptr + row);
            e1 = __ldg(rowptr + row + 1);
        }
        typename Op::Own own;
        Op::load_own(own, p, sh, row, true, g);
        typename Op::St st;
        st.reset();
        if constexpr (Op::MINARG) Op::init_state(st);
        // blocks of G edges are dealt round-robin to the NG groups; this warp's first group takes blocks
        // warp*GPW + k*NG, so its block count / last-block fill bound those of the warp's other groups
        const int nblk_all = (e1 - e0 + G - 1) / G;
        const int wfirst = warp * GPW;
        const int nblk = nblk_all > wfirst ? (nblk_all - wfirst + NG - 1) / NG : 0;
        const int last_first_edge = e0 + (wfirst + (nblk - 1) * NG) * G;
        const int cnt_last = min(G, e1 - last_first_edge);
        run_edges<Op>(st, own, p, sh, g, colidx, e0 + gi * G, e1, NG * G, nblk, cnt_last);
        // ---- cross-group merge: global max, rescale, fixed-order sum
        if (Op::SOFTMAX) {
            if (g.lead) s_max[gi * sh.H + g.hd] = st.m;
            __syncthreads();
            float mg = -INFINITY;
            if (g.act)
                for (int k = 0; k < NG; ++k) mg = fmaxf(mg, s_max[k * sh.H + g.hd]);
            const float f = (st.m == -INFINITY) ? 0.f : ex2(st.m - mg);
#pragma unroll
            for (int a = 0; a < Op::NA; ++a)
#pragma unroll
                for (int c = 0; c < CH; ++c) st.acc[a][c] *= f;
#pragma unroll
            for (int s = 0; s < Op::NS; ++s) st.sc[s] *= f;
            st.m = mg;
        }
        state_to_smem<Op>(st, s_part + gi * TEs, g, sh);
        __syncthreads();
        if constexpr (Op::MINARG) {
            for (int e = threadIdx.x; e < sh.rowe; e += kCtaThreads) {
                float bv = s_part[e];
                int bj = __float_as_int(s_part[sh.rowe + e]);
                for (int k = 1; k < NG; ++k) {
                    const float v = s_part[k * TEs + e];
                    const int j = __float_as_int(s_part[k * TEs + sh.rowe + e]);
                    if (minarg_better(v, j, bv, bj)) { bv = v; bj = j; }
                }
                s_merged[e] = bv;
                s_merged[sh.rowe + e] = __int_as_float(bj);
            }
        } else {
            for (int e = threadIdx.x; e < TEp; e += kCtaThreads) {
                float s = 0.f;
                for (int k = 0; k < NG; ++k) s += s_part[k * TEs + e];
                s_merged[e] = s;
            }
        }
        if (Op::SOFTMAX && gi == 0 && g.lead) s_merged[TEp + g.hd] = st.m;
        __syncthreads();
        if (partial) {
            for (int e = threadIdx.x; e < TE; e += kCtaThreads) partials[(size_t)seg * TE + e] = s_merged[e];
        } else if (gi == 0) {
            state_from_smem<Op>(st, s_merged, g, sh);
            Op::finalize(st, p, sh, row, g, da);
        }
        __syncthreads();
    }
    if (Op::HAS_DA) cta_write_da<Op>(da, smem, da_part, da_slot + blockIdx.x, g, sh, gi, NG);
}

// ------------------------------------------------------------------------------------------------
// hub rows: merge the chunk partials of hub slot blockIdx.x in a fixed order, finalise.
// The merge is latency-bound (one CTA walks up to nnz/split_chunk partial states), so the CTA is wide
// (kHubThreads) and every lane keeps kHubUnroll independent loads in flight.
// smem: state_floats + 4 + kHubWarps * (NA*rowe + NS*H) floats.
constexpr int kHubThreads = 512;
constexpr int kHubWarps = kHubThreads / 32;
constexpr int kHubUnroll = 8;

template <class Op>
__global__ void __launch_bounds__(kHubThreads)
hub_merge_kernel(typename Op::Params p, Shape sh, BinView bins, const float* __restrict__ partials, float* da_part,
                 int da_slot) {
    constexpr int G = Op::kG, CH = Op::kCH;
    extern __shared__ float4 smem4[];
    float* s_merged = reinterpret_cast<float*>(smem4);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    typename Op::GeoT g;
    g.init(sh, lane);
    const int TEp = Op::NA * sh.rowe + Op::NS * sh.H;
    const int TE = state_floats<Op>(sh);
    const int slot = blockIdx.x;
    const int c0 = __ldg(bins.chunk_ptr + slot), c1 = __ldg(bins.chunk_ptr + slot + 1);
    const int row = __ldg(bins.chunks + 4 * c0);
    // fixed reduction order: chunk c goes to warp (c - c0) % W, every warp walks its chunks in ascending order
    // into kHubUnroll round-robin partial sums per element (added as a fixed tree), then the W warp sums are
    // added in warp order.  s_part: [W][TEp] after s_merged[TE].
    float* s_part = s_merged + ((TE + 3) & ~3);
    if (Op::SOFTMAX) {
        for (int h = warp; h < sh.H; h += kHubWarps) {
            float mg = -INFINITY;
            for (int c = c0 + lane; c < c1; c += 32) mg = fmaxf(mg, partials[(size_t)c * TE + TEp + h]);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) mg = fmaxf(mg, __shfl_xor_sync(0xffffffffu, mg, o));
            if (lane == 0) s_merged[TEp + h] = mg;
        }
        __syncthreads();
    }
    if constexpr (Op::MINARG) {
        // same chunk-to-warp assignment; every lane keeps four independent (value, index) candidates in flight
        for (int e = lane; e < sh.rowe; e += 32) {
            float bv[4];
            int bj[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) { bv[u] = INFINITY; bj[u] = -1; }
            for (int c = c0 + warp; c < c1; c += 4 * kHubWarps) {
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int cu = c + u * kHubWarps;
                    if (cu < c1) {
                        const float v = partials[(size_t)cu * TE + e];
                        const int j = __float_as_int(partials[(size_t)cu * TE + sh.rowe + e]);
                        if (minarg_better(v, j, bv[u], bj[u])) { bv[u] = v; bj[u] = j; }
                    }
                }
            }
#pragma unroll
            for (int u = 1; u < 4; ++u)
                if (minarg_better(bv[u], bj[u], bv[0], bj[0])) { bv[0] = bv[u]; bj[0] = bj[u]; }
            s_part[warp * TEp + e] = bv[0];
            s_part[warp * TEp + sh.rowe + e] = __int_as_float(bj[0]);
        }
        __syncthreads();
        for (int e = threadIdx.x; e < sh.rowe; e += kHubThreads) {
            float bv = s_part[e];
            int bj = __float_as_int(s_part[sh.rowe + e]);
            for (int w = 1; w < kHubWarps; ++w) {
                const float v = s_part[w * TEp + e];
                const int j = __float_as_int(s_part[w * TEp + sh.rowe + e]);
                if (minarg_better(v, j, bv, bj)) { bv = v; bj = j; }
            }
            s_merged[e] = bv;
            s_merged[sh.rowe + e] = __int_as_float(bj);
        }
    } else {
    for (int e = lane; e < TEp; e += 32) {
        const int h = e < Op::NA * sh.rowe ? (e % sh.rowe) / sh.d : (e - Op::NA * sh.rowe) % sh.H;
        const float mg = Op::SOFTMAX ? s_merged[TEp + h] : 0.f;
        float su[kHubUnroll];
#pragma unroll
        for (int u = 0; u < kHubUnroll; ++u) su[u] = 0.f;
        int c = c0 + warp;
        for (; c + (kHubUnroll - 1) * kHubWarps < c1; c += kHubUnroll * kHubWarps) {
            float v[kHubUnroll], mc[kHubUnroll];
#pragma unroll
            for (int u = 0; u < kHubUnroll; ++u) {
                const size_t cc = (size_t)(c + u * kHubWarps) * TE;
                v[u] = partials[cc + e];
                mc[u] = Op::SOFTMAX ? partials[cc + TEp + h] : 0.f;
            }
#pragma unroll
            for (int u = 0; u < kHubUnroll; ++u) {
                const float f = !Op::SOFTMAX ? 1.f : (mc[u] == -INFINITY) ? 0.f : ex2(mc[u] - mg);
                su[u] = fmaf(v[u], f, su[u]);
            }
        }
#pragma unroll
        for (int u = 0; u < kHubUnroll; ++u) {
            const int cu = c + u * kHubWarps;
            if (cu < c1) {
                const size_t cc = (size_t)cu * TE;
                float f = 1.f;
                if (Op::SOFTMAX) {
                    const float mc = partials[cc + TEp + h];
                    f = (mc == -INFINITY) ? 0.f : ex2(mc - mg);
                }
                su[u] = fmaf(partials[cc + e], f, su[u]);
            }
        }
        s_part[warp * TEp + e] = ((su[0] + su[1]) + (su[2] + su[3])) + ((su[4] + su[5]) + (su[6] + su[7]));
    }
    __syncthreads();
    for (int e = threadIdx.x; e < TEp; e += kHubThreads) {
        float s = 0.f;
#pragma unroll
        for (int w = 0; w < kHubWarps; ++w) s += s_part[w * TEp + e];
        s_merged[e] = s;
    }
    }
    __syncthreads();
    float da[CH];
#pragma unroll
    for (int c = 0; c < CH; ++c) da[c] = 0.f;
    if (warp == 0 && lane < G) {
        typename Op::St st;
        state_from_smem<Op>(st, s_merged, g, sh);
        Op::finalize(st, p, sh, row, g, da);
        if (Op::HAS_DA && g.act) {
#pragma unroll
            for (int c = 0; c < CH; ++c) da_part[(size_t)(da_slot + slot) * sh.rowe + g.eoff + c] = da[c];
        }
    }
}

// ------------------------------------------------------------------------------------------------
struct GridPlan {
    int seg_grid, grp_grid, hub_grid;
    int da_slots() const { return seg_grid + grp_grid + hub_grid; }
};

inline GridPlan grid_plan(const BinView& b, int sm_count, int G) {
    const int GPW = 32 / G;
    GridPlan gp;
    const int nseg = b.n_chunks + b.n_cta;
    gp.seg_grid = nseg < sm_count * 16 ? nseg : sm_count * 16;
    const int ntiles = (b.n_group + GPW - 1) / GPW;
    const int nblk = (ntiles + kWarpsPerCta - 1) / kWarpsPerCta;
    gp.grp_grid = nblk < sm_count * 32 ? nblk : sm_count * 32;
    gp.hub_grid = b.n_hub;
    return gp;
}

template <class Op> inline size_t seg_smem_bytes(const Shape& sh) {
    constexpr int NG = kWarpsPerCta * (32 / Op::kG);
    const int TEp = Op::NA * sh.rowe + Op::NS * sh.H;
    size_t f = (size_t)NG * ((TEp + 3) & ~3) + state_floats<Op>(sh) + (size_t)NG * sh.H;
    size_t da = Op::HAS_DA ? (size_t)NG * sh.rowe : 0;
    return 4 * (f > da ? f : da) + 16;
}
template <class Op> inline size_t grp_smem_bytes(const Shape& sh) {
    constexpr int NG = kWarpsPerCta * (32 / Op::kG);
    return (Op::HAS_DA ? 4 * (size_t)NG * sh.rowe : 0) + 16;
}

template <class Op> inline cudaError_t run_op(const typename Op::Params& p, const Shape& sh, const LaunchCtx& c) {
    const BinView& b = c.bins;
    const GridPlan gp = grid_plan(b, c.sm_count, Op::kG);
    constexpr int NG = kWarpsPerCta * (32 / Op::kG);
    int slot = c.da_slot_base;
    if (gp.seg_grid > 0) {
        const size_t smem = seg_smem_bytes<Op>(sh);
        if (smem > 48 * 1024) {
            cudaError_t e = cudaFuncSetAttribute(segment_kernel<Op>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
        }
        prof_begin(Op::kName, "segment", c.stream);
        segment_kernel<Op><<<gp.seg_grid, kCtaThreads, smem, c.stream>>>(p, sh, c.rowptr, c.colidx, b, c.partials,
                                                                         c.da_part, slot);
        prof_end(c.stream);
        count_launch();
    }
    slot += gp.seg_grid;
    if (gp.grp_grid > 0) {
        const size_t smem = grp_smem_bytes<Op>(sh);
        if (smem > 48 * 1024) {
            cudaError_t e = cudaFuncSetAttribute(group_kernel<Op>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
        }
        prof_begin(Op::kName, "group", c.stream);
        // overlaps the tail of this pass's segment kernel (see there); never the previous pass, whose results it may
        // read, and not while the per-kernel event profiler brackets every launch
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(gp.grp_grid); cfg.blockDim = dim3(kCtaThreads); cfg.dynamicSmemBytes = smem; cfg.stream = c.stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at;
        cfg.numAttrs = (GNN_PDL && pdl_enabled() && gp.seg_grid > 0 && !prof_enabled()) ? 1 : 0;
        cudaError_t le = cudaLaunchKernelEx(&cfg, group_kernel<Op>, p, sh, c.rowptr, c.colidx, b.perm, b.n_hub + b.n_cta,
                                            b.n_group, c.da_part, slot);
        if (le != cudaSuccess) return le;
        prof_end(c.stream);
        count_launch();
    }
    slot += gp.grp_grid;
    if (gp.hub_grid > 0) {
        const size_t smem = 4 * ((size_t)state_floats<Op>(sh) + 4 + (size_t)kHubWarps * (Op::NA * sh.rowe + Op::NS * sh.H)) + 16;
        if (smem > 48 * 1024) {
            cudaError_t e = cudaFuncSetAttribute(hub_merge_kernel<Op>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
        }
        prof_begin(Op::kName, "hub_merge", c.stream);
        hub_merge_kernel<Op><<<gp.hub_grid, kHubThreads, smem, c.stream>>>(p, sh, b, c.partials, c.da_part, slot);
        prof_end(c.stream);
        count_launch();
    }
    return cudaGetLastError();
}

}  // namespace gnn
