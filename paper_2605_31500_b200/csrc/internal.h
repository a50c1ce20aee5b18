// internal.h - host-side declarations shared by api.cu, plan.cu and the per-pass dispatch units.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>

#include "../../include/gnn_attn.h"
#include "engine.cuh"

namespace gnn {
// general WSB layout (row f2): per 16-row window the sorted unique source columns in width-8 TCBs
struct WsbView {
    const int32_t* row_offset;   // [n_windows + 1] first TCB of every row window
    const int32_t* cols;         // [n_tcb][8] global column ids, zero padded
    const uint8_t* bitmap;       // [n_tcb][16] byte r = row r of the window, bit c = column c of the TCB
    int32_t n_tcb;
    int32_t n_dup;               // CSR entries beyond the first of their (dst, src) pair (the bitmap cannot hold them)
};
}  // namespace gnn

struct gnn_plan {
    int32_t n;
    int64_t nnz;
    gnn_plan_opts_t opts;
    int sm_count;
    const int32_t* rowptr;   // caller's CSR (device)
    const int32_t* colidx;
    gnn::BinView fwd;        // bins of the CSR (in-degrees)
    int32_t* rowptr_t;       // CSR^T (device, inside dev_mem) or nullptr
    int32_t* colidx_t;
    gnn::BinView tr;         // bins of CSR^T (out-degrees)
    // block layout (a11)
    uint16_t* blk_bitmap;    // [n_windows][16]
    int32_t* blk_rem_rowptr; // [n+1]
    int32_t* blk_rem_colidx; // [rem_nnz]
    int32_t n_windows;
    int64_t rem_nnz;
    int32_t* rem_rowptr_t;   // stable transpose of the remainder CSR + its bins (build_blocks DIAG with build_transpose)
    int32_t* rem_colidx_t;
    gnn::BinView rem_tr;
    int32_t rows_sorted;     // 1 if every CSR row lists its sources in ascending order (min / max fast path)
    int32_t has_wsb;         // build_blocks & GNN_BLOCKS_WSB
    gnn::WsbView wsb;        // of the CSR (destination windows x source columns)
    gnn::WsbView wsb_t;      // of CSR^T (source windows x destination columns); == wsb in the undirected mode
};

namespace gnn {

enum Pass { kGtFwd = 0, kGtBwdDst, kGtBwdSrc, kGatFwd, kGatBwdDst, kGatBwdSrc, kMinFwd, kNumPass };
struct PassInfo { int na, ns, softmax, has_da; };
// must match the NA / NS / SOFTMAX / HAS_DA constants of the Op structs (static_asserted in the dispatch units)
constexpr PassInfo kPassInfo[kNumPass] = {{1, 1, 1, 0}, {2, 1, 0, 0}, {2, 0, 0, 0}, {1, 1, 1, 0}, {2, 2, 0, 1}, {2, 1, 0, 1}, {2, 0, 0, 0}};

inline int pass_state_floats(Pass p, const Shape& sh) {
    return kPassInfo[p].na * sh.rowe + (kPassInfo[p].ns + kPassInfo[p].softmax) * sh.H;
}
// Lane layout of a pass: each lane owns `cb` contiguous bytes of one head (nv loads of vb bytes), a row
// takes `lanes` lanes inside a group of g lanes (power of two, 4..32).  32 bytes per lane (one 256-bit load per
// gathered row) measured best on B200 for every pass (profiles/r01_lane_width_sweep.md); 16 when head_dim*sizeof
// is 16.  GNN_MAX_CB_FWD / GNN_MAX_CB_BWD (16|32) override the width for tuning runs.
struct LaneCfg { int vb, nv, cb, g, lanes; };
constexpr int pass_max_cb(Pass) { return 32; }
// widest lane the pass is instantiated for (wide rows may exceed the preferred pass_max_cb)
constexpr int pass_inst_max_cb(Pass) { return 32; }
// edges gathered per lane group per batch, all in flight before the batch is computed (capped at the group
// width); 4 measured best on cfg 3 / 5 for every pass but the 4-accumulator GATv2 dst pass (profiles/r01_lane_width_sweep.md)
#ifndef GNN_FWD_KU
#define GNN_FWD_KU 4
#endif
#ifndef GNN_GAT_DST_KU
#define GNN_GAT_DST_KU 4
#endif
#ifndef GNN_GAT_SRC_KU
#define GNN_GAT_SRC_KU 2
#endif
#ifndef GNN_BWD_KU
#define GNN_BWD_KU 4
#endif
constexpr int pass_ku(Pass p, int cb) {
    return (p == kGatFwd || p == kGtFwd || p == kMinFwd) ? (cb == 32 ? GNN_FWD_KU : 4)
         : (p == kGatBwdDst)             ? (cb == 32 ? GNN_GAT_DST_KU : 4)   // four accumulator vectors
         : (p == kGatBwdSrc)             ? (cb == 32 ? GNN_GAT_SRC_KU : 4)
                                         : (cb == 32 ? GNN_BWD_KU : 4);
}
inline bool pick_lane_cfg(Pass p, int esz, int heads, int head_dim, LaneCfg& lc) {
    const int head_bytes = head_dim * esz, row_bytes = heads * head_bytes;
    int cb = pass_max_cb(p);
    if (const char* e = getenv((p == kGtFwd || p == kGatFwd || p == kMinFwd) ? "GNN_MAX_CB_FWD" : "GNN_MAX_CB_BWD")) {  // tuning knob
        const int v = atoi(e);
        if ((v == 16 || v == 32 || v == 64) && v <= pass_inst_max_cb(p)) cb = v;
    }
    while (cb > head_bytes) cb >>= 1;
    while (row_bytes / cb > 32 && cb * 2 <= head_bytes && cb * 2 <= pass_inst_max_cb(p)) cb <<= 1;  // wide rows
    if (cb < 16 || row_bytes / cb > 32) return false;
    lc.cb = cb;
    lc.vb = cb >= 32 ? 32 : 16;
    lc.nv = cb / lc.vb;
    lc.lanes = row_bytes / cb;
    lc.g = 4;
    while (lc.g < lc.lanes) lc.g <<= 1;
    return true;
}
// fill the lane-dependent fields of a Shape for one pass
inline Shape pass_shape(Shape sh, Pass p, int esz, LaneCfg& lc) {
    pick_lane_cfg(p, esz, sh.H, sh.d, lc);
    sh.ch = lc.cb / esz;
    sh.lanes = lc.lanes;
    sh.lpl = sh.d / sh.ch;
    sh.lpl_log2 = 0;
    while ((1 << sh.lpl_log2) < sh.lpl) ++sh.lpl_log2;
    return sh;
}

void set_error(const char* fmt, ...);

struct GtArgs {
    const void *q, *k, *v, *dout;
    void* out;
    float *lse, *delta, *dq, *dk, *dv;
    float2* stat2;   // workspace [n,H]: (L * log2(e), Delta) packed by the dst pass for the src pass (one 8-byte gather)
    int accumulate;  // src pass: add to the dk / dv already stored (block backward: tile-local part first, remainder second)
};
struct GatArgs {
    const void *xl, *xr, *dout;
    const float* a;
    void* out;
    float *lse, *g, *dxl, *dxr;
    float slope;
};
struct AggArgs {
    const void *x, *dout;
    void* out;
    int32_t* arg;
    float* dx;
    float sign;   // +1: min, -1: max
};
// `Shape` passed to the launchers carries n, H, d, rowe; the lane fields are filled per pass inside.
cudaError_t launch_gt_fwd(int dtype, const Shape&, const LaunchCtx&, const GtArgs&);
cudaError_t launch_gt_bwd_dst(int dtype, const Shape&, const LaunchCtx&, const GtArgs&);
cudaError_t launch_gt_bwd_src(int dtype, const Shape&, const LaunchCtx&, const GtArgs&);
// tile-local tensor-core part of the block backward (block_bwd.cu): Delta, dQ complete; dK, dV in-window terms; stat2
cudaError_t launch_gt_bwd_block(const gnn_plan* P, const GtArgs&, int heads, cudaStream_t);
cudaError_t launch_gat_fwd(int dtype, const Shape&, const LaunchCtx&, const GatArgs&);
cudaError_t launch_gat_bwd_dst(int dtype, const Shape&, const LaunchCtx&, const GatArgs&);
cudaError_t launch_gat_bwd_src(int dtype, const Shape&, const LaunchCtx&, const GatArgs&);
cudaError_t launch_min_fwd(int dtype, const Shape&, const LaunchCtx&, const AggArgs&, bool rows_sorted);
// dx[arg[i,c], c] += dout[i,c] over all (i, c) with arg >= 0 (dx zeroed by the caller); one red.global.add per element
cudaError_t launch_minmax_scatter(int dtype, long long n, int rowe, const AggArgs&, int sm_count, cudaStream_t);
// da[e] = sum over slots of da_part[slot][e], fixed order, fp64 accumulation (no atomics)
cudaError_t launch_da_reduce(const float* da_part, int slots, int rowe, float* da, cudaStream_t);

}  // namespace gnn
