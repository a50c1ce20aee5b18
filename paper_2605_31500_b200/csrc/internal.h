// internal.h - host-side declarations shared by api.cu, plan.cu and the per-pass dispatch units.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/gnn_attn.h"
#include "engine.cuh"

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
};

namespace gnn {

enum Pass { kGtFwd = 0, kGtBwdDst, kGtBwdSrc, kGatFwd, kGatBwdDst, kGatBwdSrc, kNumPass };
struct PassInfo { int na, ns, softmax, has_da; };
// must match the NA / NS / SOFTMAX / HAS_DA constants of the Op structs (static_asserted in the dispatch units)
constexpr PassInfo kPassInfo[kNumPass] = {{1, 1, 1, 0}, {2, 1, 0, 0}, {2, 0, 0, 0}, {1, 1, 1, 0}, {4, 1, 0, 1}, {1, 0, 0, 0}};

inline int pass_state_floats(Pass p, const Shape& sh) {
    return kPassInfo[p].na * sh.rowe + (kPassInfo[p].ns + kPassInfo[p].softmax) * sh.H;
}
// lane-group width for a feature row of `rowv` 16-byte vectors; 0 = unsupported
inline int group_width(int rowv) { return rowv <= 8 ? 8 : rowv <= 16 ? 16 : rowv <= 64 ? 32 : 0; }

void set_error(const char* fmt, ...);

struct GtArgs {
    const void *q, *k, *v, *dout;
    void* out;
    float *lse, *delta, *dq, *dk, *dv;
};
struct GatArgs {
    const void *xl, *xr, *dout;
    const float* a;
    void* out;
    float *lse, *g, *dxl, *dxr;
    float slope;
};
cudaError_t launch_gt_fwd(int dtype, const Shape&, const LaunchCtx&, const GtArgs&);
cudaError_t launch_gt_bwd_dst(int dtype, const Shape&, const LaunchCtx&, const GtArgs&);
cudaError_t launch_gt_bwd_src(int dtype, const Shape&, const LaunchCtx&, const GtArgs&);
cudaError_t launch_gat_fwd(int dtype, const Shape&, const LaunchCtx&, const GatArgs&);
cudaError_t launch_gat_bwd_dst(int dtype, const Shape&, const LaunchCtx&, const GatArgs&);
cudaError_t launch_gat_bwd_src(int dtype, const Shape&, const LaunchCtx&, const GatArgs&);
// da[e] = sum over slots of da_part[slot][e], fixed order, fp64 accumulation (no atomics)
cudaError_t launch_da_reduce(const float* da_part, int slots, int rowe, float* da, cudaStream_t);

}  // namespace gnn
