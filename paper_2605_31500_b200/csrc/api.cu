// api.cu - the C-ABI entry points of include/gnn_attn.h: argument validation and pass sequencing.
// Every step of the path runs in this library's kernels; nothing here computes on the host.
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <vector>

#include "internal.h"
#include "kernels.cuh"

namespace gnn {

static std::atomic<unsigned long long> g_launches{0};
static std::atomic<int> g_pdl_on{1};
void count_launch(int k) { g_launches.fetch_add((unsigned long long)k, std::memory_order_relaxed); }
bool pdl_enabled() { return g_pdl_on.load(std::memory_order_relaxed) != 0; }
static thread_local char t_err[512] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof(t_err), fmt, ap);
    va_end(ap);
}

// ---- per-launch event profiler (measurement aid for bench.py; off by default)
struct ProfRec { char name[48]; cudaEvent_t a, b; };
static bool g_prof_on = false;
static std::vector<ProfRec> g_prof;
void prof_begin(const char* pass, const char* kernel, cudaStream_t st) {
    if (!g_prof_on) return;
    ProfRec r;
    snprintf(r.name, sizeof(r.name), "%s/%s", pass, kernel);
    cudaEventCreate(&r.a);
    cudaEventCreate(&r.b);
    cudaEventRecord(r.a, st);
    g_prof.push_back(r);
}
bool prof_enabled() { return g_prof_on; }
void prof_end(cudaStream_t st) {
    if (!g_prof_on || g_prof.empty()) return;
    cudaEventRecord(g_prof.back().b, st);
}

namespace {

bool make_shape(int32_t n, int32_t heads, int32_t head_dim, int dtype, Shape& sh, const char* who) {
    if (dtype != GNN_F32 && dtype != GNN_BF16) { set_error("%s: unknown dtype %d", who, dtype); return false; }
    const int esz = dtype == GNN_F32 ? 4 : 2;
    LaneCfg lf, lb;
    if (heads < 1 || head_dim < 1 || (head_dim & (head_dim - 1)) || head_dim * esz < 16 ||
        (long long)heads * head_dim * esz > 1024 || !pick_lane_cfg(kGtFwd, esz, heads, head_dim, lf) ||
        !pick_lane_cfg(kGtBwdDst, esz, heads, head_dim, lb) || !pick_lane_cfg(kGatBwdDst, esz, heads, head_dim, lb)) {
        set_error("%s: unsupported shape heads=%d head_dim=%d dtype=%d (head_dim must be a power of two with "
                  "head_dim*sizeof >= 16, heads*head_dim*sizeof <= 1024, and at most 32 lanes of "
                  "min(head_dim*sizeof, 32) bytes per row)", who, heads, head_dim, dtype);
        return false;
    }
    sh.n = n; sh.H = heads; sh.d = head_dim; sh.rowe = heads * head_dim;
    sh.ld = sh.rowe; sh.ldh = heads;
    sh.ch = sh.lanes = sh.lpl = sh.lpl_log2 = 0;  // filled per pass (pass_shape)
    return true;
}

// One launch covers rows of at most 1024 bytes (32 lanes x 32 bytes).  Wider rows (e.g. the paper's fp32 H=4, D=128
// grid points) are processed as consecutive HEAD GROUPS: group g runs the same passes on heads
// [h0, h0 + H_g) through pointers offset by h0 and the full-row strides ld = heads*head_dim, ldh = heads.  Heads
// are independent in every pass (softmax, gradients and da are per head), so the result is that of one launch.
struct HeadGroup { Shape sh; int h0; };
constexpr int kMaxHeadGroups = 64;
int head_groups(int32_t n, int32_t heads, int32_t head_dim, int dtype, HeadGroup* out, const char* who) {
    Shape sh;
    if (dtype != GNN_F32 && dtype != GNN_BF16) { set_error("%s: unknown dtype %d", who, dtype); return 0; }
    const int esz = dtype == GNN_F32 ? 4 : 2;
    const long long hb = (long long)head_dim * esz;
    int hg = 0;
    if (heads >= 1 && head_dim >= 1 && !(head_dim & (head_dim - 1)) && hb >= 16 && hb <= 1024) {
        // widest group one launch supports; a group that is not the whole row must keep the 32-byte alignment of
        // the 256-bit gathers at its byte offset h0 * head_dim * sizeof
        hg = (int)(1024 / hb) < heads ? (int)(1024 / hb) : heads;
        while (hg >= 1 && !((hg == heads || (hg * hb) % 32 == 0) && make_shape(n, hg, head_dim, dtype, sh, who))) --hg;
    }
    if (hg < 1 || (heads + hg - 1) / hg > kMaxHeadGroups) {
        set_error("%s: unsupported shape heads=%d head_dim=%d dtype=%d (head_dim must be a power of two with "
                  "16 <= head_dim*sizeof <= 1024; at most %d head groups)", who, heads, head_dim, dtype, kMaxHeadGroups);
        return 0;
    }
    int ng = 0;
    for (int h0 = 0; h0 < heads; h0 += hg, ++ng) {
        const int h = heads - h0 < hg ? heads - h0 : hg;
        if (!make_shape(n, h, head_dim, dtype, sh, who)) return 0;
        sh.ld = heads * head_dim;
        sh.ldh = heads;
        out[ng] = {sh, h0};
    }
    return ng;
}
// workspace of a call = max over its head groups
template <class T> T* off_bytes(T* p, size_t bytes) { return (T*)((char*)p + bytes); }
template <class T> const T* off_bytes(const T* p, size_t bytes) { return (const T*)((const char*)p + bytes); }

bool aligned32(const void* p) { return (((uintptr_t)p) & 31) == 0; }  // 256-bit gathers need 32-byte alignment

struct WsLayout { size_t partials, da_part, stat2, total; int da_slots, da_slots_dst; };

// workspace of one API call = max over its passes of the chunk partials (+ da partials for GATv2 bwd)
WsLayout ws_layout(const gnn_plan* P, int op, const Shape& sh, int esz) {
    WsLayout w = {0, 0, 0, 0, 0, 0};
    size_t part = 0;
    auto need = [&](Pass ps, const BinView& b) {
        const size_t x = (size_t)b.n_chunks * pass_state_floats(ps, sh) * sizeof(float);
        if (x > part) part = x;
    };
    switch (op) {
        case GNN_OP_GT_FWD: need(kGtFwd, P->fwd); break;
        case GNN_OP_GT_BWD: need(kGtBwdDst, P->fwd); need(kGtBwdSrc, P->tr); break;
        case GNN_OP_GATV2_FWD: need(kGatFwd, P->fwd); break;
        case GNN_OP_GATV2_BWD: need(kGatBwdDst, P->fwd); need(kGatBwdSrc, P->tr); break;
        case GNN_OP_SEG_MINMAX_FWD: need(kMinFwd, P->fwd); break;
        default: break;
    }
    w.partials = 0;
    w.da_part = (part + 255) / 256 * 256;
    size_t da = 0;
    if (op == GNN_OP_GATV2_BWD) {
        LaneCfg lc;
        pick_lane_cfg(kGatBwdDst, esz, sh.H, sh.d, lc);
        w.da_slots_dst = grid_plan(P->fwd, P->sm_count, lc.g).da_slots();                       // dst pass (CSR bins)
        pick_lane_cfg(kGatBwdSrc, esz, sh.H, sh.d, lc);
        w.da_slots = w.da_slots_dst + grid_plan(P->tr, P->sm_count, lc.g).da_slots();          // + src pass (CSR^T bins)
        da = (size_t)w.da_slots * sh.rowe * sizeof(float);
    }
    w.stat2 = (w.da_part + da + 255) / 256 * 256;
    const size_t st2 = (op == GNN_OP_GT_BWD) ? (size_t)P->n * sh.ldh * sizeof(float2) : 0;   // (L log2e, Delta) for the GT src pass
    w.total = w.stat2 + st2 + 256;
    return w;
}

size_t ws_total(const gnn_plan* P, int op, const HeadGroup* hg, int ng, int esz) {
    size_t t = 0;
    for (int g = 0; g < ng; ++g) {
        const size_t x = ws_layout(P, op, hg[g].sh, esz).total;
        if (x > t) t = x;
    }
    return t;
}

// workspace of gnn_gt_attn_bwd_block: hub-chunk partials of the remainder src pass, then (L log2e, Delta) per (node, head)
struct BlockWs { size_t stat2, total; };
BlockWs block_bwd_ws(const gnn_plan* P, const HeadGroup* hg, int ng, int heads) {
    size_t part = 0;
    for (int g = 0; g < ng; ++g) {
        const size_t x = (size_t)P->rem_tr.n_chunks * pass_state_floats(kGtBwdSrc, hg[g].sh) * sizeof(float);
        if (x > part) part = x;
    }
    BlockWs w;
    w.stat2 = (part + 255) / 256 * 256;
    w.total = w.stat2 + (size_t)P->n * heads * sizeof(float2) + 256;
    return w;
}

bool check_common(const gnn_plan* P, const int32_t* rowptr, const int32_t* colidx, int32_t n, const char* who) {
    if (!P) { set_error("%s: NULL plan", who); return false; }
    if (rowptr != P->rowptr || colidx != P->colidx || n != P->n) {
        set_error("%s: rowptr/colidx/n differ from the arrays the plan was built from", who);
        return false;
    }
    return true;
}

LaunchCtx make_ctx(const gnn_plan* P, bool transposed, void* ws, const WsLayout& w, gnn_stream_t stream) {
    LaunchCtx c;
    c.stream = (cudaStream_t)stream;
    c.sm_count = P->sm_count;
    c.rowptr = transposed ? P->rowptr_t : P->rowptr;
    c.colidx = transposed ? P->colidx_t : P->colidx;
    c.bins = transposed ? P->tr : P->fwd;
    c.partials = (float*)((char*)ws + w.partials);
    c.da_part = (float*)((char*)ws + w.da_part);
    c.da_slot_base = 0;
    return c;
}

gnn_status_t cuda_status(cudaError_t e, const char* who) {
    if (e == cudaSuccess) return GNN_OK;
    set_error("%s: CUDA error: %s", who, cudaGetErrorString(e));
    return GNN_ECUDA;
}

}  // namespace
}  // namespace gnn

using namespace gnn;

extern "C" const char* gnn_last_error(void) { return t_err; }
extern "C" const char* gnn_version(void) { return "gnn_attn 0.1 sm_100a"; }
extern "C" int64_t gnn_launch_count(void) { return (int64_t)g_launches.load(std::memory_order_relaxed); }
extern "C" void gnn_pdl_enable(int on) { g_pdl_on.store(on != 0, std::memory_order_relaxed); }

extern "C" void gnn_profile_enable(int on) { g_prof_on = on != 0; }
extern "C" int32_t gnn_profile_collect(char* names, float* ms, int32_t max_records) {
    int32_t k = 0;
    for (auto& r : g_prof) {
        cudaEventSynchronize(r.b);
        float t = 0.f;
        cudaEventElapsedTime(&t, r.a, r.b);
        if (k < max_records && names && ms) {
            strncpy(names + (size_t)k * 48, r.name, 48);
            ms[k] = t;
            ++k;
        }
        cudaEventDestroy(r.a);
        cudaEventDestroy(r.b);
    }
    g_prof.clear();
    return k;
}

static bool agg_shape(int32_t n, int32_t channels, int dtype, Shape& sh, const char* who);

extern "C" gnn_status_t gnn_workspace_bytes(const gnn_plan_t* P, int op, int32_t heads, int32_t head_dim,
                                            gnn_dtype_t dtype, size_t* bytes) {
    if (!P || !bytes) { set_error("gnn_workspace_bytes: NULL plan or bytes"); return GNN_EINVAL; }
    if (op == GNN_OP_GT_FWD_BLOCK || op == GNN_OP_WSB_FWD || op == GNN_OP_WSB_BWD) { *bytes = 0; return GNN_OK; }   // tile-local: no workspace
    if (op == GNN_OP_GT_BWD_BLOCK) {
        if (!P->rem_rowptr_t) { set_error("gnn_workspace_bytes: plan lacks GNN_BLOCKS_DIAG with build_transpose"); return GNN_EINVAL; }
        HeadGroup hgb[kMaxHeadGroups];
        const int ngb = head_groups(P->n, heads, head_dim, dtype, hgb, "gnn_workspace_bytes");
        if (!ngb) return GNN_EUNSUPPORTED;
        *bytes = block_bwd_ws(P, hgb, ngb, heads).total;
        return GNN_OK;
    }
    if ((op < GNN_OP_GT_FWD || op > GNN_OP_GATV2_BWD) && op != GNN_OP_SEG_MINMAX_FWD) {
        set_error("gnn_workspace_bytes: unknown op %d", op);
        return GNN_EINVAL;
    }
    HeadGroup hg[kMaxHeadGroups];
    int ng = 1;
    if (op == GNN_OP_SEG_MINMAX_FWD) {
        if (heads < 1 || head_dim < 1 || !agg_shape(P->n, heads * head_dim, dtype, hg[0].sh, "gnn_workspace_bytes")) return GNN_EUNSUPPORTED;
    } else if (!(ng = head_groups(P->n, heads, head_dim, dtype, hg, "gnn_workspace_bytes"))) return GNN_EUNSUPPORTED;
    if ((op == GNN_OP_GT_BWD || op == GNN_OP_GATV2_BWD) && !P->opts.build_transpose) {
        set_error("gnn_workspace_bytes: backward needs a plan built with build_transpose");
        return GNN_EINVAL;
    }
    *bytes = ws_total(P, op, hg, ng, dtype == GNN_F32 ? 4 : 2);
    return GNN_OK;
}

extern "C" gnn_status_t gnn_gt_attn_fwd(const gnn_plan_t* P, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                        const void* q, const void* k, const void* v, int32_t heads, int32_t head_dim,
                                        gnn_dtype_t dtype, void* out, float* lse, void* ws, size_t ws_bytes,
                                        gnn_stream_t stream) {
    const char* who = "gnn_gt_attn_fwd";
    if (!check_common(P, rowptr, colidx, n, who)) return GNN_EINVAL;
    if (!q || !k || !v || !out || !lse || !ws) { set_error("%s: NULL pointer argument", who); return GNN_EINVAL; }
    if (!aligned32(q) || !aligned32(k) || !aligned32(v) || !aligned32(out) || !aligned32(ws)) {
        set_error("%s: feature pointers and workspace must be 32-byte aligned", who);
        return GNN_EINVAL;
    }
    HeadGroup hg[kMaxHeadGroups];
    const int ng = head_groups(n, heads, head_dim, dtype, hg, who), esz = dtype == GNN_F32 ? 4 : 2;
    if (!ng) return GNN_EUNSUPPORTED;
    const size_t need = ws_total(P, GNN_OP_GT_FWD, hg, ng, esz);
    if (ws_bytes < need) { set_error("%s: workspace too small (%zu < %zu)", who, ws_bytes, need); return GNN_EWORKSPACE; }
    cudaError_t e = cudaSuccess;
    for (int g = 0; g < ng && e == cudaSuccess; ++g) {
        const Shape& sh = hg[g].sh;
        const size_t fo = (size_t)hg[g].h0 * head_dim * esz;   // byte offset of the group's first head in a feature row
        const WsLayout w = ws_layout(P, GNN_OP_GT_FWD, sh, esz);
        GtArgs a = {};
        a.q = off_bytes(q, fo); a.k = off_bytes(k, fo); a.v = off_bytes(v, fo); a.out = off_bytes(out, fo); a.lse = lse + hg[g].h0;
        e = launch_gt_fwd(dtype, sh, make_ctx(P, false, ws, w, stream), a);
    }
    return cuda_status(e, who);
}

extern "C" gnn_status_t gnn_gt_attn_bwd(const gnn_plan_t* P, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                        const void* q, const void* k, const void* v, const float* lse,
                                        const void* dout, int32_t heads, int32_t head_dim, gnn_dtype_t dtype,
                                        float* delta, float* dq, float* dk, float* dv, void* ws, size_t ws_bytes,
                                        gnn_stream_t stream) {
    const char* who = "gnn_gt_attn_bwd";
    if (!check_common(P, rowptr, colidx, n, who)) return GNN_EINVAL;
    if (!P->opts.build_transpose) { set_error("%s: plan was built without build_transpose", who); return GNN_EINVAL; }
    if (!q || !k || !v || !lse || !dout || !delta || !dq || !dk || !dv || !ws) {
        set_error("%s: NULL pointer argument", who);
        return GNN_EINVAL;
    }
    if (!aligned32(q) || !aligned32(k) || !aligned32(v) || !aligned32(dout) || !aligned32(dq) || !aligned32(dk) ||
        !aligned32(dv) || !aligned32(ws)) {
        set_error("%s: feature/gradient pointers and workspace must be 32-byte aligned", who);
        return GNN_EINVAL;
    }
    HeadGroup hg[kMaxHeadGroups];
    const int ng = head_groups(n, heads, head_dim, dtype, hg, who), esz = dtype == GNN_F32 ? 4 : 2;
    if (!ng) return GNN_EUNSUPPORTED;
    const size_t need = ws_total(P, GNN_OP_GT_BWD, hg, ng, esz);
    if (ws_bytes < need) { set_error("%s: workspace too small (%zu < %zu)", who, ws_bytes, need); return GNN_EWORKSPACE; }
    cudaError_t e = cudaSuccess;
    for (int g = 0; g < ng && e == cudaSuccess; ++g) {
        const Shape& sh = hg[g].sh;
        const int h0 = hg[g].h0;
        const size_t fo = (size_t)h0 * head_dim * esz, go = (size_t)h0 * head_dim;
        const WsLayout w = ws_layout(P, GNN_OP_GT_BWD, sh, esz);
        GtArgs a = {};
        a.q = off_bytes(q, fo); a.k = off_bytes(k, fo); a.v = off_bytes(v, fo); a.dout = off_bytes(dout, fo);
        a.lse = const_cast<float*>(lse) + h0; a.delta = delta + h0;
        a.dq = dq + go; a.dk = dk + go; a.dv = dv + go;
        a.stat2 = (float2*)((char*)ws + w.stat2) + h0;
        e = launch_gt_bwd_dst(dtype, sh, make_ctx(P, false, ws, w, stream), a);                        // dQ, Delta
        if (e == cudaSuccess) e = launch_gt_bwd_src(dtype, sh, make_ctx(P, true, ws, w, stream), a);   // dK, dV
    }
    return cuda_status(e, who);
}

extern "C" gnn_status_t gnn_gatv2_fwd(const gnn_plan_t* P, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                      const void* xl, const void* xr, const float* a_, int32_t heads, int32_t head_dim,
                                      gnn_dtype_t dtype, float slope, void* out, float* lse, void* ws, size_t ws_bytes,
                                      gnn_stream_t stream) {
    const char* who = "gnn_gatv2_fwd";
    if (!check_common(P, rowptr, colidx, n, who)) return GNN_EINVAL;
    if (!xl || !xr || !a_ || !out || !lse || !ws) { set_error("%s: NULL pointer argument", who); return GNN_EINVAL; }
    if (!(slope >= 0.f) || !(slope < INFINITY)) { set_error("%s: LeakyReLU slope must be finite and >= 0", who); return GNN_EINVAL; }
    if (!aligned32(xl) || !aligned32(xr) || !aligned32(a_) || !aligned32(out) || !aligned32(ws)) {
        set_error("%s: feature pointers, a and workspace must be 32-byte aligned", who);
        return GNN_EINVAL;
    }
    HeadGroup hg[kMaxHeadGroups];
    const int ng = head_groups(n, heads, head_dim, dtype, hg, who), esz = dtype == GNN_F32 ? 4 : 2;
    if (!ng) return GNN_EUNSUPPORTED;
    const size_t need = ws_total(P, GNN_OP_GATV2_FWD, hg, ng, esz);
    if (ws_bytes < need) { set_error("%s: workspace too small (%zu < %zu)", who, ws_bytes, need); return GNN_EWORKSPACE; }
    cudaError_t e = cudaSuccess;
    for (int g = 0; g < ng && e == cudaSuccess; ++g) {
        const Shape& sh = hg[g].sh;
        const size_t fo = (size_t)hg[g].h0 * head_dim * esz;
        const WsLayout w = ws_layout(P, GNN_OP_GATV2_FWD, sh, esz);
        GatArgs a = {};
        a.xl = off_bytes(xl, fo); a.xr = off_bytes(xr, fo); a.a = a_ + (size_t)hg[g].h0 * head_dim;
        a.out = off_bytes(out, fo); a.lse = lse + hg[g].h0; a.slope = slope;
        e = launch_gat_fwd(dtype, sh, make_ctx(P, false, ws, w, stream), a);
    }
    return cuda_status(e, who);
}

extern "C" gnn_status_t gnn_gatv2_bwd(const gnn_plan_t* P, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                      const void* xl, const void* xr, const float* a_, const float* lse,
                                      const void* dout, int32_t heads, int32_t head_dim, gnn_dtype_t dtype,
                                      float slope, float* g, float* dxl, float* dxr, float* da, void* ws,
                                      size_t ws_bytes, gnn_stream_t stream) {
    const char* who = "gnn_gatv2_bwd";
    if (!check_common(P, rowptr, colidx, n, who)) return GNN_EINVAL;
    if (!P->opts.build_transpose) { set_error("%s: plan was built without build_transpose", who); return GNN_EINVAL; }
    if (!xl || !xr || !a_ || !lse || !dout || !g || !dxl || !dxr || !da || !ws) {
        set_error("%s: NULL pointer argument", who);
        return GNN_EINVAL;
    }
    if (!(slope >= 0.f) || !(slope < INFINITY)) { set_error("%s: LeakyReLU slope must be finite and >= 0", who); return GNN_EINVAL; }
    if (!aligned32(xl) || !aligned32(xr) || !aligned32(a_) || !aligned32(dout) || !aligned32(dxl) || !aligned32(dxr) ||
        !aligned32(ws)) {
        set_error("%s: feature/gradient pointers, a and workspace must be 32-byte aligned", who);
        return GNN_EINVAL;
    }
    HeadGroup hg[kMaxHeadGroups];
    const int ng = head_groups(n, heads, head_dim, dtype, hg, who), esz = dtype == GNN_F32 ? 4 : 2;
    if (!ng) return GNN_EUNSUPPORTED;
    const size_t need = ws_total(P, GNN_OP_GATV2_BWD, hg, ng, esz);
    if (ws_bytes < need) { set_error("%s: workspace too small (%zu < %zu)", who, ws_bytes, need); return GNN_EWORKSPACE; }
    cudaError_t e = cudaSuccess;
    for (int gi = 0; gi < ng && e == cudaSuccess; ++gi) {
        const Shape& sh = hg[gi].sh;
        const int h0 = hg[gi].h0;
        const size_t fo = (size_t)h0 * head_dim * esz, go = (size_t)h0 * head_dim;
        const WsLayout w = ws_layout(P, GNN_OP_GATV2_BWD, sh, esz);
        GatArgs a = {};
        a.xl = off_bytes(xl, fo); a.xr = off_bytes(xr, fo); a.a = a_ + go; a.dout = off_bytes(dout, fo);
        a.lse = const_cast<float*>(lse) + h0; a.g = g + h0; a.dxl = dxl + go; a.dxr = dxr + go;
        a.slope = slope;
        const LaunchCtx c = make_ctx(P, false, ws, w, stream);
        LaunchCtx ct = make_ctx(P, true, ws, w, stream);
        ct.da_slot_base = w.da_slots_dst;
        e = launch_gat_bwd_dst(dtype, sh, c, a);                                                       // dxl, G, da partials (xl . S)
        if (e == cudaSuccess) e = launch_gat_bwd_src(dtype, sh, ct, a);                                // dxr, da partials (xr . U)
        if (e == cudaSuccess) e = launch_da_reduce(c.da_part, w.da_slots, sh.rowe, da + go, c.stream);  // da
    }
    return cuda_status(e, who);
}

extern "C" gnn_status_t gnn_gt_attn_bwd_block(const gnn_plan_t* P, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                              const void* q, const void* k, const void* v, const float* lse, const void* dout,
                                              int32_t heads, int32_t head_dim, gnn_dtype_t dtype, float* delta, float* dq,
                                              float* dk, float* dv, void* ws, size_t ws_bytes, gnn_stream_t stream) {
    const char* who = "gnn_gt_attn_bwd_block";
    if (!check_common(P, rowptr, colidx, n, who)) return GNN_EINVAL;
    if (!P->blk_bitmap || !P->rem_rowptr_t) { set_error("%s: plan was built without GNN_BLOCKS_DIAG and build_transpose", who); return GNN_EINVAL; }
    if (!q || !k || !v || !lse || !dout || !delta || !dq || !dk || !dv || !ws) { set_error("%s: NULL pointer argument", who); return GNN_EINVAL; }
    if (!aligned32(q) || !aligned32(k) || !aligned32(v) || !aligned32(dout) || !aligned32(dq) || !aligned32(dk) || !aligned32(dv) ||
        !aligned32(ws)) {
        set_error("%s: feature / gradient pointers and workspace must be 32-byte aligned", who);
        return GNN_EINVAL;
    }
    if (dtype != GNN_BF16 || head_dim != 64 || heads < 1) {
        set_error("%s: unsupported shape heads=%d head_dim=%d dtype=%d (bf16, head_dim 64 only)", who, heads, head_dim, dtype);
        return GNN_EUNSUPPORTED;
    }
    HeadGroup hg[kMaxHeadGroups];
    const int ng = head_groups(n, heads, head_dim, dtype, hg, who);
    if (!ng) return GNN_EUNSUPPORTED;
    const BlockWs w = block_bwd_ws(P, hg, ng, heads);
    if (ws_bytes < w.total) { set_error("%s: workspace too small (%zu < %zu)", who, ws_bytes, w.total); return GNN_EWORKSPACE; }
    cudaStream_t st = (cudaStream_t)stream;
    GtArgs a = {};
    a.q = q; a.k = k; a.v = v; a.dout = dout; a.lse = const_cast<float*>(lse); a.delta = delta; a.dq = dq; a.dk = dk; a.dv = dv;
    a.stat2 = (float2*)((char*)ws + w.stat2);
    cudaError_t e = launch_gt_bwd_block(P, a, heads, st);         // Delta, dQ; tile-local dK, dV; (L, Delta) pairs
    if (e == cudaErrorNotSupported) { set_error("%s: cuTensorMapEncodeTiled unavailable or failed", who); return GNN_ECUDA; }
    // out-of-window edges of the source side: CSR src pass over the transposed remainder CSR, adding to dK / dV
    for (int g = 0; g < ng && e == cudaSuccess; ++g) {
        const Shape& sh = hg[g].sh;
        const int h0 = hg[g].h0;
        const size_t fo = (size_t)h0 * head_dim * 2, go = (size_t)h0 * head_dim;
        GtArgs b = {};
        b.q = off_bytes(q, fo); b.k = off_bytes(k, fo); b.v = off_bytes(v, fo); b.dout = off_bytes(dout, fo);
        b.dk = dk + go; b.dv = dv + go; b.stat2 = a.stat2 + h0; b.accumulate = 1;
        LaunchCtx c;
        c.stream = st; c.sm_count = P->sm_count; c.rowptr = P->rem_rowptr_t; c.colidx = P->rem_colidx_t; c.bins = P->rem_tr;
        c.partials = (float*)ws; c.da_part = nullptr; c.da_slot_base = 0;
        e = launch_gt_bwd_src(dtype, sh, c, b);
    }
    return cuda_status(e, who);
}

// ---- row f3: min / max aggregation.  The lane layout wants a power-of-two "head": factor channels = heads * head_dim
// with head_dim the largest power of two that divides it (the pass has no per-head arithmetic).
static int agg_groups(int32_t n, int32_t channels, int dtype, HeadGroup* hg, const char* who) {
    if (channels < 1) { set_error("%s: channels must be >= 1", who); return 0; }
    int hd = channels & -channels;
    const int cap = 1024 / (dtype == GNN_F32 ? 4 : 2);       // a "head" here is just a slice: keep it within one launch
    if (hd > cap) hd = cap;
    return head_groups(n, channels / hd, hd, dtype, hg, who);
}
static bool agg_shape(int32_t n, int32_t channels, int dtype, Shape& sh, const char* who) {
    HeadGroup hg[kMaxHeadGroups];
    if (!agg_groups(n, channels, dtype, hg, who)) return false;
    sh = hg[0].sh;    // the widest group: sizes the workspace
    return true;
}

extern "C" gnn_status_t gnn_seg_minmax_fwd(const gnn_plan_t* P, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                           const void* x, int32_t channels, gnn_dtype_t dtype, int32_t mode, void* out,
                                           int32_t* arg, void* ws, size_t ws_bytes, gnn_stream_t stream) {
    const char* who = "gnn_seg_minmax_fwd";
    if (!check_common(P, rowptr, colidx, n, who)) return GNN_EINVAL;
    if (!x || !out || !arg || !ws) { set_error("%s: NULL pointer argument", who); return GNN_EINVAL; }
    if (mode != GNN_AGG_MIN && mode != GNN_AGG_MAX) { set_error("%s: unknown mode %d", who, mode); return GNN_EINVAL; }
    if (!aligned32(x) || !aligned32(out) || !aligned32(arg) || !aligned32(ws)) {
        set_error("%s: x, out, arg and workspace must be 32-byte aligned", who);
        return GNN_EINVAL;
    }
    HeadGroup hg[kMaxHeadGroups];
    const int ng = agg_groups(n, channels, dtype, hg, who), esz = dtype == GNN_F32 ? 4 : 2;
    if (!ng) return GNN_EUNSUPPORTED;
    const size_t need = ws_total(P, GNN_OP_SEG_MINMAX_FWD, hg, ng, esz);
    if (ws_bytes < need) { set_error("%s: workspace too small (%zu < %zu)", who, ws_bytes, need); return GNN_EWORKSPACE; }
    cudaError_t e = cudaSuccess;
    for (int g = 0; g < ng && e == cudaSuccess; ++g) {      // channel groups of at most 1024 bytes (see head_groups)
        const Shape& sh = hg[g].sh;
        const size_t co = (size_t)hg[g].h0 * sh.d;           // first channel of the group
        const WsLayout w = ws_layout(P, GNN_OP_SEG_MINMAX_FWD, sh, esz);
        AggArgs a = {};
        a.x = off_bytes(x, co * esz); a.out = off_bytes(out, co * esz); a.arg = arg + co;
        a.sign = mode == GNN_AGG_MIN ? 1.f : -1.f;
        e = launch_min_fwd(dtype, sh, make_ctx(P, false, ws, w, stream), a, P->rows_sorted != 0);
    }
    return cuda_status(e, who);
}

extern "C" gnn_status_t gnn_seg_minmax_bwd(int32_t n, const int32_t* arg, const void* dout, int32_t channels,
                                           gnn_dtype_t dtype, float* dx, gnn_stream_t stream) {
    const char* who = "gnn_seg_minmax_bwd";
    if (n < 1 || !arg || !dout || !dx) { set_error("%s: n < 1 or NULL pointer argument", who); return GNN_EINVAL; }
    if (!aligned32(arg) || !aligned32(dout) || !aligned32(dx)) {
        set_error("%s: arg, dout and dx must be 32-byte aligned", who);
        return GNN_EINVAL;
    }
    Shape sh;
    if (!agg_shape(n, channels, dtype, sh, who)) return GNN_EUNSUPPORTED;
    cudaError_t e = cudaMemsetAsync(dx, 0, sizeof(float) * (size_t)n * channels, (cudaStream_t)stream);
    AggArgs a = {};
    a.arg = const_cast<int32_t*>(arg); a.dout = dout; a.dx = dx;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = launch_minmax_scatter(dtype, n, channels, a, sms, (cudaStream_t)stream);
    return cuda_status(e, who);
}
