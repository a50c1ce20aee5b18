// static_ws.cu - gnn_gt_attn_fwd_static: the Graph Transformer forward (gnn_gt_attn_fwd) for callers
// that cannot allocate device memory at all (code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc).  The pass's scratch - the per-chunk partial softmax states (m, l, acc) of split hub rows that
// segment_kernel writes and hub_merge_kernel reads - lives in a file-scope __device__ array of
// kStaticWsBytes bytes instead of a caller-supplied workspace.  Every GPU that loads the library holds that array until
// the process exits.
//
// The array's NAME is a host-side stand-in in host code, not a device address: its device address is looked up once per
// device with cudaGetSymbolAddress (with that device current) and that pointer is what the kernels receive.
//
// Shared state: every call on a device uses the same array.  Nothing in it has to start at zero - each chunk's partial
// state is written in full by the segment kernel before the hub merge of the same call reads it - so no clearing is
// needed and the previous call's contents are simply overwritten.  Calls that may OVERLAP on the GPU (different streams
// without an ordering between them, or two host threads) race on the array; order them on one stream or with events.
//
// The entry point calls no cudaMalloc / cudaFree / allocating library routine: cudaGetDevice, cudaGetSymbolAddress,
// the size query and the launches of the existing path only.
#include <cuda_runtime.h>

#include <atomic>

#include "../../include/gnn_attn.h"
#include "internal.h"

namespace {

constexpr size_t kStaticWsBytes = (size_t)16 << 20;     // 16 MiB: cfg 3 (2.4 M nodes, 126 M edges, H = 4, d = 64) needs < 4 MiB
constexpr int kMaxDevices = 64;

static __device__ __align__(256) unsigned char g_static_ws[kStaticWsBytes];

// device address of g_static_ws per device ordinal (0 = not looked up yet); the lookup is idempotent, so a benign race
// between two host threads stores the same value twice
std::atomic<void*> g_ws_addr[kMaxDevices];

}  // namespace

extern "C" size_t gnn_static_workspace_limit(void) { return kStaticWsBytes; }

extern "C" gnn_status_t gnn_gt_attn_fwd_static(const gnn_plan_t* plan, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                               const void* q, const void* k, const void* v, int32_t heads, int32_t head_dim,
                                               gnn_dtype_t dtype, void* out, float* lse, gnn_stream_t stream) {
    const char* who = "gnn_gt_attn_fwd_static";
    if (!plan) { gnn::set_error("%s: NULL plan", who); return GNN_EINVAL; }
    size_t need = 0;
    const gnn_status_t s = gnn_workspace_bytes(plan, GNN_OP_GT_FWD, heads, head_dim, dtype, &need);
    if (s != GNN_OK) return s;                            // the size query has set the error text
    if (need > kStaticWsBytes) {
        gnn::set_error("%s: this graph / shape needs %zu bytes of scratch, the built-in array holds %zu "
                       "(use gnn_gt_attn_fwd with a caller-supplied workspace)", who, need, kStaticWsBytes);
        return GNN_EWORKSPACE;
    }
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { gnn::set_error("%s: cudaGetDevice: %s", who, cudaGetErrorString(e)); return GNN_ECUDA; }
    if (dev < 0 || dev >= kMaxDevices) { gnn::set_error("%s: device ordinal %d outside [0, %d)", who, dev, kMaxDevices); return GNN_EUNSUPPORTED; }
    void* ws = g_ws_addr[dev].load(std::memory_order_acquire);
    if (!ws) {                                            // set-up, once per device, with that device current
        e = cudaGetSymbolAddress(&ws, g_static_ws);
        if (e != cudaSuccess || !ws) {
            gnn::set_error("%s: cudaGetSymbolAddress: %s", who, cudaGetErrorString(e));
            return GNN_ECUDA;
        }
        g_ws_addr[dev].store(ws, std::memory_order_release);
    }
    return gnn_gt_attn_fwd(plan, rowptr, colidx, n, q, k, v, heads, head_dim, dtype, out, lse, ws, kStaticWsBytes, stream);
}
