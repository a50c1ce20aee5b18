/*
 * gnn_attn.h - C ABI of libgnn_attn.so: fused CSR graph attention for sm_100a (B200).
 *
 * The operations are the attention-family layers of arxiv/paper_2605_31500 (section 2.2,
 * lines 68-76), computed without ever writing an edge-wise E x H score / softmax / message tensor
 * to HBM:
 *
 *   h_i = sum_{j in N(i)} alpha_ij v_j,   alpha_ij = softmax_{j in N(i)} (e_ij)
 *   Graph Transformer:  e_ij = <q_i, k_j> / sqrt(head_dim),        v_j = v_j
 *   GATv2:              e_ij = a^T LeakyReLU(xl_i + xr_j),         v_j = xr_j
 *                       (xl = W_l h, xr = W_r h are projected by the caller)
 *   saved statistic:    L[i,h] = ln sum_j exp(e_ij)   (natural log)
 *
 * CONVENTIONS (all entry points)
 *   - Every data pointer is a DEVICE pointer owned by the caller; the library never allocates or
 *     frees device memory.  Feature, gradient and workspace pointers must be 32-byte aligned (256-bit gathers).
 *   - Graph: int32 CSR; ROW i = DESTINATION node, colidx[rowptr[i] .. rowptr[i+1]) = its sources j
 *     (in-neighbours).  The library processes exactly the stored entries: the caller stores the
 *     self-loop of N(i) u {i}; duplicate entries are separate softmax terms; a row with no
 *     entries yields O = 0, L = -inf and contributes no gradient.  nnz < 2^31.  colidx values are
 *     not range-checked.
 *   - Features: [n, heads, head_dim] row-major (node-major), dtype GNN_F32 or GNN_BF16.
 *     a: [heads, head_dim] fp32.  L, Delta, G: [n, heads] fp32.  ALL GRADIENT OUTPUTS ARE fp32
 *     [n, heads, head_dim] regardless of the feature dtype (reading A9); the forward
 *     output O has the feature dtype (bf16: round-to-nearest-even of the fp32 accumulator).
 *     All arithmetic is fp32.
 *   - Supported shapes: head_dim a power of two with 16 <= head_dim*sizeof(elt) <= 1024 bytes, any heads >= 1.
 *     One launch covers a row slice of at most 1024 bytes (32 lanes x 32 bytes); wider rows - e.g. the paper's
 *     fp32 (H, D) = (4, 128), (8, 64), (2, 256) grid points, PAPER.md:126-153 - are processed as consecutive
 *     head groups (at most 64) through the full-row strides, which changes no result because heads are
 *     independent in every pass.  Anything else returns GNN_EUNSUPPORTED.  gnn_seg_minmax_fwd and
 *     gnn_gt_attn_fwd_block state their own limits.
 *   - Every compute call is asynchronous on `stream` and never synchronises.  gnn_plan_build
 *     synchronises `stream` (it reads a few counters back to the host).
 *   - Return value: GNN_OK or an error code; nothing is launched when an error is returned for
 *     argument validation.  gnn_last_error() returns a thread-local message for the last error.
 *   - Determinism: the attention entry points (forward, backward, block / WSB variants) and gnn_seg_minmax_fwd
 *     use no floating-point atomics; their results are bit-reproducible run to run for the same plan
 *     options and device.  The one exception is gnn_seg_minmax_bwd, the paper's scatter-add:
 *     it uses red.global.add.f32, so dx is reproducible only up to fp32 rounding (stated at the call).
 */
#ifndef GNN_ATTN_H_
#define GNN_ATTN_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Opaque stream handle: pass a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream). */
typedef void* gnn_stream_t;

typedef enum { GNN_OK = 0, GNN_EINVAL = 1, GNN_EUNSUPPORTED = 2, GNN_EWORKSPACE = 3, GNN_ECUDA = 4 } gnn_status_t;
typedef enum { GNN_F32 = 0, GNN_BF16 = 1 } gnn_dtype_t;

/* Degree-aware row binning (PAPER.md:326, :456-460, :472 describe a light/heavy split with its own
 * launch shape per bucket; the thresholds and the chunking rule below are this library's own).
 *   deg <= warp_max_deg            : "group rows"  - one lane group (row_bytes/16 lanes) per row
 *   warp_max_deg < deg <= cta_max  : "CTA rows"    - one CTA per row, merged in shared memory
 *   deg > cta_max_deg              : "hub rows"    - cut into ceil(deg/split_chunk) near-equal chunks,
 *                                    one CTA per chunk, partial states merged by a second pass
 * Zero in any threshold selects the default (4096 / 16384 / 4096 if nnz >= 2^24, else 256 / 1024 / 512).
 * build_transpose: GNN_TRANSPOSE_NONE (0) forward only; GNN_TRANSPOSE_BUILD (1) also builds CSR^T and its bins
 * (needed by the backward calls); GNN_TRANSPOSE_UNDIRECTED (2) is the direction-aware mode of PAPER.md:343: the
 * caller declares the graph undirected (rows strictly ascending, a mirror (j, i) for every entry (i, j));
 * gnn_plan_build verifies that on the device (GNN_EINVAL if it does not hold) and the backward calls then traverse
 * the forward CSR and its bins: no transposed structure is built or stored (plan storage drops by 4*(nnz + n) bytes
 * plus the second bin set), and the gradients are bit-identical to mode 1, for which CSR^T == CSR bit for bit.
 * build_blocks: bit mask.  GNN_BLOCKS_DIAG (1) also builds the diagonal 16-row block layout (gnn_gt_attn_fwd_block);
 * GNN_BLOCKS_WSB (2) also builds the general WSB layout of PAPER.md:545 (gnn_gt_attn_fwd_wsb / _bwd_wsb) for the CSR
 * and - with build_transpose - for CSR^T (in the undirected mode the two coincide and one copy is stored).       */
enum { GNN_TRANSPOSE_NONE = 0, GNN_TRANSPOSE_BUILD = 1, GNN_TRANSPOSE_UNDIRECTED = 2 };
enum { GNN_BLOCKS_NONE = 0, GNN_BLOCKS_DIAG = 1, GNN_BLOCKS_WSB = 2 };
typedef struct {
    int32_t warp_max_deg;
    int32_t cta_max_deg;
    int32_t split_chunk;
    int32_t build_transpose;
    int32_t build_blocks;
} gnn_plan_opts_t;

typedef struct gnn_plan gnn_plan_t; /* host handle; views caller-provided device storage */

/* Bytes of device storage a plan for (n, nnz, opts) needs: `dev_bytes` must stay allocated for the
 * life of the plan, `scratch_bytes` only during gnn_plan_build.  Needs a CUDA device.            */
gnn_status_t gnn_plan_bytes(int32_t n, int64_t nnz, const gnn_plan_opts_t* opts, size_t* dev_bytes,
                            size_t* scratch_bytes);

/* Build the integer metadata, a pure function of (rowptr, colidx, opts) (bit-exact against
 * oracle/plan_ref.py):
 *   bins   : perm[n] = row ids sorted by (key, row id), key = 0 for hub rows, 1 + (32 - bitlen(deg))
 *            for CTA rows, 34 + (32 - bitlen(deg)) for group rows  (heaviest first)
 *   chunks : (row, e_begin, e_end, hub_slot) int32 x4 per chunk, in (hub_slot, chunk) order,
 *            chunk t of a hub row with degree g and c chunks = [b + floor(t g / c), b + floor((t+1) g / c))
 *   CSR^T  : rowptr_t[n+1], colidx_t[nnz] by a STABLE sort on the source id,
 *            plus the same bins / chunks for CSR^T (out-degrees)
 *   blocks : see gnn_gt_attn_fwd_block
 *   WSB    : per 16-row window the sorted unique source columns cut into Tensor Core Blocks of width 8; per TCB
 *            8 column ids (zero padded) and a 128-bit bitmap of its 16 x 8 edges; tcb_row_offset per window
 *            (PAPER.md:545).  n_dup = entries beyond the first of their (dst, src) pair (not representable).
 * rowptr/colidx: device, must outlive the plan (the plan keeps the pointers, not a copy).
 * On success *plan is a host handle to free with gnn_plan_destroy (device storage stays the caller's). */
gnn_status_t gnn_plan_build(gnn_plan_t** plan, void* dev_mem, size_t dev_bytes, void* scratch, size_t scratch_bytes,
                            int32_t n, int64_t nnz, const int32_t* rowptr, const int32_t* colidx,
                            const gnn_plan_opts_t* opts, gnn_stream_t stream);
void gnn_plan_destroy(gnn_plan_t* plan);

/* Optional input check (the compute calls never range-check colidx: a bad index is an out-of-bounds gather).
 * Verifies on the device that rowptr[0] == 0, rowptr[n] == nnz, rowptr is non-decreasing and every colidx is in
 * [0, n).  rowptr / colidx: device.  Synchronises the stream.  GNN_EINVAL (message names the first kind of
 * violation and the smallest offending position) if the CSR is malformed; uses no plan and no workspace
 * beyond 16 bytes it takes from `scratch` (device, 16-byte aligned).                                 */
gnn_status_t gnn_csr_validate(int32_t n, int64_t nnz, const int32_t* rowptr, const int32_t* colidx, void* scratch,
                              gnn_stream_t stream);

/* Plan introspection for the bit-exact metadata check.  `what`:                                    */
enum {
    GNN_PLAN_COUNTS = 0,    /* int32[8]: n_hub, n_cta, n_group, n_chunks, then the same 4 for CSR^T  */
    GNN_PLAN_PERM = 1,      /* int32[n]                                                             */
    GNN_PLAN_CHUNKS = 2,    /* int32[n_chunks][4]                                                   */
    GNN_PLAN_CHUNK_PTR = 3, /* int32[n_hub + 1]                                                     */
    GNN_PLAN_ROWPTR_T = 4,  /* int32[n + 1]                                                         */
    GNN_PLAN_COLIDX_T = 5,  /* int32[nnz]                                                           */
    GNN_PLAN_PERM_T = 6,
    GNN_PLAN_CHUNKS_T = 7,
    GNN_PLAN_CHUNK_PTR_T = 8,
    GNN_PLAN_BLOCK_BITMAP = 9,      /* uint16[n_windows][16]                                         */
    GNN_PLAN_BLOCK_REM_ROWPTR = 10, /* int32[n + 1]                                                  */
    GNN_PLAN_BLOCK_REM_COLIDX = 11, /* int32[rem_nnz]                                                */
    GNN_PLAN_FLAGS = 12,            /* int32[2]: [0] = 1 if every CSR row lists its sources in ascending order;
                                       [1] = 1 if the backward traverses the forward CSR (GNN_TRANSPOSE_UNDIRECTED) */
    /* general WSB layout, bit-exact against oracle/plan_ref.py::build_wsb:                  */
    GNN_PLAN_WSB_INFO = 13,         /* int32[6]: has_wsb, n_windows, n_tcb, n_dup, n_tcb of CSR^T, n_dup of CSR^T   */
    GNN_PLAN_WSB_ROW_OFFSET = 14,   /* int32[n_windows + 1]: tcb_row_offset                                        */
    GNN_PLAN_WSB_COLS = 15,         /* int32[n_tcb][8]: global column ids of each TCB, zero padded                 */
    GNN_PLAN_WSB_BITMAP = 16,       /* uint8[n_tcb][16]: byte r = row r of the window, bit c = column c of the TCB */
    GNN_PLAN_WSB_ROW_OFFSET_T = 17, /* the same three for CSR^T (source windows x destination columns)             */
    GNN_PLAN_WSB_COLS_T = 18,
    GNN_PLAN_WSB_BITMAP_T = 19,
    GNN_PLAN_BLOCK_REM_ROWPTR_T = 20, /* int32[n + 1]: stable transpose of the remainder CSR of the diagonal block layout   */
    GNN_PLAN_BLOCK_REM_COLIDX_T = 21  /* int32[rem_nnz] (plans built with GNN_BLOCKS_DIAG and build_transpose)             */
};
/* Copies the item to HOST memory `host_dst` (synchronous).  *bytes in = capacity, out = size needed;
 * with host_dst == NULL only the size is returned.                                                 */
gnn_status_t gnn_plan_export(const gnn_plan_t* plan, int what, void* host_dst, size_t* bytes);
/* Device pointers to CSR^T held by the plan (NULL if build_transpose was 0; the caller's own rowptr / colidx
 * in the undirected mode).                                                                          */
const int32_t* gnn_plan_rowptr_t(const gnn_plan_t* plan);
const int32_t* gnn_plan_colidx_t(const gnn_plan_t* plan);

/* Workspace (device bytes) a compute call needs: hub-chunk partial states
 * [n_chunks][(n_acc * heads*head_dim + n_scalar * heads)] fp32 and, for gnn_gatv2_bwd, the per-CTA
 * `da` partials.  O(#chunks * H * d), never O(E * H).  `op`:                                         */
enum { GNN_OP_GT_FWD = 0, GNN_OP_GT_BWD = 1, GNN_OP_GATV2_FWD = 2, GNN_OP_GATV2_BWD = 3,
       GNN_OP_GT_FWD_BLOCK = 4 /* needs no workspace: 0 bytes */,
       GNN_OP_SEG_MINMAX_FWD = 5 /* pass heads = 1, head_dim = channels */,
       GNN_OP_WSB_FWD = 6, GNN_OP_WSB_BWD = 7 /* tile-local: 0 bytes */,
       GNN_OP_GT_BWD_BLOCK = 8 };
gnn_status_t gnn_workspace_bytes(const gnn_plan_t* plan, int op, int32_t heads, int32_t head_dim, gnn_dtype_t dtype,
                                 size_t* bytes);

/* ---------------------------------------------------------------------------------------------
 * Graph Transformer attention, forward (fused CSR kernel PAPER.md:484-492).
 *   s_ij = <q[i,h,:], k[j,h,:]> / sqrt(head_dim);  L[i,h] = ln sum_j exp(s_ij);
 *   out[i,h,:] = sum_j exp(s_ij - L[i,h]) v[j,h,:]        (online softmax)
 * q, k, v: [n,H,d] `dtype`, in.  out: [n,H,d] `dtype`, out.  lse: [n,H] fp32, out.
 * rowptr/colidx must be the arrays the plan was built from.  ws: >= gnn_workspace_bytes(GT_FWD).  */
gnn_status_t gnn_gt_attn_fwd(const gnn_plan_t* plan, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                             const void* q, const void* k, const void* v, int32_t heads, int32_t head_dim,
                             gnn_dtype_t dtype, void* out, float* lse, void* ws, size_t ws_bytes,
                             gnn_stream_t stream);

/* Graph Transformer attention, backward, recomputing alpha from lse:
 *   alpha_ij = exp(s_ij - L_i);  dP_ij = <dout_i, v_j>;  Delta_i = sum_j alpha_ij dP_ij (= <O_i, dO_i>)
 *   dS_ij = alpha_ij (dP_ij - Delta_i)
 *   dq_i = sum_j dS_ij k_j / sqrt(d)      (dst pass over CSR, row-local, no atomics)
 *   dk_j = sum_i dS_ij q_i / sqrt(d);  dv_j = sum_i alpha_ij dout_i
 *                                         (src pass over CSR^T in CSR^T order: deterministic, no atomics)
 * q, k, v, dout: [n,H,d] `dtype`, in.  lse: [n,H] fp32, in (from the forward).
 * delta: [n,H] fp32, OUT (scratch the caller provides; holds Delta on return).
 * dq, dk, dv: [n,H,d] fp32, out.  The plan must have been built with build_transpose.
 * The forward output O is not needed (Delta is formed in fp32 inside the dst pass).              */
gnn_status_t gnn_gt_attn_bwd(const gnn_plan_t* plan, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                             const void* q, const void* k, const void* v, const float* lse, const void* dout,
                             int32_t heads, int32_t head_dim, gnn_dtype_t dtype, float* delta, float* dq,
                             float* dk, float* dv, void* ws, size_t ws_bytes, gnn_stream_t stream);

/* GATv2 attention, forward:
 *   s_ij = sum_c a[h,c] LeakyReLU_slope(xl[i,h,c] + xr[j,h,c]);  softmax / lse / out as above with
 *   value xr[j,h,:].  xl, xr: [n,H,d] `dtype`, in.  a: [H,d] fp32, in.  out, lse: as gnn_gt_attn_fwd.
 *   slope: finite and >= 0 (GNN_EINVAL otherwise; same for gnn_gatv2_bwd).                            */
gnn_status_t gnn_gatv2_fwd(const gnn_plan_t* plan, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                           const void* xl, const void* xr, const float* a, int32_t heads, int32_t head_dim,
                           gnn_dtype_t dtype, float slope, void* out, float* lse, void* ws, size_t ws_bytes,
                           gnn_stream_t stream);

/* GATv2 attention, backward:
 *   z_ij = xl_i + xr_j;  alpha_ij = exp(s_ij - L_i);  dP_ij = <dout_i, xr_j>;  G_i = sum_j alpha_ij dP_ij
 *   de_ij = alpha_ij (dP_ij - G_i);  LeakyReLU'(z) = 1 if z > 0 else slope
 *   dxl_i = sum_j de_ij a . LeakyReLU'(z_ij)                              (dst pass, "AL" kernel)
 *   da    = sum_ij de_ij LeakyReLU(z_ij)    (= sum_i xl_i . S_i + sum_j xr_j . U_j with S, U the LeakyReLU'-weighted
 *                                            sums of de of the two passes; per-CTA fp32 partials, fixed-order fp64 final reduction)
 *   dxr_j = sum_i ( alpha_ij dout_i + de_ij a . LeakyReLU'(z_ij) )        (src pass over CSR^T, "R" kernel)
 * g: [n,H] fp32, OUT (holds G on return).  dxl, dxr: [n,H,d] fp32, out.  da: [H,d] fp32, out.     */
gnn_status_t gnn_gatv2_bwd(const gnn_plan_t* plan, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                           const void* xl, const void* xr, const float* a, const float* lse, const void* dout,
                           int32_t heads, int32_t head_dim, gnn_dtype_t dtype, float slope, float* g, float* dxl,
                           float* dxr, float* da, void* ws, size_t ws_bytes, gnn_stream_t stream);

/* Graph Transformer attention forward, block-sparse tensor-core variant for locally dense graphs (the paper's
 * WSB / Tensor-Core forward, re-designed for tcgen05 + TMEM): tiles of 128 destination rows
 * (8 windows of 16) compute S = Q_tile K_tile^T and O = P V_tile with tcgen05.mma, masked by the plan's per-row
 * 16-bit bitmaps of in-window edges; every other edge (the remainder CSR of the plan) is gathered as in
 * gnn_gt_attn_fwd and merged into the same online softmax.  Same result as gnn_gt_attn_fwd up to rounding
 * (P is rounded to bf16 for the second product).  The plan must have been built with build_blocks;
 * bf16 features, head_dim == 64 only (GNN_EUNSUPPORTED otherwise); feature pointers 32-byte aligned; no workspace. */
gnn_status_t gnn_gt_attn_fwd_block(const gnn_plan_t* plan, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                   const void* q, const void* k, const void* v, int32_t heads, int32_t head_dim,
                                   gnn_dtype_t dtype, void* out, float* lse, gnn_stream_t stream);

/* Backward of the same function on the diagonal block layout, tensor cores for the in-window edges (PAPER.md:563:
 * P = exp(S - L), dV = P^T dO, dP = dO V^T, dS = P o (dP - Delta), dQ = dS K, dK = dS^T Q) - tile-local, hence no atomics
 * - and the remainder CSR for every other edge: its dst-side terms (Delta, dQ) inside the tile kernel, its src-side terms
 * (dK, dV) through the CSR src pass over the transposed remainder CSR of the plan, added to the tile-local part.
 * Same results as gnn_gt_attn_bwd up to rounding (dS / P rounded to bf16 for the in-window products; Delta fp32).
 * Plan: GNN_BLOCKS_DIAG and build_transpose != 0.  bf16, head_dim == 64.  Arguments as gnn_gt_attn_bwd;
 * ws >= gnn_workspace_bytes(GNN_OP_GT_BWD_BLOCK).                                                                  */
gnn_status_t gnn_gt_attn_bwd_block(const gnn_plan_t* plan, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                   const void* q, const void* k, const void* v, const float* lse, const void* dout,
                                   int32_t heads, int32_t head_dim, gnn_dtype_t dtype, float* delta, float* dq, float* dk,
                                   float* dv, void* ws, size_t ws_bytes, gnn_stream_t stream);

/* ---------------------------------------------------------------------------------------------
 * Graph Transformer attention on the general WSB block-sparse layout, forward and backward on the
 * tensor cores (tcgen05 / TMEM).  Same functions as gnn_gt_attn_fwd / _bwd up to rounding (the softmax weights P and
 * the score gradients dS are rounded to bf16 before their second products).  A CTA owns 128 rows = 8 row windows and
 * walks the windows' TCB pairs: S = Q K_blk^T, bitmap mask, online softmax, acc += P V_blk (forward);
 * P = exp(S - L), dV = P^T dO, dP = dO V^T, dS = P o (dP - Delta), dQ = dS K, dK = dS^T Q (backward) - with the
 * source-side gradients computed over the WSB layout of the TRANSPOSED graph, so that no atomics are needed (the
 * paper accumulates dK / dV with atomicAdd; on an undirected graph both layouts are the same arrays).
 * The plan must have been built with GNN_BLOCKS_WSB (and build_transpose for the backward) from a CSR WITHOUT duplicate
 * entries (a bitmap stores each (dst, src) pair once: GNN_EUNSUPPORTED otherwise).  bf16 features, head_dim 32, 64 or 128
 * (GNN_EUNSUPPORTED otherwise); feature / gradient pointers 32-byte aligned; no workspace; asynchronous on `stream`.
 *   forward : q, k, v [n,H,d] bf16 in; out [n,H,d] bf16, lse [n,H] fp32 out.
 *   backward: q, k, v, dout in; out = the forward output O (bf16, in: its row dot <O_i, dO_i> centres the bf16-staged
 *             products; Delta itself is accumulated in fp32 and the result does not depend on O's rounding); lse in;
 *             delta [n,H] fp32 OUT; dq, dk, dv [n,H,d] fp32 out.                                                  */
gnn_status_t gnn_gt_attn_fwd_wsb(const gnn_plan_t* plan, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                 const void* q, const void* k, const void* v, int32_t heads, int32_t head_dim,
                                 gnn_dtype_t dtype, void* out, float* lse, gnn_stream_t stream);
gnn_status_t gnn_gt_attn_bwd_wsb(const gnn_plan_t* plan, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                 const void* q, const void* k, const void* v, const void* out, const float* lse,
                                 const void* dout, int32_t heads, int32_t head_dim, gnn_dtype_t dtype, float* delta,
                                 float* dq, float* dk, float* dv, gnn_stream_t stream);

/* ---------------------------------------------------------------------------------------------
 * Degree-aware min / max neighbourhood aggregation with argmin (PAPER.md:124-151 section 3.1, :452-474 App. D.1):
 *   out[i,c] = min (mode GNN_AGG_MIN) or max (GNN_AGG_MAX) over the stored in-neighbours j of i of x[j,c]
 *   arg[i,c] = the source j that attains it; ties go to the smaller j (the paper's packed (value, index)
 *              atomicMin); values compare as IEEE numbers (-0.0 == +0.0; +-inf are ordinary values: a row
 *              whose candidates are all +inf returns +inf and the smallest such j); NaN inputs are outside the contract
 *              (result unspecified); rows without entries give 0 / -1.
 * x, out: [n, channels] `dtype`; arg: [n, channels] int32, out.  channels*sizeof(dtype) must be a multiple of 16
 * (GNN_EUNSUPPORTED otherwise); rows wider than 1024 bytes run as consecutive channel groups (at most 64).  Runs on the plan's degree bins (packed rows, CTA rows, hub chunks
 * merged by the lexicographic (value, index) minimum): no atomics, deterministic.
 * ws: >= gnn_workspace_bytes(GNN_OP_SEG_MINMAX_FWD, heads = 1, head_dim = channels).  Pointers 32-byte aligned. */
enum { GNN_AGG_MIN = 0, GNN_AGG_MAX = 1 };
gnn_status_t gnn_seg_minmax_fwd(const gnn_plan_t* plan, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                const void* x, int32_t channels, gnn_dtype_t dtype, int32_t mode, void* out,
                                int32_t* arg, void* ws, size_t ws_bytes, gnn_stream_t stream);
/* Backward: dx[arg[i,c], c] += dout[i,c] for every (i,c) with arg >= 0, a sparse scatter-add
 * through the indices the forward saved.  arg: [n, channels] int32, in; dout: [n, channels] `dtype`, in;
 * dx: [n, channels] fp32, out (the call zeroes it first).  Uses red.global.add.f32: the order of the additions
 * into one dx element is not fixed, so dx is reproducible only up to fp32 rounding.  Needs no plan, no workspace. */
gnn_status_t gnn_seg_minmax_bwd(int32_t n, const int32_t* arg, const void* dout, int32_t channels, gnn_dtype_t dtype,
                                float* dx, gnn_stream_t stream);

/* Thread-local message describing the last error returned on this thread ("" if none).           */
const char* gnn_last_error(void);
/* Library version string, e.g. "gnn_attn 0.1 sm_100a".                                            */
const char* gnn_version(void);
/* Number of kernel launches the library has issued in this process (all threads; atomic counter). */
int64_t gnn_launch_count(void);
/* Test / measurement aid: switches the programmatic-dependent-launch overlap of a pass's two traversal kernels
 * off (0) or on (1, the default) for the whole process.  Results are bit-identical either way (the overlapped
 * kernels touch disjoint rows, and the dependent kernel ends in griddepcontrol.wait).      */
void gnn_pdl_enable(int on);

/* Measurement aid (bench.py): when enabled, every kernel launch of the library is bracketed by two
 * CUDA events on the launch stream.  gnn_profile_collect synchronises on them, writes up to
 * max_records records - names[i] is a 48-byte NUL-terminated "pass/kernel" string, ms[i] its device
 * time in milliseconds, in launch order - clears the list and returns the number written.  Not
 * thread-safe; off by default (the timed `value` runs have it off).                                */
void gnn_profile_enable(int on);
int32_t gnn_profile_collect(char* names, float* ms, int32_t max_records);

/* ---------------------------------------------------------------------------------------------
 * The rest of the Graph Transformer block the paper timed: LayerNorm fused into the QKV projection.
 *   y[i,:] = (x[i,:] - mean_i) / sqrt(var_i + eps) * gamma + beta    (over the c_in features, biased variance)
 *   q | k | v [i,:] = y[i,:] W^T + bias,  W = [W_Q; W_K; W_V]: [3*heads*head_dim, c_in] row-major
 * One tcgen05 GEMM whose A operand is normalised on the way into shared memory: y never exists in HBM.
 * x: [n, c_in] bf16; gamma, beta: [c_in] fp32; w: bf16; bias: [3*heads*head_dim] fp32 or NULL; q, k, v: [n,H,d] bf16 out
 * (fp32 accumulation, one bf16 rounding of y and one of the outputs).  c_in a multiple of 64 in [64, 512],
 * heads*head_dim a multiple of 128 (GNN_EUNSUPPORTED otherwise); x, w, q, k, v 32-byte aligned; no workspace; async. */
gnn_status_t gnn_ln_qkv_fwd(int32_t n, int32_t c_in, int32_t heads, int32_t head_dim, const void* x, const float* gamma,
                            const float* beta, float eps, const void* w, const float* bias, void* q, void* k, void* v,
                            gnn_stream_t stream);

/* The paper's `dot-aggr` locality micro-benchmark: out[i] = sum over the stored in-neighbours j of i
 * of <x[i,:], x[j,:]>, fp32, as two warp-per-node kernels with identical arithmetic: mode 0 = feature-parallel (lanes
 * over the features, neighbours scanned sequentially, coalesced loads), mode 1 = neighbour-parallel (every lane walks a
 * different neighbour's row, gather-like loads); vec 0 = 4-byte loads, 1 = 16-byte loads.  x: [n, dim] fp32, dim a
 * multiple of 4, 16-byte aligned; out: [n] fp32.  Needs no plan.  Summation order differs between the modes (results
 * agree to fp32 rounding).  Asynchronous on `stream`.                                                              */
gnn_status_t gnn_dot_aggr(int32_t n, const int32_t* rowptr, const int32_t* colidx, const float* x, int32_t dim, int32_t mode,
                          int32_t vec, float* out, gnn_stream_t stream);

/* Measurement aid (bench.py): ONE launch that gathers n_idx rows of row_bytes (256 | 512 | 1024) bytes at the row
 * indices idx[0..n_idx) (each in [0, table_rows)) from `table` and discards them - the achievable gather-ingest rate
 * ("ceiling 2" of DESIGN.md section 6: HBM-resident when the table is far larger than L2, L2-resident when it fits),
 * which the caller times with CUDA events on `stream`.  mode 0: one 256-bit load per lane per row, `depth` (1|2|4|8)
 * rows in flight per lane group, as the traversal kernels do; mode 1: cp.async.bulk copies into a shared-memory ring,
 * `depth` (4|8|16) rows per stage.  ctas_per_sm (1..16) CTAs of 128 threads per SM.  table, idx, sink: device;
 * table 32-byte aligned; sink: one float the kernel never writes for finite table contents.  Asynchronous.        */
gnn_status_t gnn_probe_gather(const void* table, int64_t table_rows, int32_t row_bytes, const int32_t* idx, int64_t n_idx,
                              int32_t mode, int32_t depth, int32_t ctas_per_sm, float* sink, gnn_stream_t stream);

/* Graph Transformer attention forward WITHOUT any caller-supplied or allocated scratch: gnn_gt_attn_fwd (same operation,
 * same arguments and layouts) with the pass's scratch - the per-chunk partial softmax states of
 * split hub rows - in a file-scope __device__ array inside the library, for callers that cannot
 * call cudaMalloc (CUDA graph capture, serving loops).  The array holds gnn_static_workspace_limit() bytes (16 MiB; every
 * GPU that loads the library holds it until exit); a graph / shape whose gnn_workspace_bytes(GNN_OP_GT_FWD) exceeds it is
 * refused with GNN_EWORKSPACE and a message.  The call allocates and frees nothing on host or device.  ALL calls on a
 * device share the array (it keeps the previous call's contents; nothing in it needs clearing - every partial is
 * written before it is read within a call): calls that may overlap on the GPU (unordered streams, two host threads)
 * RACE on it - order them.  The plan must live on the current device.  Asynchronous on `stream`.                    */
size_t gnn_static_workspace_limit(void);
gnn_status_t gnn_gt_attn_fwd_static(const gnn_plan_t* plan, const int32_t* rowptr, const int32_t* colidx, int32_t n,
                                    const void* q, const void* k, const void* v, int32_t heads, int32_t head_dim,
                                    gnn_dtype_t dtype, void* out, float* lse, gnn_stream_t stream);

#ifdef __cplusplus
}
#endif
#endif /* GNN_ATTN_H_ */
