"""ctypes binding of include/gnn_attn.h.  Same names as the C ABI; tensors are marshalled to raw
device pointers, nothing is computed here."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libgnn_attn.so")

GNN_OK, GNN_EINVAL, GNN_EUNSUPPORTED, GNN_EWORKSPACE, GNN_ECUDA = range(5)
GNN_F32, GNN_BF16 = 0, 1
GNN_OP_GT_FWD, GNN_OP_GT_BWD, GNN_OP_GATV2_FWD, GNN_OP_GATV2_BWD = 0, 1, 2, 3
GNN_OP_GT_FWD_BLOCK, GNN_OP_SEG_MINMAX_FWD, GNN_OP_WSB_FWD, GNN_OP_WSB_BWD, GNN_OP_GT_BWD_BLOCK = 4, 5, 6, 7, 8
GNN_AGG_MIN, GNN_AGG_MAX = 0, 1
GNN_TRANSPOSE_NONE, GNN_TRANSPOSE_BUILD, GNN_TRANSPOSE_UNDIRECTED = 0, 1, 2
(GNN_PLAN_COUNTS, GNN_PLAN_PERM, GNN_PLAN_CHUNKS, GNN_PLAN_CHUNK_PTR, GNN_PLAN_ROWPTR_T, GNN_PLAN_COLIDX_T,
 GNN_PLAN_PERM_T, GNN_PLAN_CHUNKS_T, GNN_PLAN_CHUNK_PTR_T, GNN_PLAN_BLOCK_BITMAP, GNN_PLAN_BLOCK_REM_ROWPTR,
 GNN_PLAN_BLOCK_REM_COLIDX, GNN_PLAN_FLAGS, GNN_PLAN_WSB_INFO, GNN_PLAN_WSB_ROW_OFFSET, GNN_PLAN_WSB_COLS,
 GNN_PLAN_WSB_BITMAP, GNN_PLAN_WSB_ROW_OFFSET_T, GNN_PLAN_WSB_COLS_T, GNN_PLAN_WSB_BITMAP_T,
 GNN_PLAN_BLOCK_REM_ROWPTR_T, GNN_PLAN_BLOCK_REM_COLIDX_T) = range(22)
GNN_BLOCKS_NONE, GNN_BLOCKS_DIAG, GNN_BLOCKS_WSB = 0, 1, 2

EXPORTED_SYMBOLS = [
    "gnn_csr_validate", "gnn_plan_bytes", "gnn_plan_build", "gnn_plan_destroy", "gnn_plan_export", "gnn_plan_rowptr_t",
    "gnn_plan_colidx_t", "gnn_workspace_bytes", "gnn_gt_attn_fwd", "gnn_gt_attn_bwd", "gnn_gatv2_fwd",
    "gnn_gatv2_bwd", "gnn_gt_attn_fwd_block", "gnn_gt_attn_fwd_wsb", "gnn_gt_attn_bwd_wsb", "gnn_gt_attn_bwd_block", "gnn_seg_minmax_fwd", "gnn_seg_minmax_bwd", "gnn_last_error", "gnn_version", "gnn_launch_count", "gnn_profile_enable",
    "gnn_profile_collect", "gnn_pdl_enable", "gnn_probe_gather", "gnn_ln_qkv_fwd", "gnn_dot_aggr",
    "gnn_static_workspace_limit", "gnn_gt_attn_fwd_static",
]


class GnnError(RuntimeError):
    pass


class PlanOpts(C.Structure):
    _fields_ = [("warp_max_deg", C.c_int32), ("cta_max_deg", C.c_int32), ("split_chunk", C.c_int32),
                ("build_transpose", C.c_int32), ("build_blocks", C.c_int32)]


_lib = None
_vp, _i32, _i64, _sz, _f = C.c_void_p, C.c_int32, C.c_int64, C.c_size_t, C.c_float


def lib() -> C.CDLL:
    """Load libgnn_attn.so (built in-tree by paper_2605_31500_b200.build).  Fails loudly if missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise GnnError(f"{_LIB_PATH} is missing: run `python -m paper_2605_31500_b200.build` "
                           "(there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        L.gnn_csr_validate.argtypes = [_i32, _i64, _vp, _vp, _vp, _vp]
        L.gnn_plan_bytes.argtypes = [_i32, _i64, C.POINTER(PlanOpts), C.POINTER(_sz), C.POINTER(_sz)]
        L.gnn_plan_build.argtypes = [C.POINTER(_vp), _vp, _sz, _vp, _sz, _i32, _i64, _vp, _vp, C.POINTER(PlanOpts), _vp]
        L.gnn_plan_destroy.argtypes = [_vp]
        L.gnn_plan_destroy.restype = None
        L.gnn_plan_export.argtypes = [_vp, C.c_int, _vp, C.POINTER(_sz)]
        L.gnn_plan_rowptr_t.argtypes = [_vp]
        L.gnn_plan_rowptr_t.restype = _vp
        L.gnn_plan_colidx_t.argtypes = [_vp]
        L.gnn_plan_colidx_t.restype = _vp
        L.gnn_workspace_bytes.argtypes = [_vp, C.c_int, _i32, _i32, C.c_int, C.POINTER(_sz)]
        L.gnn_gt_attn_fwd.argtypes = [_vp, _vp, _vp, _i32, _vp, _vp, _vp, _i32, _i32, C.c_int, _vp, _vp, _vp, _sz, _vp]
        L.gnn_gt_attn_bwd.argtypes = [_vp, _vp, _vp, _i32, _vp, _vp, _vp, _vp, _vp, _i32, _i32, C.c_int,
                                      _vp, _vp, _vp, _vp, _vp, _sz, _vp]
        L.gnn_gatv2_fwd.argtypes = [_vp, _vp, _vp, _i32, _vp, _vp, _vp, _i32, _i32, C.c_int, _f, _vp, _vp, _vp, _sz, _vp]
        L.gnn_gatv2_bwd.argtypes = [_vp, _vp, _vp, _i32, _vp, _vp, _vp, _vp, _vp, _i32, _i32, C.c_int, _f,
                                    _vp, _vp, _vp, _vp, _vp, _sz, _vp]
        L.gnn_seg_minmax_fwd.argtypes = [_vp, _vp, _vp, _i32, _vp, _i32, C.c_int, _i32, _vp, _vp, _vp, _sz, _vp]
        L.gnn_seg_minmax_bwd.argtypes = [_i32, _vp, _vp, _i32, C.c_int, _vp, _vp]
        L.gnn_gt_attn_fwd_block.argtypes = [_vp, _vp, _vp, _i32, _vp, _vp, _vp, _i32, _i32, C.c_int, _vp, _vp, _vp]
        L.gnn_gt_attn_bwd_block.argtypes = [_vp, _vp, _vp, _i32, _vp, _vp, _vp, _vp, _vp, _i32, _i32, C.c_int,
                                            _vp, _vp, _vp, _vp, _vp, _sz, _vp]
        L.gnn_gt_attn_fwd_wsb.argtypes = [_vp, _vp, _vp, _i32, _vp, _vp, _vp, _i32, _i32, C.c_int, _vp, _vp, _vp]
        L.gnn_gt_attn_bwd_wsb.argtypes = [_vp, _vp, _vp, _i32, _vp, _vp, _vp, _vp, _vp, _vp, _i32, _i32, C.c_int,
                                          _vp, _vp, _vp, _vp, _vp]
        L.gnn_last_error.restype = C.c_char_p
        L.gnn_version.restype = C.c_char_p
        L.gnn_launch_count.restype = _i64
        L.gnn_profile_enable.argtypes = [C.c_int]
        L.gnn_profile_enable.restype = None
        L.gnn_probe_gather.argtypes = [_vp, _i64, _i32, _vp, _i64, _i32, _i32, _i32, _vp, _vp]
        L.gnn_ln_qkv_fwd.argtypes = [_i32, _i32, _i32, _i32, _vp, _vp, _vp, _f, _vp, _vp, _vp, _vp, _vp, _vp]
        L.gnn_dot_aggr.argtypes = [_i32, _vp, _vp, _vp, _i32, _i32, _i32, _vp, _vp]
        L.gnn_static_workspace_limit.restype = _sz
        L.gnn_gt_attn_fwd_static.argtypes = [_vp, _vp, _vp, _i32, _vp, _vp, _vp, _i32, _i32, C.c_int, _vp, _vp, _vp]
        L.gnn_pdl_enable.argtypes = [C.c_int]
        L.gnn_pdl_enable.restype = None
        L.gnn_profile_collect.argtypes = [_vp, _vp, _i32]
        L.gnn_profile_collect.restype = _i32
        for s in EXPORTED_SYMBOLS:
            getattr(L, s)
        _lib = L
    return _lib


def gnn_last_error() -> str:
    return lib().gnn_last_error().decode()


def gnn_version() -> str:
    return lib().gnn_version().decode()


def gnn_launch_count() -> int:
    return int(lib().gnn_launch_count())


def gnn_profile_enable(on: bool) -> None:
    lib().gnn_profile_enable(1 if on else 0)


def gnn_pdl_enable(on: bool) -> None:
    lib().gnn_pdl_enable(1 if on else 0)


def gnn_profile_collect(max_records: int = 4096):
    """[(name, ms), ...] for every launch since the last collect (synchronises)."""
    names = C.create_string_buffer(48 * max_records)
    ms = (C.c_float * max_records)()
    k = lib().gnn_profile_collect(C.cast(names, _vp), C.cast(ms, _vp), max_records)
    return [(names.raw[48 * i:48 * (i + 1)].split(b"\0", 1)[0].decode(), float(ms[i])) for i in range(k)]


def _check(rc: int):
    if rc != GNN_OK:
        raise GnnError(f"gnn status {rc}: {gnn_last_error()}")


def _require_cuda():
    import torch
    if not torch.cuda.is_available():
        raise GnnError("no CUDA device: paper_2605_31500_b200 has no CPU fallback")
    return torch


def _ptr(t):
    """Raw device pointer of a contiguous CUDA tensor (None -> NULL)."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise GnnError("expected a contiguous CUDA tensor")
    return t.data_ptr()


def _stream(stream=None):
    torch = _require_cuda()
    s = torch.cuda.current_stream() if stream is None else stream
    return s.cuda_stream


def _dtype_code(t) -> int:
    import torch
    if t.dtype == torch.float32:
        return GNN_F32
    if t.dtype == torch.bfloat16:
        return GNN_BF16
    raise GnnError(f"unsupported feature dtype {t.dtype}")


# ------------------------------------------------------------------------------------ plan
def gnn_plan_bytes(n: int, nnz: int, opts: PlanOpts):
    _require_cuda()
    d, s = _sz(0), _sz(0)
    _check(lib().gnn_plan_bytes(n, nnz, C.byref(opts), C.byref(d), C.byref(s)))
    return d.value, s.value


def gnn_plan_build(dev_mem, scratch, n: int, nnz: int, rowptr, colidx, opts: PlanOpts, stream=None):
    h = _vp(None)
    _check(lib().gnn_plan_build(C.byref(h), _ptr(dev_mem), dev_mem.numel(), _ptr(scratch), scratch.numel(), n, nnz,
                                _ptr(rowptr), _ptr(colidx), C.byref(opts), _stream(stream)))
    return h


def gnn_csr_validate(rowptr, colidx, stream=None):
    """Raises GnnError unless (rowptr, colidx) is a well-formed int32 CSR with sources in [0, n) (device tensors)."""
    torch = _require_cuda()
    scratch = torch.empty(16, dtype=torch.uint8, device=rowptr.device)
    _check(lib().gnn_csr_validate(int(rowptr.numel()) - 1, int(colidx.numel()), _ptr(rowptr), _ptr(colidx), _ptr(scratch),
                                  _stream(stream)))


def gnn_plan_destroy(handle):
    lib().gnn_plan_destroy(handle)


def gnn_plan_export(handle, what: int, dtype=np.int32) -> np.ndarray:
    need = _sz(0)
    _check(lib().gnn_plan_export(handle, what, None, C.byref(need)))
    out = np.empty(need.value // np.dtype(dtype).itemsize, dtype=dtype)
    cap = _sz(out.nbytes)
    _check(lib().gnn_plan_export(handle, what, out.ctypes.data_as(_vp), C.byref(cap)))
    return out


def gnn_workspace_bytes(handle, op: int, heads: int, head_dim: int, dtype_code: int) -> int:
    b = _sz(0)
    _check(lib().gnn_workspace_bytes(handle, op, heads, head_dim, dtype_code, C.byref(b)))
    return b.value


class Plan:
    """Owns the torch allocations behind a gnn_plan_t (plan storage, workspace) for one CSR graph."""

    def __init__(self, rowptr, colidx, warp_max_deg=0, cta_max_deg=0, split_chunk=0, transpose=True, blocks=False,
                 wsb=False, stream=None):
        torch = _require_cuda()
        if rowptr.dtype != torch.int32 or colidx.dtype != torch.int32:
            raise GnnError("rowptr / colidx must be int32")
        self.rowptr, self.colidx = rowptr.contiguous(), colidx.contiguous()
        self.n, self.nnz = int(rowptr.numel()) - 1, int(colidx.numel())
        # transpose: False (forward only), True (build CSR^T) or "undirected" (the backward reuses
        # the forward CSR; the library verifies the graph is undirected and raises GnnError if not)
        mode = GNN_TRANSPOSE_UNDIRECTED if transpose == "undirected" else (GNN_TRANSPOSE_BUILD if transpose else GNN_TRANSPOSE_NONE)
        # blocks: the diagonal 16-row block layout (gnn_gt_attn_fwd_block); wsb: the general WSB layout
        self.opts = PlanOpts(warp_max_deg, cta_max_deg, split_chunk, mode,
                             (GNN_BLOCKS_DIAG if blocks else 0) | (GNN_BLOCKS_WSB if wsb else 0))
        dev_bytes, scratch_bytes = gnn_plan_bytes(self.n, self.nnz, self.opts)
        self.dev_mem = torch.empty(dev_bytes, dtype=torch.uint8, device=rowptr.device)
        scratch = torch.empty(scratch_bytes, dtype=torch.uint8, device=rowptr.device)
        self.handle = gnn_plan_build(self.dev_mem, scratch, self.n, self.nnz, self.rowptr, self.colidx, self.opts, stream)
        del scratch
        self._ws = None
        self.plan_bytes = dev_bytes

    def export(self, what: int, dtype=np.int32) -> np.ndarray:
        return gnn_plan_export(self.handle, what, dtype)

    def counts(self) -> dict:
        c = self.export(GNN_PLAN_COUNTS)
        keys = ["n_hub", "n_cta", "n_group", "n_chunks"]
        return {**{k: int(v) for k, v in zip(keys, c[:4])}, **{k + "_t": int(v) for k, v in zip(keys, c[4:])}}

    def wsb_info(self) -> dict:
        v = self.export(GNN_PLAN_WSB_INFO)
        return dict(zip(("has_wsb", "n_windows", "n_tcb", "n_dup", "n_tcb_t", "n_dup_t"), (int(x) for x in v)))

    def rows_sorted(self) -> bool:
        """True if every CSR row lists its sources in ascending order (selects the min / max fast path)."""
        return bool(self.export(GNN_PLAN_FLAGS)[0])

    def undirected(self) -> bool:
        """True if the backward traverses the forward CSR (plan built with transpose="undirected")."""
        return bool(self.export(GNN_PLAN_FLAGS)[1])

    def workspace(self, op: int, heads: int, head_dim: int, dtype_code: int):
        import torch
        need = gnn_workspace_bytes(self.handle, op, heads, head_dim, dtype_code)
        if self._ws is None or self._ws.numel() < need:
            self._ws = torch.empty(need, dtype=torch.uint8, device=self.rowptr.device)
        return self._ws

    def __del__(self):
        h = getattr(self, "handle", None)
        if h is not None and _lib is not None:
            _lib.gnn_plan_destroy(h)
            self.handle = None


# ------------------------------------------------------------------------------------ compute
def gnn_gt_attn_fwd(plan: Plan, q, k, v, out, lse, stream=None):
    n, H, d = q.shape
    ws = plan.workspace(GNN_OP_GT_FWD, H, d, _dtype_code(q))
    _check(lib().gnn_gt_attn_fwd(plan.handle, _ptr(plan.rowptr), _ptr(plan.colidx), n, _ptr(q), _ptr(k), _ptr(v), H, d,
                                 _dtype_code(q), _ptr(out), _ptr(lse), _ptr(ws), ws.numel(), _stream(stream)))


def gnn_static_workspace_limit() -> int:
    return int(lib().gnn_static_workspace_limit())


def gnn_gt_attn_fwd_static(plan: Plan, q, k, v, out, lse, stream=None):
    """gnn_gt_attn_fwd with the scratch in the library's built-in device array: no workspace tensor, no allocation."""
    n, H, d = q.shape
    _check(lib().gnn_gt_attn_fwd_static(plan.handle, _ptr(plan.rowptr), _ptr(plan.colidx), n, _ptr(q), _ptr(k), _ptr(v), H, d,
                                        _dtype_code(q), _ptr(out), _ptr(lse), _stream(stream)))


def gnn_gt_attn_fwd_block(plan: Plan, q, k, v, out, lse, stream=None):
    n, H, d = q.shape
    _check(lib().gnn_gt_attn_fwd_block(plan.handle, _ptr(plan.rowptr), _ptr(plan.colidx), n, _ptr(q), _ptr(k), _ptr(v), H, d,
                                       _dtype_code(q), _ptr(out), _ptr(lse), _stream(stream)))


def gnn_gt_attn_bwd_block(plan: Plan, q, k, v, lse, dout, delta, dq, dk, dv, stream=None):
    n, H, d = q.shape
    ws = plan.workspace(GNN_OP_GT_BWD_BLOCK, H, d, _dtype_code(q))
    _check(lib().gnn_gt_attn_bwd_block(plan.handle, _ptr(plan.rowptr), _ptr(plan.colidx), n, _ptr(q), _ptr(k), _ptr(v),
                                       _ptr(lse), _ptr(dout), H, d, _dtype_code(q), _ptr(delta), _ptr(dq), _ptr(dk), _ptr(dv),
                                       _ptr(ws), ws.numel(), _stream(stream)))


def gnn_gt_attn_fwd_wsb(plan: Plan, q, k, v, out, lse, stream=None):
    n, H, d = q.shape
    _check(lib().gnn_gt_attn_fwd_wsb(plan.handle, _ptr(plan.rowptr), _ptr(plan.colidx), n, _ptr(q), _ptr(k), _ptr(v), H, d,
                                     _dtype_code(q), _ptr(out), _ptr(lse), _stream(stream)))


def gnn_gt_attn_bwd_wsb(plan: Plan, q, k, v, out, lse, dout, delta, dq, dk, dv, stream=None):
    n, H, d = q.shape
    _check(lib().gnn_gt_attn_bwd_wsb(plan.handle, _ptr(plan.rowptr), _ptr(plan.colidx), n, _ptr(q), _ptr(k), _ptr(v),
                                     _ptr(out), _ptr(lse), _ptr(dout), H, d, _dtype_code(q), _ptr(delta), _ptr(dq), _ptr(dk),
                                     _ptr(dv), _stream(stream)))


def gnn_gt_attn_bwd(plan: Plan, q, k, v, lse, dout, delta, dq, dk, dv, stream=None):
    n, H, d = q.shape
    ws = plan.workspace(GNN_OP_GT_BWD, H, d, _dtype_code(q))
    _check(lib().gnn_gt_attn_bwd(plan.handle, _ptr(plan.rowptr), _ptr(plan.colidx), n, _ptr(q), _ptr(k), _ptr(v),
                                 _ptr(lse), _ptr(dout), H, d, _dtype_code(q), _ptr(delta), _ptr(dq), _ptr(dk), _ptr(dv),
                                 _ptr(ws), ws.numel(), _stream(stream)))


def gnn_gatv2_fwd(plan: Plan, xl, xr, a, slope, out, lse, stream=None):
    n, H, d = xl.shape
    ws = plan.workspace(GNN_OP_GATV2_FWD, H, d, _dtype_code(xl))
    _check(lib().gnn_gatv2_fwd(plan.handle, _ptr(plan.rowptr), _ptr(plan.colidx), n, _ptr(xl), _ptr(xr), _ptr(a), H, d,
                               _dtype_code(xl), float(slope), _ptr(out), _ptr(lse), _ptr(ws), ws.numel(), _stream(stream)))


def gnn_gatv2_bwd(plan: Plan, xl, xr, a, lse, dout, slope, g, dxl, dxr, da, stream=None):
    n, H, d = xl.shape
    ws = plan.workspace(GNN_OP_GATV2_BWD, H, d, _dtype_code(xl))
    _check(lib().gnn_gatv2_bwd(plan.handle, _ptr(plan.rowptr), _ptr(plan.colidx), n, _ptr(xl), _ptr(xr), _ptr(a),
                               _ptr(lse), _ptr(dout), H, d, _dtype_code(xl), float(slope), _ptr(g), _ptr(dxl), _ptr(dxr),
                               _ptr(da), _ptr(ws), ws.numel(), _stream(stream)))


def gnn_ln_qkv_fwd(x, gamma, beta, eps, w, bias, q, k, v, stream=None):
    """x [n, C] bf16; gamma, beta [C] fp32; w [3*H*d, C] bf16; bias [3*H*d] fp32 or None; q, k, v [n, H, d] bf16 out."""
    n, c_in = x.shape
    _, H, d = q.shape
    _check(lib().gnn_ln_qkv_fwd(n, c_in, H, d, _ptr(x), _ptr(gamma), _ptr(beta), float(eps), _ptr(w), _ptr(bias), _ptr(q),
                                _ptr(k), _ptr(v), _stream(stream)))


def gnn_dot_aggr(rowptr, colidx, x, mode: int, vec: bool, out, stream=None):
    """out[i] = sum_j <x_i, x_j> over the CSR row of i; mode 0 feature-parallel, 1 neighbour-parallel."""
    n, dim = x.shape
    _check(lib().gnn_dot_aggr(n, _ptr(rowptr), _ptr(colidx), _ptr(x), dim, int(mode), 1 if vec else 0, _ptr(out), _stream(stream)))


def gnn_probe_gather(table, row_bytes: int, idx, mode: int, depth: int, ctas_per_sm: int, sink, stream=None):
    """One launch gathering idx.numel() random rows of `row_bytes` from `table` (uint8 [rows * row_bytes]); time it
    with CUDA events on the stream.  mode 0: 256-bit register gathers; mode 1: cp.async.bulk ring."""
    _check(lib().gnn_probe_gather(_ptr(table), table.numel() // row_bytes, row_bytes, _ptr(idx), idx.numel(), mode, depth,
                                  ctas_per_sm, _ptr(sink), _stream(stream)))


def gnn_seg_minmax_fwd(plan: Plan, x, mode, out, arg, stream=None):
    """x, out: [n, channels] (fp32 / bf16); arg: [n, channels] int32; mode: GNN_AGG_MIN | GNN_AGG_MAX."""
    n, ch = x.shape
    ws = plan.workspace(GNN_OP_SEG_MINMAX_FWD, 1, ch, _dtype_code(x))
    _check(lib().gnn_seg_minmax_fwd(plan.handle, _ptr(plan.rowptr), _ptr(plan.colidx), n, _ptr(x), ch, _dtype_code(x),
                                    int(mode), _ptr(out), _ptr(arg), _ptr(ws), ws.numel(), _stream(stream)))


def gnn_seg_minmax_bwd(arg, dout, dx, stream=None):
    """arg: [n, channels] int32 from the forward; dout: [n, channels] (fp32 / bf16); dx: [n, channels] fp32, out."""
    n, ch = arg.shape
    _check(lib().gnn_seg_minmax_bwd(n, _ptr(arg), _ptr(dout), ch, _dtype_code(dout), _ptr(dx), _stream(stream)))
