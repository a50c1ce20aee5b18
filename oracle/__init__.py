"""fp64 CPU ORACLE for the fused graph-attention hot path (GT + GATv2, fwd + bwd).

TEST INFRASTRUCTURE ONLY.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It shares no code with
``paper_2605_31500_b200`` (the CUDA path) and neither imports the other.

* ``gnn_oracle.c``  - the layer definitions of PAPER.md section 2.2 (lines 68-76) and the backward
  identities of PAPER.md:494 / :496 / :539 / :563 written out in plain C, all arithmetic in
  double, OpenMP over rows.  Built by ``oracle.build()`` with gcc.
* ``agg_ref.py``    - the min / max neighbourhood aggregation with argmin (SURVEY 8 row
  f3) written as its definition in numpy, and its scatter-add backward.
* ``plan_ref.py``   - numpy reference for the integer metadata (degree bins + hub chunk
  table, transposed CSR, 16-row block layout) that the CUDA plan must reproduce bit-exactly.

Pins (tests/test_oracle_pins.py, all ``-m "not gpu"``): dense brute-force masked attention in
numpy; library SDPA on the complete graph; torch.autograd through the dense formulation;
central finite differences; closed forms (2-node softmax, slope = 1 => dxl = 0); invariants
(alpha sums to 1, degree-1 row, constant scores => mean, neighbour-order invariance, key shift,
conservation identities); golden fixtures under tests/golden/.  No function is unpinned.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gnn_oracle.c")
_SO = {np.dtype(np.float32): os.path.join(_HERE, "libgnn_oracle.so"),
       np.dtype(np.float64): os.path.join(_HERE, "libgnn_oracle_f64in.so")}
_CT = {np.dtype(np.float32): "float", np.dtype(np.float64): "double"}
_libs = {}


def build(force: bool = False) -> list:
    """Compile the C oracle with gcc (-O2, OpenMP, no fast-math: fp64 semantics stay IEEE).
    Two builds of the same source: float inputs (the stored values) and double inputs (used only
    by the finite-difference pins)."""
    for dt, so in _SO.items():
        if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
            subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11",
                                   f"-DORACLE_IN_T={_CT[dt]}", "-o", so, _SRC, "-lm"])
    return list(_SO.values())


def lib(dtype=np.float32) -> ctypes.CDLL:
    dt = np.dtype(dtype)
    if dt not in _libs:
        build()
        _libs[dt] = ctypes.CDLL(_SO[dt])
        _libs[dt].oracle_num_threads.restype = ctypes.c_int
    return _libs[dt]


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(t: int) -> None:
    lib().oracle_set_num_threads(ctypes.c_int(int(t)))


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ct))


def _feats(*xs):
    """Contiguous feature arrays, all float32 (default) or all float64 (finite-difference pins)."""
    dt = np.float64 if all(np.asarray(x).dtype == np.float64 for x in xs) else np.float32
    return [np.ascontiguousarray(x, dtype=dt) for x in xs]


def _i32(x):
    return None if x is None else np.ascontiguousarray(x, dtype=np.int32)


def _f64(x):
    return np.ascontiguousarray(x, dtype=np.float64)


I32, F32, F64 = ctypes.c_int32, ctypes.c_float, ctypes.c_double


def _fp(x):
    """ctypes pointer to a feature array in its own dtype (float32 or float64)."""
    return x.ctypes.data_as(ctypes.POINTER(F64 if x.dtype == np.float64 else F32))


# ------------------------------------------------------------------------------ forward
def gt_forward(rowptr, colidx, q, k, v, rows=None):
    """GT forward.  Returns (O [R,H,d] f64, L [R,H] f64), R = len(rows) or N."""
    q, k, v = _feats(q, k, v)
    n, H, d = q.shape
    rowptr, colidx, rows = _i32(rowptr), _i32(colidx), _i32(rows)
    R = n if rows is None else rows.size
    O = np.empty((R, H, d), np.float64)
    L = np.empty((R, H), np.float64)
    lib(q.dtype).oracle_gt_fwd(I32(n), _p(rowptr, I32), _p(colidx, I32), _fp(q), _fp(k), _fp(v), I32(H), I32(d),
                               _p(rows, I32), I32(R), _p(O, F64), _p(L, F64))
    return O, L


def gatv2_forward(rowptr, colidx, xl, xr, a, slope, rows=None):
    """GATv2 forward.  Returns (O [R,H,d] f64, L [R,H] f64)."""
    xl, xr, a = _feats(xl, xr, a)
    n, H, d = xl.shape
    assert a.shape == (H, d)
    rowptr, colidx, rows = _i32(rowptr), _i32(colidx), _i32(rows)
    R = n if rows is None else rows.size
    O = np.empty((R, H, d), np.float64)
    L = np.empty((R, H), np.float64)
    lib(xl.dtype).oracle_gatv2_fwd(I32(n), _p(rowptr, I32), _p(colidx, I32), _fp(xl), _fp(xr), _fp(a),
                                   F64(slope), I32(H), I32(d), _p(rows, I32), I32(R), _p(O, F64), _p(L, F64))
    return O, L


def rowdot(O, dO, rows=None):
    """Delta (GT) or G (GATv2): <O[t], dO[rows[t]]> per head."""
    O = _f64(O)
    (dO,) = _feats(dO)
    R, H, d = O.shape
    rows = _i32(rows)
    out = np.empty((R, H), np.float64)
    lib(dO.dtype).oracle_rowdot(_p(O, F64), _fp(dO), I32(H), I32(d), _p(rows, I32), I32(R), _p(out, F64))
    return out


# ------------------------------------------------------------------------------ GT backward
def gt_backward_dst(rowptr, colidx, q, k, v, dO, L_full, Delta_full, rows=None):
    q, k, v, dO = _feats(q, k, v, dO)
    n, H, d = q.shape
    rowptr, colidx, rows = _i32(rowptr), _i32(colidx), _i32(rows)
    L_full, Delta_full = _f64(L_full), _f64(Delta_full)
    assert L_full.shape == (n, H) and Delta_full.shape == (n, H)
    R = n if rows is None else rows.size
    dQ = np.empty((R, H, d), np.float64)
    lib(q.dtype).oracle_gt_bwd_dst(I32(n), _p(rowptr, I32), _p(colidx, I32), _fp(q), _fp(k), _fp(v), _fp(dO),
                                   _p(L_full, F64), _p(Delta_full, F64), I32(H), I32(d), _p(rows, I32), I32(R),
                                   _p(dQ, F64))
    return dQ


def gt_backward_src(rowptr_t, colidx_t, q, k, v, dO, L_full, Delta_full, srcs=None):
    q, k, v, dO = _feats(q, k, v, dO)
    n, H, d = q.shape
    rowptr_t, colidx_t, srcs = _i32(rowptr_t), _i32(colidx_t), _i32(srcs)
    L_full, Delta_full = _f64(L_full), _f64(Delta_full)
    assert L_full.shape == (n, H) and Delta_full.shape == (n, H)
    R = n if srcs is None else srcs.size
    dK = np.empty((R, H, d), np.float64)
    dV = np.empty((R, H, d), np.float64)
    lib(q.dtype).oracle_gt_bwd_src(I32(n), _p(rowptr_t, I32), _p(colidx_t, I32), _fp(q), _fp(k), _fp(v), _fp(dO),
                                   _p(L_full, F64), _p(Delta_full, F64), I32(H), I32(d), _p(srcs, I32), I32(R),
                                   _p(dK, F64), _p(dV, F64))
    return dK, dV


def gt_backward(rowptr, colidx, q, k, v, dO):
    """Full GT forward + backward.  Returns dict(O, L, Delta, dQ, dK, dV), all f64."""
    from .plan_ref import transpose_csr
    O, L = gt_forward(rowptr, colidx, q, k, v)
    Delta = rowdot(O, dO)
    dQ = gt_backward_dst(rowptr, colidx, q, k, v, dO, L, Delta)
    rp_t, ci_t = transpose_csr(rowptr, colidx)
    dK, dV = gt_backward_src(rp_t, ci_t, q, k, v, dO, L, Delta)
    return dict(O=O, L=L, Delta=Delta, dQ=dQ, dK=dK, dV=dV)


# ------------------------------------------------------------------------------ GATv2 backward
def gatv2_backward_dst(rowptr, colidx, xl, xr, a, slope, dO, L_full, G_full, rows=None):
    """Returns (dxl [R,H,d], da_rows [R,H,d]); da = da_rows.sum(0) when rows covers all rows."""
    xl, xr, a, dO = _feats(xl, xr, a, dO)
    n, H, d = xl.shape
    rowptr, colidx, rows = _i32(rowptr), _i32(colidx), _i32(rows)
    L_full, G_full = _f64(L_full), _f64(G_full)
    R = n if rows is None else rows.size
    dxl = np.empty((R, H, d), np.float64)
    da_rows = np.empty((R, H, d), np.float64)
    lib(xl.dtype).oracle_gatv2_bwd_dst(I32(n), _p(rowptr, I32), _p(colidx, I32), _fp(xl), _fp(xr), _fp(a),
                                       F64(slope), _fp(dO), _p(L_full, F64), _p(G_full, F64), I32(H), I32(d),
                                       _p(rows, I32), I32(R), _p(dxl, F64), _p(da_rows, F64))
    return dxl, da_rows


def gatv2_backward_src(rowptr_t, colidx_t, xl, xr, a, slope, dO, L_full, G_full, srcs=None):
    xl, xr, a, dO = _feats(xl, xr, a, dO)
    n, H, d = xl.shape
    rowptr_t, colidx_t, srcs = _i32(rowptr_t), _i32(colidx_t), _i32(srcs)
    L_full, G_full = _f64(L_full), _f64(G_full)
    R = n if srcs is None else srcs.size
    dxr = np.empty((R, H, d), np.float64)
    lib(xl.dtype).oracle_gatv2_bwd_src(I32(n), _p(rowptr_t, I32), _p(colidx_t, I32), _fp(xl), _fp(xr), _fp(a),
                                       F64(slope), _fp(dO), _p(L_full, F64), _p(G_full, F64), I32(H), I32(d),
                                       _p(srcs, I32), I32(R), _p(dxr, F64))
    return dxr


def gatv2_backward(rowptr, colidx, xl, xr, a, slope, dO):
    """Full GATv2 forward + backward.  Returns dict(O, L, G, dxl, dxr, da), all f64."""
    from .plan_ref import transpose_csr
    O, L = gatv2_forward(rowptr, colidx, xl, xr, a, slope)
    G = rowdot(O, dO)
    dxl, da_rows = gatv2_backward_dst(rowptr, colidx, xl, xr, a, slope, dO, L, G)
    rp_t, ci_t = transpose_csr(rowptr, colidx)
    dxr = gatv2_backward_src(rp_t, ci_t, xl, xr, a, slope, dO, L, G)
    return dict(O=O, L=L, G=G, dxl=dxl, dxr=dxr, da=da_rows.sum(axis=0))


def scatter_full(n, rows, vals):
    """Place sampled per-row values into a full [n, ...] array (NaN elsewhere)."""
    full = np.full((n,) + vals.shape[1:], np.nan, np.float64)
    full[np.asarray(rows)] = vals
    return full
