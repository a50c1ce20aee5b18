"""fp64 CPU ORACLE for the degree-aware min / max aggregation with argmin.

TEST INFRASTRUCTURE ONLY (see ``oracle/__init__.py``): shares no code with the CUDA path.

The operator (section 3.1; App. D.1): for every destination node i and
feature c,

    out[i, c] = min over the stored in-neighbours j of i of x[j, c]          (``mode = "min"``)
    arg[i, c] = the source node that attains it

and the backward pass is a sparse scatter-add through the saved indices:

    dx[arg[i, c], c] += dout[i, c].

Readings where the paper is silent (A20):
* ties: the paper's packed (value, index) atomicMin breaks ties by the smaller source index;
  values are compared as IEEE numbers (-0.0 == +0.0 is a tie) - its order-preserving integer key would put
  -0.0 first; inputs are finite;
* ``mode = "max"``: the maximum, ties again to the smaller source index;
* a row without in-neighbours: out = 0, arg = -1, and it sends no gradient;
* duplicate CSR entries change nothing (min is idempotent).

Written as the definition: a Python loop over rows, numpy over the neighbour axis.  Pins:
``tests/test_oracle_pins.py`` (dense brute force, degree-1 rows, constant features, order invariance,
autograd of the dense formulation, conservation of the gradient mass).
"""
from __future__ import annotations

import numpy as np


def seg_minmax_forward(rowptr, colidx, x, mode: str = "min"):
    """x: [n, C].  Returns (out [n, C] float64, arg [n, C] int32)."""
    assert mode in ("min", "max")
    rowptr = np.asarray(rowptr, np.int64)
    colidx = np.asarray(colidx, np.int64)
    x = np.asarray(x, np.float64)
    n, C = rowptr.size - 1, x.shape[1]
    out = np.zeros((n, C), np.float64)
    arg = np.full((n, C), -1, np.int32)
    for i in range(n):
        nb = np.unique(colidx[rowptr[i]:rowptr[i + 1]])      # ascending source ids, duplicates dropped
        if nb.size == 0:
            continue
        X = x[nb]                                            # [deg, C]
        pos = np.argmin(X, axis=0) if mode == "min" else np.argmax(X, axis=0)   # first hit = smallest source id
        out[i] = X[pos, np.arange(C)]
        arg[i] = nb[pos]
    return out, arg


def seg_minmax_backward(arg, dout, n_src: int):
    """dx[arg[i, c], c] += dout[i, c] for arg >= 0.  Returns dx [n_src, C] float64."""
    arg = np.asarray(arg, np.int64)
    dout = np.asarray(dout, np.float64)
    C = arg.shape[1]
    dx = np.zeros((n_src, C), np.float64)
    sel = arg >= 0
    cols = np.broadcast_to(np.arange(C), arg.shape)
    np.add.at(dx, (arg[sel], cols[sel]), dout[sel])          # unbuffered scatter-add, row-major order of (i, c)
    return dx
