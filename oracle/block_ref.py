"""fp64 numpy ORACLE for the rest of the block the paper timed: layer normalisation followed by
the QKV projection in front of the Graph Transformer attention ("our measurements include the full attention
block comprising layer normalization, QKV projection, and the attention mechanism itself"), and the `dot-aggr` locality
micro-benchmark's arithmetic.

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py); shares no code with the CUDA path.  Readings (A21-A23): the
paper states neither the LayerNorm variant nor eps - taken as the standard one over the feature dimension with the
biased variance, eps = 1e-5, elementwise affine (gamma, beta); the projection is x_norm W^T + b with one stacked weight
[3*H*d, C] whose row blocks are W_Q, W_K, W_V; dot-aggr: out[i] = sum over the stored in-neighbours j of i of <x_i, x_j>
(a dot product per edge aggregated at the destination - the one arithmetic both access patterns share).
"""
from __future__ import annotations

import numpy as np


def layer_norm(x, gamma, beta, eps: float = 1e-5) -> np.ndarray:
    """y[i, :] = (x[i, :] - mean_i) / sqrt(var_i + eps) * gamma + beta, var_i the biased variance over the features."""
    x = np.asarray(x, dtype=np.float64)
    mean = x.sum(axis=1, keepdims=True) / x.shape[1]
    cen = x - mean
    var = (cen * cen).sum(axis=1, keepdims=True) / x.shape[1]
    return cen / np.sqrt(var + eps) * np.asarray(gamma, np.float64)[None, :] + np.asarray(beta, np.float64)[None, :]


def ln_qkv(x, gamma, beta, w, bias, heads: int, head_dim: int, eps: float = 1e-5):
    """(Q, K, V), each [n, heads, head_dim] fp64: LayerNorm(x) W^T + bias, W = [W_Q; W_K; W_V] of shape [3*H*d, C]."""
    y = layer_norm(x, gamma, beta, eps)
    w = np.asarray(w, dtype=np.float64)
    r = heads * head_dim
    assert w.shape == (3 * r, y.shape[1])
    out = y @ w.T
    if bias is not None:
        out = out + np.asarray(bias, np.float64)[None, :]
    n = y.shape[0]
    return tuple(out[:, t * r:(t + 1) * r].reshape(n, heads, head_dim) for t in range(3))


def dot_aggr(rowptr, colidx, x) -> np.ndarray:
    """out[i] = sum_{e in row i} <x[i, :], x[colidx[e], :]>  (the dot-aggr micro-benchmark)."""
    x = np.asarray(x, dtype=np.float64)
    rowptr = np.asarray(rowptr, dtype=np.int64)
    colidx = np.asarray(colidx, dtype=np.int64)
    n = rowptr.size - 1
    out = np.zeros(n)
    for i in range(n):
        for e in range(rowptr[i], rowptr[i + 1]):
            out[i] += float(np.dot(x[i], x[colidx[e]]))
    return out
