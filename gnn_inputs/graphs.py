"""Seeded synthetic graph generators -> int32 CSR (row = destination, entries = sources).

Every generator ends in ``csr_from_pairs``: drop self-pairs, dedupe, add exactly one
self-loop per node (the softmax runs over N(i) U {i}; the caller stores the
self-loop, reading A3), sort by (dst, src).  Nothing here is part of the method:
no plan, no binning, no transposition.
"""
from __future__ import annotations

import numpy as np


def _sorted_unique(key: np.ndarray) -> np.ndarray:
    """np.unique(key) for int64 keys via sort + neighbour compare (numpy 2.3's np.unique is ~100x slower here)."""
    if key.size == 0:
        return key
    k = np.sort(key)
    keep = np.empty(k.size, dtype=bool)
    keep[0] = True
    np.not_equal(k[1:], k[:-1], out=keep[1:])
    return k[keep]


def csr_from_pairs(n: int, dst: np.ndarray, src: np.ndarray, self_loops: bool = True, dedupe: bool = True):
    """(dst, src) pairs -> (rowptr int32 [n+1], colidx int32 [nnz]) sorted by (dst, src)."""
    dst = np.asarray(dst, dtype=np.int64)
    src = np.asarray(src, dtype=np.int64)
    if self_loops:
        keep = dst != src
        dst, src = dst[keep], src[keep]
        loops = np.arange(n, dtype=np.int64)
        dst = np.concatenate([dst, loops])
        src = np.concatenate([src, loops])
    key = (dst << np.int64(32)) | src
    if dedupe:
        key = _sorted_unique(key)
    else:
        key = np.sort(key, kind="stable")
    assert key.size < 2**31, "nnz must fit int32"
    d = (key >> np.int64(32)).astype(np.int64)
    colidx = (key & np.int64(0xFFFFFFFF)).astype(np.int32)
    counts = np.bincount(d, minlength=n)
    rowptr = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(counts, out=rowptr[1:])
    return rowptr.astype(np.int32), colidx


def erdos_renyi(n: int, avg_in_deg: float, rng: np.random.Generator):
    """Directed G(n, p): each ordered pair (j -> i), i != j, present with p = avg/(n-1)."""
    p = avg_in_deg / (n - 1)
    if n <= 4096:
        m = rng.random((n, n)) < p
        dst, src = np.nonzero(m)
    else:  # sparse sampling for larger n: binomial number of pairs, uniform endpoints
        cnt = rng.binomial(n * (n - 1), p)
        dst = rng.integers(0, n, size=cnt)
        src = rng.integers(0, n, size=cnt)
    return csr_from_pairs(n, dst, src)


def _chung_lu_weights(n: int, gamma: float, w_max: float, w_sum: float) -> np.ndarray:
    """w_i = c (i + i0)^(-1/(gamma-1)) with w_0 = w_max and sum w = w_sum (bisection on i0)."""
    alpha = 1.0 / (gamma - 1.0)
    i = np.arange(n, dtype=np.float64)

    def total(i0):
        c = w_max * i0 ** alpha
        return c * np.sum((i + i0) ** (-alpha))

    lo, hi = 1e-3, 1e6
    for _ in range(200):
        mid = np.sqrt(lo * hi)
        if total(mid) < w_sum:
            lo = mid
        else:
            hi = mid
    i0 = np.sqrt(lo * hi)
    c = w_max * i0 ** alpha
    return c * (i + i0) ** (-alpha)


def chung_lu(n: int, n_pairs: int, gamma: float, w_max: float, rng: np.random.Generator, rng_relabel):
    """Chung-Lu style power-law in-degrees: dst ~ w / sum(w), src ~ uniform; random relabel."""
    w = _chung_lu_weights(n, gamma, w_max, float(n_pairs))
    cdf = np.cumsum(w)
    cdf /= cdf[-1]
    dst = np.searchsorted(cdf, rng.random(n_pairs), side="right").astype(np.int64)
    np.minimum(dst, n - 1, out=dst)
    src = rng.integers(0, n, size=n_pairs, dtype=np.int64)
    perm = rng_relabel.permutation(n).astype(np.int64)
    return csr_from_pairs(n, perm[dst], perm[src])


def _rmat_pairs(bits: int, m: int, a: float, b: float, c: float, rng: np.random.Generator, chunk: int = 1 << 24):
    """R-MAT in a 2^bits id space; quadrants (a,b,c,d) <-> (src-bit, dst-bit) = (0,0),(0,1),(1,0),(1,1)."""
    src = np.zeros(m, dtype=np.int64)
    dst = np.zeros(m, dtype=np.int64)
    ab, abc = a + b, a + b + c
    for s in range(0, m, chunk):
        e = min(m, s + chunk)
        sv = np.zeros(e - s, dtype=np.int64)
        dv = np.zeros(e - s, dtype=np.int64)
        for _ in range(bits):
            r = rng.random(e - s, dtype=np.float32)
            sbit = r >= ab
            dbit = ((r >= a) & (r < ab)) | (r >= abc)
            sv = (sv << 1) | sbit
            dv = (dv << 1) | dbit
        src[s:e] = sv
        dst[s:e] = dv
    return dst, src


def rmat_symmetric(n: int, bits: int, n_samples: int, abc, rng: np.random.Generator, rng_relabel=None):
    """Symmetrised R-MAT: reject endpoints >= n, add both directions, dedupe, + self-loops."""
    dst, src = _rmat_pairs(bits, n_samples, abc[0], abc[1], abc[2], rng)
    keep = (dst < n) & (src < n)
    dst, src = dst[keep], src[keep]
    if rng_relabel is not None:
        perm = rng_relabel.permutation(n).astype(np.int64)
        dst, src = perm[dst], perm[src]
    return csr_from_pairs(n, np.concatenate([dst, src]), np.concatenate([src, dst]))


def community_graph(n: int, csize: int, p_intra: float, n_long: int, rng: np.random.Generator, rng_long):
    """Communities of ``csize`` consecutive ids (aligned to row windows, no relabel): every
    ordered intra-community pair (j -> i), i != j, with probability p_intra; plus ``n_long``
    distinct uniform sources from outside the community per node."""
    assert n % csize == 0
    nc = n // csize
    # intra-community: a [nc, csize, csize] Bernoulli mask drawn in chunks
    dst_parts, src_parts = [], []
    step = max(1, (1 << 22) // (csize * csize))
    for c0 in range(0, nc, step):
        c1 = min(nc, c0 + step)
        m = rng.random((c1 - c0, csize, csize), dtype=np.float32) < p_intra
        cc, ii, jj = np.nonzero(m)
        base = (cc.astype(np.int64) + c0) * csize
        dst_parts.append(base + ii)
        src_parts.append(base + jj)
    # long-range: n_long draws per node from outside its community (redraw collisions once
    # deterministically by shifting by one community)
    node = np.repeat(np.arange(n, dtype=np.int64), n_long)
    far = rng_long.integers(0, n - csize, size=n * n_long, dtype=np.int64)
    cstart = (node // csize) * csize
    far = np.where(far >= cstart, far + csize, far)  # skip own community: uniform over the rest
    dst_parts.append(node)
    src_parts.append(far)
    return csr_from_pairs(n, np.concatenate(dst_parts), np.concatenate(src_parts))


def rmat_hubs(n: int, bits: int, n_samples: int, abc, hub_degrees, rng, rng_relabel, rng_hub):
    """Directed high-skew R-MAT with planted hubs: the len(hub_degrees) largest-in-degree
    nodes (ties -> smaller id) receive extra distinct uniform sources until their in-degree
    reaches hub_degrees[k]; random relabel; + self-loops.  (Plain R-MAT at these parameters
    does not reach in-degree > 1M after dedupe, SURVEY.md section 8(d) cfg 5.)"""
    dst, src = _rmat_pairs(bits, n_samples, abc[0], abc[1], abc[2], rng)
    keep = (dst < n) & (src < n) & (dst != src)
    key = _sorted_unique((dst[keep] << np.int64(32)) | src[keep])
    dst = key >> np.int64(32)
    src = key & np.int64(0xFFFFFFFF)
    indeg = np.bincount(dst, minlength=n)
    order = np.lexsort((np.arange(n), -indeg))  # degree desc, id asc
    extra_d, extra_s = [], []
    for k, target in enumerate(hub_degrees):
        h = int(order[k])
        target = min(int(target), n - 1)
        have = src[dst == h]
        need = target - have.size
        if need <= 0:
            continue
        mask = np.ones(n, dtype=bool)
        mask[have] = False
        mask[h] = False
        cand = np.nonzero(mask)[0]
        pick = rng_hub.choice(cand, size=need, replace=False)
        extra_d.append(np.full(need, h, dtype=np.int64))
        extra_s.append(pick.astype(np.int64))
    if extra_d:
        dst = np.concatenate([dst] + extra_d)
        src = np.concatenate([src] + extra_s)
    perm = rng_relabel.permutation(n).astype(np.int64)
    return csr_from_pairs(n, perm[dst], perm[src])


def degree_stats(rowptr: np.ndarray, colidx: np.ndarray) -> dict:
    """N, E, max / median / p99 in- and out-degree and in-degree skewness (the statistic the
    paper correlates with its degree-aware win)."""
    n = rowptr.size - 1
    indeg = np.diff(rowptr.astype(np.int64))
    outdeg = np.bincount(colidx, minlength=n)
    mu, sd = indeg.mean(), indeg.std()
    skew = float(((indeg - mu) ** 3).mean() / sd ** 3) if sd > 0 else 0.0
    return {
        "n": int(n),
        "e": int(colidx.size),
        "in_max": int(indeg.max()), "in_median": float(np.median(indeg)), "in_p99": float(np.percentile(indeg, 99)),
        "out_max": int(outdeg.max()), "out_median": float(np.median(outdeg)), "out_p99": float(np.percentile(outdeg, 99)),
        "in_skewness": skew,
    }
