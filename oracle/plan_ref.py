"""numpy reference for the integer plan metadata.

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  The CUDA plan builder must reproduce
every array here bit-exactly; the definitions are stated in include/gnn_attn.h and DESIGN.md
section 3 and restated below.  No code is shared with the CUDA path.

a1 - degree bins (paper: light / heavy split with per-bucket warp counts, PAPER.md:326,
     PAPER.md:456-460, :472; the thresholds here are the build's own):
     deg(i) = rowptr[i+1] - rowptr[i];  bl(x) = bit length of x (bl(0) = 0)
       key(i) = 0                      if deg > cta_max_deg               ("hub": split into chunks)
              = 1  + (32 - bl(deg))    if warp_max_deg < deg <= cta_max_deg  ("CTA rows")
              = 34 + (32 - bl(deg))    otherwise                          ("group rows"; deg 0 -> 66)
     perm = row ids sorted by (key ascending, row id ascending)  (heaviest first; stable)
     hub row r (in perm order) with degree g is cut into c = ceil(g / split_chunk) chunks,
     chunk t = [rowptr[r] + floor(t*g/c), rowptr[r] + floor((t+1)*g/c)); the chunk table lists
     (row, e_begin, e_end, hub_slot) in (hub_slot, t) order; hub_chunk_ptr is its row pointer.
a2 - transposed CSR by a STABLE counting sort on the source id: row j of
     CSR^T lists the destinations i of j's out-edges ordered by (i ascending, original position).
f1 - direction-aware backward: a CSR is "undirected" iff every row is strictly
     ascending and its set of (dst, src) pairs equals its set of (src, dst) pairs; then
     transpose_csr(CSR) == CSR bit for bit, which is why the backward may reuse the forward CSR.
a11 - 16-row block layout for the locally dense graph (own layout; the paper's WSB, PAPER.md:545,
     is prior art): window w = rows [16w, 16w+16); bitmap[w][r] bit c is set iff the FIRST
     occurrence of edge (dst 16w+r <- src 16w+c) exists; every other entry (sources outside
     the window, and duplicate in-window entries) goes to a remainder CSR in original order.
"""
from __future__ import annotations

import numpy as np


def _bit_length(x: np.ndarray) -> np.ndarray:
    x = x.astype(np.int64)
    bl = np.zeros(x.shape, dtype=np.int64)
    v = x.copy()
    while np.any(v > 0):
        bl += (v > 0)
        v >>= 1
    return bl


def degree_keys(rowptr, warp_max_deg: int, cta_max_deg: int) -> np.ndarray:
    deg = np.diff(np.asarray(rowptr, dtype=np.int64))
    bl = _bit_length(deg)
    key = 34 + (32 - bl)
    key = np.where(deg > warp_max_deg, 1 + (32 - bl), key)
    key = np.where(deg > cta_max_deg, 0, key)
    return key.astype(np.int32)


def build_bins(rowptr, warp_max_deg: int, cta_max_deg: int, split_chunk: int) -> dict:
    rowptr = np.asarray(rowptr, dtype=np.int64)
    n = rowptr.size - 1
    key = degree_keys(rowptr, warp_max_deg, cta_max_deg)
    perm = np.argsort(key, kind="stable").astype(np.int32)
    n_hub = int(np.sum(key == 0))
    n_cta = int(np.sum((key >= 1) & (key <= 33)))
    chunks = []
    hub_chunk_ptr = [0]
    for slot in range(n_hub):
        r = int(perm[slot])
        b = int(rowptr[r])
        g = int(rowptr[r + 1]) - b
        c = -(-g // split_chunk)
        for t in range(c):
            chunks.append((r, b + (t * g) // c, b + ((t + 1) * g) // c, slot))
        hub_chunk_ptr.append(len(chunks))
    return dict(
        n=n, n_hub=n_hub, n_cta=n_cta, n_group=n - n_hub - n_cta,
        perm=perm,
        chunks=np.asarray(chunks, dtype=np.int32).reshape(-1, 4),
        hub_chunk_ptr=np.asarray(hub_chunk_ptr, dtype=np.int32),
    )


def transpose_csr(rowptr, colidx):
    rowptr = np.asarray(rowptr, dtype=np.int64)
    colidx = np.asarray(colidx, dtype=np.int64)
    n = rowptr.size - 1
    row_of_edge = np.repeat(np.arange(n, dtype=np.int64), np.diff(rowptr))
    order = np.argsort(colidx, kind="stable")
    colidx_t = row_of_edge[order].astype(np.int32)
    rowptr_t = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(np.bincount(colidx, minlength=n), out=rowptr_t[1:])
    return rowptr_t.astype(np.int32), colidx_t


def is_undirected(rowptr, colidx) -> bool:
    """f1: strictly ascending rows and edge set == mirrored edge set (plain set comparison)."""
    rowptr = np.asarray(rowptr, dtype=np.int64)
    colidx = np.asarray(colidx, dtype=np.int64)
    n = rowptr.size - 1
    if colidx.size and (colidx.min() < 0 or colidx.max() >= n):
        return False
    for i in range(n):
        row = colidx[rowptr[i]:rowptr[i + 1]]
        if np.any(np.diff(row) <= 0):
            return False
    row_of_edge = np.repeat(np.arange(n, dtype=np.int64), np.diff(rowptr))
    fwd = np.sort(row_of_edge * n + colidx)
    rev = np.sort(colidx * n + row_of_edge)
    return bool(np.array_equal(fwd, rev))


def build_blocks(rowptr, colidx) -> dict:
    """a11: per-window 16x16 bitmaps of in-window edges + remainder CSR."""
    rowptr = np.asarray(rowptr, dtype=np.int64)
    colidx = np.asarray(colidx, dtype=np.int64)
    n = rowptr.size - 1
    nw = (n + 15) // 16
    row_of_edge = np.repeat(np.arange(n, dtype=np.int64), np.diff(rowptr))
    in_win = (colidx // 16) == (row_of_edge // 16)
    # first occurrence of each (row, col) among in-window entries
    first = np.zeros(colidx.size, dtype=bool)
    idx = np.nonzero(in_win)[0]
    pair = row_of_edge[idx] * 16 + (colidx[idx] % 16)
    _, first_pos = np.unique(pair, return_index=True)   # first occurrence (idx is ascending)
    first[idx[first_pos]] = True
    bitmap = np.zeros(nw * 16, dtype=np.uint16)
    np.bitwise_or.at(bitmap, row_of_edge[first], (np.uint16(1) << (colidx[first] % 16).astype(np.uint16)))
    rem = ~first
    rem_colidx = colidx[rem].astype(np.int32)
    rem_rowptr = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(np.bincount(row_of_edge[rem], minlength=n), out=rem_rowptr[1:])
    return dict(n_windows=nw, bitmap=bitmap.reshape(nw, 16), rem_rowptr=rem_rowptr.astype(np.int32),
                rem_colidx=rem_colidx)
