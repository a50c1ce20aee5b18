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
f2 - general WSB layout ("WSB format and TCB construction", storage PAPER.md:573): destination rows are cut
     into row windows of R = 16; for each window the UNIQUE source columns of all its edges are sorted ascending and
     split into Tensor Core Blocks (TCBs) of width W = 8; a TCB stores its 8 global column indices (padded with zeros
     if fewer than 8) and a 128-bit bitmap of which of its 16 x 8 edges exist; tcb_row_offset maps each row window to
     its contiguous range of TCBs.  Bitmap layout here: 16 bytes per TCB, byte r = row r of the window, bit c = column
     c of the TCB (read as two little-endian 64-bit words: word 0 = rows 0-7, word 1 = rows 8-15).  A bitmap cannot
     say that an entry occurs twice: n_dup counts the CSR entries beyond the first of each (dst, src) pair (0 for a
     simple graph; the CUDA WSB entry points refuse plans with n_dup > 0).
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


def build_wsb(rowptr, colidx) -> dict:
    """f2: the paper's WSB layout for the attention path (no weight tiles)."""
    rowptr = np.asarray(rowptr, dtype=np.int64)
    colidx = np.asarray(colidx, dtype=np.int64)
    n = rowptr.size - 1
    nw = (n + 15) // 16
    row_of_edge = np.repeat(np.arange(n, dtype=np.int64), np.diff(rowptr))
    win = row_of_edge // 16
    # unique (window, column) pairs in (window, column) order = per window the sorted unique columns
    pair = np.unique(win * n + colidx) if colidx.size else np.zeros(0, np.int64)
    uwin, ucol = pair // max(n, 1), pair % max(n, 1)
    ucount = np.bincount(uwin, minlength=nw) if pair.size else np.zeros(nw, np.int64)
    ntcb = (ucount + 7) // 8
    tcb_row_offset = np.zeros(nw + 1, dtype=np.int64)
    np.cumsum(ntcb, out=tcb_row_offset[1:])
    total = int(tcb_row_offset[-1])
    ustart = np.zeros(nw + 1, dtype=np.int64)
    np.cumsum(ucount, out=ustart[1:])
    pos = np.arange(pair.size, dtype=np.int64) - ustart[uwin]          # rank of the column inside its window
    cols = np.zeros(total * 8, dtype=np.int32)                          # padded with zeros
    cols[tcb_row_offset[uwin] * 8 + pos] = ucol
    # bitmap: one bit per distinct (dst, src) pair
    bitmap = np.zeros(total * 16, dtype=np.uint8)
    epos = np.searchsorted(pair, win * n + colidx) - ustart[win] if colidx.size else np.zeros(0, np.int64)
    byte = (tcb_row_offset[win] + epos // 8) * 16 + (row_of_edge % 16)
    np.bitwise_or.at(bitmap, byte, (np.uint8(1) << (epos % 8).astype(np.uint8)))
    nbits = int(np.unpackbits(bitmap).sum())
    return dict(n_windows=nw, n_tcb=total, tcb_row_offset=tcb_row_offset.astype(np.int32), tcb_cols=cols.reshape(total, 8),
                tcb_bitmap=bitmap.reshape(total, 16), n_dup=int(colidx.size) - nbits)
