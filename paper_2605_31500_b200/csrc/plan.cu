// plan.cu - integer metadata of the hot path, built on the device (rows a1, a2 of the scope table):
// degree bins + hub chunk table and the transposed CSR by a stable
// sort on the source id.  Pure functions of (rowptr, colidx, opts); the numpy
// reference in oracle/plan_ref.py states the same definitions independently and the tests compare
// bit for bit.  Sorting / scanning uses CUB's stable LSD radix sort (a library primitive, one-time
// preprocessing outside the timed layer, like the paper's format construction).
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>
#include <cub/device/device_select.cuh>

#include <new>

#include "internal.h"

namespace gnn {

namespace {

constexpr size_t kAlign = 256;
inline size_t up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

__device__ __forceinline__ int bit_length(int x) { return 32 - __clz(x); }

// key(i): 0 hub; 1 + (32 - bl(deg)) CTA rows; 34 + (32 - bl(deg)) group rows
__global__ void key_kernel(const int32_t* __restrict__ rowptr, int n, int warp_max, int cta_max,
                           uint32_t* __restrict__ key, int32_t* __restrict__ rowid) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int deg = rowptr[i + 1] - rowptr[i];
    const int bl = bit_length(deg);
    uint32_t k = 34 + (32 - bl);
    if (deg > warp_max) k = 1 + (32 - bl);
    if (deg > cta_max) k = 0;
    key[i] = k;
    rowid[i] = i;
}

__device__ int lower_bound_u32(const uint32_t* a, int n, uint32_t v) {
    int lo = 0, hi = n;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (a[mid] < v) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// counts[0..3] = n_hub, n_cta, n_group, n_chunks; chunk_ptr[0..n_hub]  (single thread: n_hub is small)
__global__ void count_kernel(const uint32_t* __restrict__ key_sorted, const int32_t* __restrict__ perm,
                             const int32_t* __restrict__ rowptr, int n, int split, int32_t* __restrict__ counts,
                             int32_t* __restrict__ chunk_ptr, int max_hub) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const int n_hub = lower_bound_u32(key_sorted, n, 1u);
    const int n_heavy = lower_bound_u32(key_sorted, n, 34u);
    int acc = 0;
    chunk_ptr[0] = 0;
    for (int s = 0; s < n_hub && s < max_hub; ++s) {
        const int r = perm[s];
        const int g = rowptr[r + 1] - rowptr[r];
        acc += (g + split - 1) / split;
        chunk_ptr[s + 1] = acc;
    }
    counts[0] = n_hub;
    counts[1] = n_heavy - n_hub;
    counts[2] = n - n_heavy;
    counts[3] = acc;
}

// one CTA per hub slot: chunk t = [b + floor(t g / c), b + floor((t+1) g / c))
__global__ void chunk_kernel(const int32_t* __restrict__ perm, const int32_t* __restrict__ rowptr,
                             const int32_t* __restrict__ chunk_ptr, int32_t* __restrict__ chunks) {
    const int slot = blockIdx.x;
    const int r = perm[slot];
    const int b = rowptr[r];
    const long long g = rowptr[r + 1] - b;
    const int c0 = chunk_ptr[slot];
    const long long c = chunk_ptr[slot + 1] - c0;
    for (int t = threadIdx.x; t < c; t += blockDim.x) {
        int4 v;
        v.x = r;
        v.y = b + (int)((t * g) / c);
        v.z = b + (int)(((t + 1) * g) / c);
        v.w = slot;
        reinterpret_cast<int4*>(chunks)[c0 + t] = v;
    }
}

__global__ void row_of_edge_kernel(const int32_t* __restrict__ rowptr, int n, long long nnz,
                                   int32_t* __restrict__ row_of_edge) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= nnz) return;
    int lo = 0, hi = n;  // last row with rowptr[row] <= e
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if ((long long)rowptr[mid] <= e) lo = mid; else hi = mid;
    }
    row_of_edge[e] = lo;
}

// flag = 1 if some row lists its sources out of ascending order: a descent colidx[e-1] > colidx[e] is harmless only
// when e starts a row (binary search in rowptr, reached by ~one entry per row on a sorted CSR)
__global__ void rows_unsorted_kernel(const int32_t* __restrict__ rowptr, const int32_t* __restrict__ colidx, int n,
                                     long long nnz, int32_t* __restrict__ flag) {
    const long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x + 1;
    if (e >= nnz || __ldg(colidx + e - 1) <= __ldg(colidx + e)) return;
    int lo = 0, hi = n;
    while (lo < hi) {
        const int mid = (int)(((long long)lo + hi + 1) >> 1);
        if (__ldg(rowptr + mid) <= e) lo = mid; else hi = mid - 1;
    }
    if (__ldg(rowptr + lo) != e) *flag = 1;
}

// Undirected check: flag = 1 unless every row is STRICTLY ascending and every entry (i, j) has its
// mirror (j, i).  For such a CSR the stable transpose is the CSR itself, bit for bit (row j of CSR^T lists the
// destinations of j ascending = the sources of j ascending = row j of the CSR).  One thread per entry: binary
// search of its row in rowptr, then of i in row j.
__global__ void undirected_check_kernel(const int32_t* __restrict__ rowptr, const int32_t* __restrict__ colidx, int n,
                                        long long nnz, int32_t* __restrict__ flag) {
    const long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (e >= nnz) return;
    int lo = 0, hi = n;
    while (lo < hi) {
        const int mid = (int)(((long long)lo + hi + 1) >> 1);
        if (__ldg(rowptr + mid) <= e) lo = mid; else hi = mid - 1;
    }
    const int i = lo, j = __ldg(colidx + e);
    if ((unsigned)j >= (unsigned)n) { *flag = 1; return; }
    if (e > __ldg(rowptr + i) && __ldg(colidx + e - 1) >= j) { *flag = 1; return; }
    int a = __ldg(rowptr + j), b = __ldg(rowptr + j + 1);
    while (a < b) {
        const int mid = a + ((b - a) >> 1);
        if (__ldg(colidx + mid) < i) a = mid + 1; else b = mid;
    }
    if (a >= __ldg(rowptr + j + 1) || __ldg(colidx + a) != i) *flag = 1;
}

// gnn_csr_validate: err[0] = smallest row r with rowptr[r] > rowptr[r+1] (or n if none), err[1] = smallest entry with
// colidx outside [0, n) (or nnz if none), kept in 64 bits as two atomicMin targets
__global__ void csr_validate_kernel(const int32_t* __restrict__ rowptr, const int32_t* __restrict__ colidx, int n,
                                    long long nnz, unsigned long long* __restrict__ err) {
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t < n && __ldg(rowptr + t) > __ldg(rowptr + t + 1)) atomicMin(err, (unsigned long long)t);
    if (t < nnz && (unsigned)__ldg(colidx + t) >= (unsigned)n) atomicMin(err + 1, (unsigned long long)t);
}

// rowptr_t[j] = number of entries with source id < j = lower_bound(sorted source ids, j)
__global__ void rowptr_t_kernel(const uint32_t* __restrict__ src_sorted, long long nnz, int n,
                                int32_t* __restrict__ rowptr_t) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j > n) return;
    long long lo = 0, hi = nnz;
    while (lo < hi) {
        const long long mid = (lo + hi) >> 1;
        if (src_sorted[mid] < (uint32_t)j) lo = mid + 1; else hi = mid;
    }
    rowptr_t[j] = (int32_t)lo;
}

// a11 - 16-row block layout (own layout; the paper's WSB, is prior art): window w = rows
// [16w, 16w+16); bit c of bitmap[row] is set iff the FIRST entry (row <- 16w + c) exists; every other entry
// (sources outside the window, duplicate in-window entries) goes to the remainder CSR in original order.
// One thread per row (rows of the locally dense graphs are short); pass 0 counts, pass 1 writes.
__global__ void block_layout_kernel(const int32_t* __restrict__ rowptr, const int32_t* __restrict__ colidx, int n,
                                    int pass, uint16_t* __restrict__ bitmap, int32_t* __restrict__ rem_cnt,
                                    const int32_t* __restrict__ rem_rowptr, int32_t* __restrict__ rem_colidx) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int w0 = (i >> 4) << 4;
    uint32_t seen = 0;
    int cnt = 0;
    int32_t* out = pass ? rem_colidx + rem_rowptr[i] : nullptr;
    for (int e = rowptr[i]; e < rowptr[i + 1]; ++e) {
        const int j = colidx[e];
        const unsigned c = (unsigned)(j - w0);
        if (c < 16u && !((seen >> c) & 1u)) { seen |= 1u << c; continue; }
        if (pass) out[cnt] = j;
        ++cnt;
    }
    if (!pass) { bitmap[i] = (uint16_t)seen; rem_cnt[i] = cnt; }
}
__global__ void pad_bitmap_kernel(uint16_t* bitmap, int n, int n_pad) {
    const int i = n + blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_pad) bitmap[i] = 0;
}

// ---- row f2: general WSB layout.  key = (row window << 32) | source column per CSR entry
__global__ void wsb_key_kernel(const int32_t* __restrict__ rowptr, const int32_t* __restrict__ colidx, int n, long long nnz,
                               unsigned long long* __restrict__ key) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= nnz) return;
    int lo = 0, hi = n;  // last row with rowptr[row] <= e
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if ((long long)__ldg(rowptr + mid) <= e) lo = mid; else hi = mid;
    }
    key[e] = ((unsigned long long)(lo >> 4) << 32) | (unsigned int)__ldg(colidx + e);
}
__device__ __forceinline__ long long lower_bound_u64(const unsigned long long* a, long long lo, long long hi, unsigned long long v) {
    while (lo < hi) {
        const long long mid = (lo + hi) >> 1;
        if (a[mid] < v) lo = mid + 1; else hi = mid;
    }
    return lo;
}
// win_uptr[w] = first unique (window, column) key of window w, w = 0 .. n_win
__global__ void wsb_winptr_kernel(const unsigned long long* __restrict__ ukey, const int* __restrict__ n_unique, int n_win,
                                  int32_t* __restrict__ win_uptr) {
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w > n_win) return;
    win_uptr[w] = (int32_t)lower_bound_u64(ukey, 0, *n_unique, (unsigned long long)w << 32);
}
__global__ void wsb_ntcb_kernel(const int32_t* __restrict__ win_uptr, int n_win, int32_t* __restrict__ ntcb) {
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w < n_win) ntcb[w] = (win_uptr[w + 1] - win_uptr[w] + 7) >> 3;
}
// the k-th unique column of window w goes to slot k of the window's TCB range (cols is zero-filled beforehand)
__global__ void wsb_cols_kernel(const unsigned long long* __restrict__ ukey, const int* __restrict__ n_unique,
                                const int32_t* __restrict__ win_uptr, const int32_t* __restrict__ row_offset,
                                int32_t* __restrict__ cols) {
    const long long u = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= *n_unique) return;
    const unsigned long long k = ukey[u];
    const int w = (int)(k >> 32);
    cols[(long long)row_offset[w] * 8 + (u - win_uptr[w])] = (int32_t)(unsigned int)k;
}
// one bit per CSR entry (integer atomicOr: the result does not depend on the order); a bit found set = duplicate entry
__global__ void wsb_bitmap_kernel(const int32_t* __restrict__ rowptr, const int32_t* __restrict__ colidx, int n, long long nnz,
                                  const unsigned long long* __restrict__ ukey, const int32_t* __restrict__ win_uptr,
                                  const int32_t* __restrict__ row_offset, unsigned int* __restrict__ bitmap32,
                                  int32_t* __restrict__ n_dup) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= nnz) return;
    int lo = 0, hi = n;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if ((long long)__ldg(rowptr + mid) <= e) lo = mid; else hi = mid;
    }
    const int w = lo >> 4, r = lo & 15;
    const unsigned long long k = ((unsigned long long)w << 32) | (unsigned int)__ldg(colidx + e);
    const long long pos = lower_bound_u64(ukey, win_uptr[w], win_uptr[w + 1], k) - win_uptr[w];
    const long long byte = ((long long)row_offset[w] + (pos >> 3)) * 16 + r;
    const unsigned int bit = 1u << ((pos & 7) + 8 * (byte & 3));
    const unsigned int old = atomicOr(bitmap32 + (byte >> 2), bit);
    if (old & bit) atomicAdd(n_dup, 1);
}

struct Layout {
    // persistent
    size_t perm, chunks, chunk_ptr, counts, rowptr_t, colidx_t, perm_t, chunks_t, chunk_ptr_t, dev_total;
    size_t blk_bitmap, blk_rem_rowptr, blk_rem_colidx, blk_cnt;
    size_t rem_rowptr_t, rem_colidx_t, rem_perm_t, rem_chunks_t, rem_chunk_ptr_t;
    size_t wsb_row_offset[2], wsb_cols[2], wsb_bitmap[2];          // [0] CSR, [1] CSR^T (only when the plan stores CSR^T)
    size_t wsb_key, wsb_key_sorted, wsb_nuniq, wsb_win_uptr, wsb_ntcb;  // scratch
    long long max_tcb;
    int n_win;
    // scratch
    size_t key, key_sorted, rowid, ekey_sorted, erow, cub, scratch_total;
    size_t cub_bytes;
    long long max_chunks, max_hub;
};

// defaults: large graphs (nnz >= 2^24) 4096 / 16384 / 4096 - enough rows in flight that long single-group rows and
// 4096-edge chunks do not form a tail; small graphs 256 / 1024 / 512 - heavy rows are cut finer so that the few
// CTAs that own them do not outlast the rest of the launch (profiles/r01_lane_width_sweep.md)
gnn_plan_opts_t resolve(const gnn_plan_opts_t* o, int64_t nnz) {
    const bool big = nnz >= (1ll << 24);
    gnn_plan_opts_t r = {big ? 4096 : 256, big ? 16384 : 1024, big ? 4096 : 512, 0, 0};
    if (o) {
        if (o->warp_max_deg > 0) r.warp_max_deg = o->warp_max_deg;
        if (o->cta_max_deg > 0) r.cta_max_deg = o->cta_max_deg;
        if (o->split_chunk > 0) r.split_chunk = o->split_chunk;
        r.build_transpose = o->build_transpose;
        r.build_blocks = o->build_blocks;
    }
    if (r.cta_max_deg < r.warp_max_deg) r.cta_max_deg = r.warp_max_deg;
    return r;
}

int n_bits(int n) {
    int b = 1;
    while (b < 32 && (1ll << b) < (long long)n) ++b;
    return b;
}

cudaError_t make_layout(int32_t n, int64_t nnz, const gnn_plan_opts_t& o, Layout& L) {
    const bool own_t = o.build_transpose != 0 && o.build_transpose != GNN_TRANSPOSE_UNDIRECTED;  // CSR^T stored in the plan
    L.max_hub = nnz / (o.cta_max_deg + 1) + 1;
    L.max_chunks = nnz / o.split_chunk + L.max_hub + 1;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t at = off; off += up(bytes); return at; };
    L.perm = take(sizeof(int32_t) * (size_t)n);
    L.chunks = take(sizeof(int32_t) * 4 * (size_t)L.max_chunks);
    L.chunk_ptr = take(sizeof(int32_t) * (size_t)(L.max_hub + 1));
    L.counts = take(sizeof(int32_t) * 16);   // 8 bin counts + flags + WSB info
    L.rowptr_t = L.colidx_t = L.perm_t = L.chunks_t = L.chunk_ptr_t = 0;
    if (own_t) {
        L.rowptr_t = take(sizeof(int32_t) * ((size_t)n + 1));
        L.colidx_t = take(sizeof(int32_t) * (size_t)(nnz > 0 ? nnz : 1));
        L.perm_t = take(sizeof(int32_t) * (size_t)n);
        L.chunks_t = take(sizeof(int32_t) * 4 * (size_t)L.max_chunks);
        L.chunk_ptr_t = take(sizeof(int32_t) * (size_t)(L.max_hub + 1));
    }
    L.blk_bitmap = L.blk_rem_rowptr = L.blk_rem_colidx = 0;
    L.n_win = (n + 15) / 16;
    L.max_tcb = nnz / 8 + L.n_win + 1;          // sum over windows of ceil(unique_w / 8) <= nnz / 8 + n_windows
    for (int t = 0; t < 2; ++t) L.wsb_row_offset[t] = L.wsb_cols[t] = L.wsb_bitmap[t] = 0;
    if (o.build_blocks & GNN_BLOCKS_WSB) {
        for (int t = 0; t < (own_t ? 2 : 1); ++t) {
            L.wsb_row_offset[t] = take(sizeof(int32_t) * ((size_t)L.n_win + 1));
            L.wsb_cols[t] = take(sizeof(int32_t) * 8 * (size_t)L.max_tcb);
            L.wsb_bitmap[t] = take(16 * (size_t)L.max_tcb);
        }
    }
    if (o.build_blocks & GNN_BLOCKS_DIAG) {
        L.blk_bitmap = take(sizeof(uint16_t) * (((size_t)n + 15) / 16 * 16));
        L.blk_rem_rowptr = take(sizeof(int32_t) * ((size_t)n + 1));
        L.blk_rem_colidx = take(sizeof(int32_t) * (size_t)(nnz > 0 ? nnz : 1));
    }
    // transposed remainder CSR + its bins (tensor-core backward on the diagonal layout: the out-of-window edges of the
    // source side run through the CSR src pass restricted to this structure)
    L.rem_rowptr_t = L.rem_colidx_t = L.rem_perm_t = L.rem_chunks_t = L.rem_chunk_ptr_t = 0;
    const bool rem_t = (o.build_blocks & GNN_BLOCKS_DIAG) && o.build_transpose != 0;
    if (rem_t) {
        L.rem_rowptr_t = take(sizeof(int32_t) * ((size_t)n + 1));
        L.rem_colidx_t = take(sizeof(int32_t) * (size_t)(nnz > 0 ? nnz : 1));
        L.rem_perm_t = take(sizeof(int32_t) * (size_t)n);
        L.rem_chunks_t = take(sizeof(int32_t) * 4 * (size_t)L.max_chunks);
        L.rem_chunk_ptr_t = take(sizeof(int32_t) * (size_t)(L.max_hub + 1));
    }
    L.dev_total = off;
    size_t t1 = 0, t2 = 0, t3 = 0, t4 = 0, t5 = 0, t6 = 0;
    cudaError_t e = cub::DeviceRadixSort::SortPairs(nullptr, t1, (const uint32_t*)nullptr, (uint32_t*)nullptr,
                                                    (const int32_t*)nullptr, (int32_t*)nullptr, (long long)n, 0, 7);
    if (e != cudaSuccess) return e;
    if (own_t || rem_t) {
        e = cub::DeviceRadixSort::SortPairs(nullptr, t2, (const uint32_t*)nullptr, (uint32_t*)nullptr,
                                            (const int32_t*)nullptr, (int32_t*)nullptr, (long long)nnz, 0, n_bits(n));
        if (e != cudaSuccess) return e;
    }
    if (o.build_blocks & GNN_BLOCKS_DIAG) {
        e = cub::DeviceScan::InclusiveSum(nullptr, t3, (const int32_t*)nullptr, (int32_t*)nullptr, n);
        if (e != cudaSuccess) return e;
    }
    if (o.build_blocks & GNN_BLOCKS_WSB) {
        e = cub::DeviceRadixSort::SortKeys(nullptr, t4, (const unsigned long long*)nullptr, (unsigned long long*)nullptr,
                                           (long long)nnz, 0, 32 + n_bits(L.n_win + 1));
        if (e == cudaSuccess)
            e = cub::DeviceSelect::Unique(nullptr, t5, (const unsigned long long*)nullptr, (unsigned long long*)nullptr,
                                          (int*)nullptr, (long long)nnz);
        if (e == cudaSuccess) e = cub::DeviceScan::InclusiveSum(nullptr, t6, (const int32_t*)nullptr, (int32_t*)nullptr, L.n_win);
        if (e != cudaSuccess) return e;
    }
    L.cub_bytes = t1 > t2 ? t1 : t2;
    for (size_t t : {t3, t4, t5, t6})
        if (t > L.cub_bytes) L.cub_bytes = t;
    off = 0;
    L.key = take(sizeof(uint32_t) * (size_t)n);
    L.key_sorted = take(sizeof(uint32_t) * (size_t)n);
    L.rowid = take(sizeof(int32_t) * (size_t)n);
    L.ekey_sorted = L.erow = 0;
    if (own_t || rem_t) {
        L.ekey_sorted = take(sizeof(uint32_t) * (size_t)(nnz > 0 ? nnz : 1));
        L.erow = take(sizeof(int32_t) * (size_t)(nnz > 0 ? nnz : 1));
    }
    L.blk_cnt = (o.build_blocks & GNN_BLOCKS_DIAG) ? take(sizeof(int32_t) * (size_t)n) : 0;
    L.wsb_key = L.wsb_key_sorted = L.wsb_nuniq = L.wsb_win_uptr = L.wsb_ntcb = 0;
    if (o.build_blocks & GNN_BLOCKS_WSB) {
        L.wsb_key = take(sizeof(unsigned long long) * (size_t)(nnz > 0 ? nnz : 1));        // keys, later the unique keys
        L.wsb_key_sorted = take(sizeof(unsigned long long) * (size_t)(nnz > 0 ? nnz : 1));
        L.wsb_nuniq = take(16);
        L.wsb_win_uptr = take(sizeof(int32_t) * ((size_t)L.n_win + 1));
        L.wsb_ntcb = take(sizeof(int32_t) * (size_t)L.n_win);
    }
    L.cub = take(L.cub_bytes + 16);
    L.scratch_total = off;
    return cudaSuccess;
}

// bins + chunk table of one CSR (rowptr); synchronises to read the counts back
cudaError_t build_bins(const int32_t* rowptr, int n, const gnn_plan_opts_t& o, const Layout& L, char* scratch,
                       int32_t* perm, int32_t* chunks, int32_t* chunk_ptr, int32_t* counts_dev, int32_t* counts_host,
                       cudaStream_t st) {
    uint32_t* key = (uint32_t*)(scratch + L.key);
    uint32_t* key_sorted = (uint32_t*)(scratch + L.key_sorted);
    int32_t* rowid = (int32_t*)(scratch + L.rowid);
    const int tb = 256;
    key_kernel<<<(n + tb - 1) / tb, tb, 0, st>>>(rowptr, n, o.warp_max_deg, o.cta_max_deg, key, rowid);
    size_t cb = L.cub_bytes;
    cudaError_t e = cub::DeviceRadixSort::SortPairs(scratch + L.cub, cb, (const uint32_t*)key, key_sorted,
                                                    (const int32_t*)rowid, perm, (long long)n, 0, 7, st);
    if (e != cudaSuccess) return e;
    count_kernel<<<1, 32, 0, st>>>(key_sorted, perm, rowptr, n, o.split_chunk, counts_dev, chunk_ptr, (int)L.max_hub);
    count_launch(3);
    e = cudaMemcpyAsync(counts_host, counts_dev, 4 * sizeof(int32_t), cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) return e;
    e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return e;
    if (counts_host[0] > 0) {
        chunk_kernel<<<counts_host[0], 128, 0, st>>>(perm, rowptr, chunk_ptr, chunks);
        count_launch();
    }
    return cudaGetLastError();
}

// WSB of one CSR (row f2): everything on the device; info_dev[0] = n_tcb, info_dev[1] = n_dup on return (async)
cudaError_t build_wsb(const int32_t* rowptr, const int32_t* colidx, int n, long long nnz, const Layout& L, char* sc,
                      int32_t* row_offset, int32_t* cols, uint8_t* bitmap, int32_t* info_dev, cudaStream_t st) {
    unsigned long long* key = (unsigned long long*)(sc + L.wsb_key);
    unsigned long long* key_sorted = (unsigned long long*)(sc + L.wsb_key_sorted);
    int* n_unique = (int*)(sc + L.wsb_nuniq);
    int32_t* win_uptr = (int32_t*)(sc + L.wsb_win_uptr);
    int32_t* ntcb = (int32_t*)(sc + L.wsb_ntcb);
    const int n_win = L.n_win, tb = 256;
    cudaError_t e = cudaMemsetAsync(cols, 0, sizeof(int32_t) * 8 * (size_t)L.max_tcb, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(bitmap, 0, 16 * (size_t)L.max_tcb, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(n_unique, 0, 16, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(row_offset, 0, sizeof(int32_t) * ((size_t)n_win + 1), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(info_dev, 0, 2 * sizeof(int32_t), st);
    if (e != cudaSuccess) return e;
    if (nnz > 0) {
        const unsigned nb = (unsigned)((nnz + tb - 1) / tb);
        wsb_key_kernel<<<nb, tb, 0, st>>>(rowptr, colidx, n, nnz, key);
        size_t cb = L.cub_bytes;
        e = cub::DeviceRadixSort::SortKeys(sc + L.cub, cb, (const unsigned long long*)key, key_sorted, nnz, 0,
                                           32 + n_bits(n_win + 1), st);
        if (e != cudaSuccess) return e;
        cb = L.cub_bytes;
        e = cub::DeviceSelect::Unique(sc + L.cub, cb, (const unsigned long long*)key_sorted, key, n_unique, nnz, st);   // key := unique keys
        if (e != cudaSuccess) return e;
        wsb_winptr_kernel<<<(n_win + 1 + tb - 1) / tb, tb, 0, st>>>(key, n_unique, n_win, win_uptr);
        wsb_ntcb_kernel<<<(n_win + tb - 1) / tb, tb, 0, st>>>(win_uptr, n_win, ntcb);
        cb = L.cub_bytes;
        e = cub::DeviceScan::InclusiveSum(sc + L.cub, cb, (const int32_t*)ntcb, row_offset + 1, n_win, st);
        if (e != cudaSuccess) return e;
        wsb_cols_kernel<<<nb, tb, 0, st>>>(key, n_unique, win_uptr, row_offset, cols);
        wsb_bitmap_kernel<<<nb, tb, 0, st>>>(rowptr, colidx, n, nnz, key, win_uptr, row_offset, (unsigned int*)bitmap, info_dev + 1);
        count_launch(7);
    }
    return cudaMemcpyAsync(info_dev, row_offset + n_win, sizeof(int32_t), cudaMemcpyDeviceToDevice, st);
}

}  // namespace
}  // namespace gnn

using namespace gnn;

extern "C" gnn_status_t gnn_plan_bytes(int32_t n, int64_t nnz, const gnn_plan_opts_t* opts, size_t* dev_bytes,
                                       size_t* scratch_bytes) {
    if (n < 1 || nnz < 0 || nnz >= (1ll << 31) || !dev_bytes || !scratch_bytes) {
        set_error("gnn_plan_bytes: need n >= 1, 0 <= nnz < 2^31 and non-NULL outputs");
        return GNN_EINVAL;
    }
    const gnn_plan_opts_t o = resolve(opts, nnz);
    Layout L;
    cudaError_t e = make_layout(n, nnz, o, L);
    if (e != cudaSuccess) {
        set_error("gnn_plan_bytes: CUDA error: %s", cudaGetErrorString(e));
        return GNN_ECUDA;
    }
    *dev_bytes = L.dev_total;
    *scratch_bytes = L.scratch_total;
    return GNN_OK;
}

extern "C" gnn_status_t gnn_plan_build(gnn_plan_t** plan, void* dev_mem, size_t dev_bytes, void* scratch,
                                       size_t scratch_bytes, int32_t n, int64_t nnz, const int32_t* rowptr,
                                       const int32_t* colidx, const gnn_plan_opts_t* opts, gnn_stream_t stream) {
    if (!plan || !dev_mem || !scratch || !rowptr || (!colidx && nnz > 0) || n < 1 || nnz < 0 || nnz >= (1ll << 31)) {
        set_error("gnn_plan_build: NULL pointer or bad sizes (n=%d nnz=%lld)", n, (long long)nnz);
        return GNN_EINVAL;
    }
    if (((uintptr_t)dev_mem | (uintptr_t)scratch) & 255) {
        set_error("gnn_plan_build: dev_mem and scratch must be 256-byte aligned");
        return GNN_EINVAL;
    }
    const gnn_plan_opts_t o = resolve(opts, nnz);
    Layout L;
    cudaError_t e = make_layout(n, nnz, o, L);
    if (e != cudaSuccess) {
        set_error("gnn_plan_build: CUDA error: %s", cudaGetErrorString(e));
        return GNN_ECUDA;
    }
    if (dev_bytes < L.dev_total || scratch_bytes < L.scratch_total) {
        set_error("gnn_plan_build: storage too small (dev %zu < %zu or scratch %zu < %zu)", dev_bytes, L.dev_total,
                  scratch_bytes, L.scratch_total);
        return GNN_EWORKSPACE;
    }
    cudaStream_t st = (cudaStream_t)stream;
    char* dm = (char*)dev_mem;
    char* sc = (char*)scratch;
    gnn_plan* P = new (std::nothrow) gnn_plan();
    if (!P) { set_error("gnn_plan_build: out of host memory"); return GNN_EINVAL; }
    P->n = n; P->nnz = nnz; P->opts = o; P->rowptr = rowptr; P->colidx = colidx;
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&P->sm_count, cudaDevAttrMultiProcessorCount, dev);
    int32_t* counts_dev = (int32_t*)(dm + L.counts);
    int32_t hc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    e = build_bins(rowptr, n, o, L, sc, (int32_t*)(dm + L.perm), (int32_t*)(dm + L.chunks),
                   (int32_t*)(dm + L.chunk_ptr), counts_dev, hc, st);
    int32_t directed = 0;
    if (e == cudaSuccess && o.build_transpose == GNN_TRANSPOSE_UNDIRECTED) {
        // direction-aware backward: the caller declares an undirected graph; verified here, then the
        // backward passes traverse the forward CSR and its bins - no transposed structure is built or stored
        e = cudaMemsetAsync(counts_dev + 9, 0, sizeof(int32_t), st);
        if (e == cudaSuccess && nnz > 0) {
            undirected_check_kernel<<<(unsigned)((nnz + 255) / 256), 256, 0, st>>>(rowptr, colidx, n, nnz, counts_dev + 9);
            count_launch();
        }
        if (e == cudaSuccess) e = cudaMemcpyAsync(&directed, counts_dev + 9, sizeof(int32_t), cudaMemcpyDeviceToHost, st);
        P->rowptr_t = const_cast<int32_t*>(rowptr);
        P->colidx_t = const_cast<int32_t*>(colidx);
        for (int t = 0; t < 4; ++t) hc[4 + t] = hc[t];
    } else if (e == cudaSuccess && o.build_transpose) {
        P->rowptr_t = (int32_t*)(dm + L.rowptr_t);
        P->colidx_t = (int32_t*)(dm + L.colidx_t);
        uint32_t* ekey_sorted = (uint32_t*)(sc + L.ekey_sorted);
        int32_t* erow = (int32_t*)(sc + L.erow);
        if (nnz > 0) {
            row_of_edge_kernel<<<(unsigned)((nnz + 255) / 256), 256, 0, st>>>(rowptr, n, nnz, erow);
            count_launch();
            size_t cb = L.cub_bytes;
            e = cub::DeviceRadixSort::SortPairs(sc + L.cub, cb, (const uint32_t*)colidx, ekey_sorted,
                                                (const int32_t*)erow, P->colidx_t, (long long)nnz, 0, n_bits(n), st);
        }
        if (e == cudaSuccess) {
            rowptr_t_kernel<<<(n + 1 + 255) / 256, 256, 0, st>>>(ekey_sorted, nnz, n, P->rowptr_t);
            count_launch();
            e = build_bins(P->rowptr_t, n, o, L, sc, (int32_t*)(dm + L.perm_t), (int32_t*)(dm + L.chunks_t),
                           (int32_t*)(dm + L.chunk_ptr_t), counts_dev + 4, hc + 4, st);
        }
    }
    int32_t unsorted = 0;
    if (e == cudaSuccess) e = cudaMemsetAsync(counts_dev + 8, 0, sizeof(int32_t), st);
    if (e == cudaSuccess && nnz > 1) {
        rows_unsorted_kernel<<<(unsigned)((nnz + 255) / 256), 256, 0, st>>>(rowptr, colidx, n, nnz, counts_dev + 8);
        count_launch();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(&unsorted, counts_dev + 8, sizeof(int32_t), cudaMemcpyDeviceToHost, st);
    int32_t wsb_info[4] = {0, 0, 0, 0};
    if (e == cudaSuccess && (o.build_blocks & GNN_BLOCKS_WSB)) {
        const bool own_t = o.build_transpose == GNN_TRANSPOSE_BUILD;
        P->has_wsb = 1;
        e = build_wsb(rowptr, colidx, n, nnz, L, sc, (int32_t*)(dm + L.wsb_row_offset[0]), (int32_t*)(dm + L.wsb_cols[0]),
                      (uint8_t*)(dm + L.wsb_bitmap[0]), counts_dev + 10, st);
        if (e == cudaSuccess && own_t)
            e = build_wsb(P->rowptr_t, P->colidx_t, n, nnz, L, sc, (int32_t*)(dm + L.wsb_row_offset[1]),
                          (int32_t*)(dm + L.wsb_cols[1]), (uint8_t*)(dm + L.wsb_bitmap[1]), counts_dev + 12, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(wsb_info, counts_dev + 10, (own_t ? 4 : 2) * sizeof(int32_t), cudaMemcpyDeviceToHost, st);
    }
    int32_t rem_nnz = 0;
    if (e == cudaSuccess && (o.build_blocks & GNN_BLOCKS_DIAG)) {
        P->n_windows = (n + 15) / 16;
        P->blk_bitmap = (uint16_t*)(dm + L.blk_bitmap);
        P->blk_rem_rowptr = (int32_t*)(dm + L.blk_rem_rowptr);
        P->blk_rem_colidx = (int32_t*)(dm + L.blk_rem_colidx);
        int32_t* cnt = (int32_t*)(sc + L.blk_cnt);
        const int tb = 128, gb = (n + tb - 1) / tb;
        block_layout_kernel<<<gb, tb, 0, st>>>(rowptr, colidx, n, 0, P->blk_bitmap, cnt, nullptr, nullptr);
        if (P->n_windows * 16 > n) pad_bitmap_kernel<<<1, 32, 0, st>>>(P->blk_bitmap, n, P->n_windows * 16);
        e = cudaMemsetAsync(P->blk_rem_rowptr, 0, sizeof(int32_t), st);
        size_t cb = L.cub_bytes;
        if (e == cudaSuccess) e = cub::DeviceScan::InclusiveSum(sc + L.cub, cb, (const int32_t*)cnt, P->blk_rem_rowptr + 1, n, st);
        if (e == cudaSuccess) {
            block_layout_kernel<<<gb, tb, 0, st>>>(rowptr, colidx, n, 1, nullptr, nullptr, P->blk_rem_rowptr, P->blk_rem_colidx);
            count_launch(3);
            e = cudaMemcpyAsync(&rem_nnz, P->blk_rem_rowptr + n, sizeof(int32_t), cudaMemcpyDeviceToHost, st);
        }
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    P->rem_nnz = rem_nnz;
    P->rows_sorted = unsorted ? 0 : 1;
    int32_t hr[4] = {0, 0, 0, 0};
    if (e == cudaSuccess && (o.build_blocks & GNN_BLOCKS_DIAG) && o.build_transpose != 0) {
        // stable transpose of the remainder CSR (same construction as CSR^T above) and its out-degree bins
        P->rem_rowptr_t = (int32_t*)(dm + L.rem_rowptr_t);
        P->rem_colidx_t = (int32_t*)(dm + L.rem_colidx_t);
        uint32_t* ekey_sorted = (uint32_t*)(sc + L.ekey_sorted);
        int32_t* erow = (int32_t*)(sc + L.erow);
        if (rem_nnz > 0) {
            row_of_edge_kernel<<<(unsigned)((rem_nnz + 255) / 256), 256, 0, st>>>(P->blk_rem_rowptr, n, rem_nnz, erow);
            count_launch();
            size_t cb = L.cub_bytes;
            e = cub::DeviceRadixSort::SortPairs(sc + L.cub, cb, (const uint32_t*)P->blk_rem_colidx, ekey_sorted,
                                                (const int32_t*)erow, P->rem_colidx_t, (long long)rem_nnz, 0, n_bits(n), st);
        }
        if (e == cudaSuccess) {
            rowptr_t_kernel<<<(n + 1 + 255) / 256, 256, 0, st>>>(ekey_sorted, rem_nnz, n, P->rem_rowptr_t);
            count_launch();
            e = build_bins(P->rem_rowptr_t, n, o, L, sc, (int32_t*)(dm + L.rem_perm_t), (int32_t*)(dm + L.rem_chunks_t),
                           (int32_t*)(dm + L.rem_chunk_ptr_t), counts_dev + 4, hr, st);   // counts slot reused (already read back)
        }
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        P->rem_tr = BinView{(int32_t*)(dm + L.rem_perm_t), (int32_t*)(dm + L.rem_chunks_t), (int32_t*)(dm + L.rem_chunk_ptr_t),
                            hr[0], hr[1], hr[2], hr[3]};
    }
    if (P->has_wsb) {
        P->wsb = WsbView{(int32_t*)(dm + L.wsb_row_offset[0]), (int32_t*)(dm + L.wsb_cols[0]), (uint8_t*)(dm + L.wsb_bitmap[0]),
                         wsb_info[0], wsb_info[1]};
        if (o.build_transpose == GNN_TRANSPOSE_BUILD)
            P->wsb_t = WsbView{(int32_t*)(dm + L.wsb_row_offset[1]), (int32_t*)(dm + L.wsb_cols[1]),
                               (uint8_t*)(dm + L.wsb_bitmap[1]), wsb_info[2], wsb_info[3]};
        else if (o.build_transpose == GNN_TRANSPOSE_UNDIRECTED)
            P->wsb_t = P->wsb;          // the stable transpose of an undirected CSR is the CSR itself
    }
    if (e != cudaSuccess) {
        set_error("gnn_plan_build: CUDA error: %s", cudaGetErrorString(e));
        delete P;
        return GNN_ECUDA;
    }
    if (directed) {
        set_error("gnn_plan_build: GNN_TRANSPOSE_UNDIRECTED needs strictly ascending rows and a mirror (j, i) for every entry (i, j)");
        delete P;
        return GNN_EINVAL;
    }
    P->fwd = BinView{(int32_t*)(dm + L.perm), (int32_t*)(dm + L.chunks), (int32_t*)(dm + L.chunk_ptr), hc[0], hc[1], hc[2], hc[3]};
    if (o.build_transpose == GNN_TRANSPOSE_UNDIRECTED)
        P->tr = P->fwd;
    else if (o.build_transpose)
        P->tr = BinView{(int32_t*)(dm + L.perm_t), (int32_t*)(dm + L.chunks_t), (int32_t*)(dm + L.chunk_ptr_t), hc[4], hc[5], hc[6], hc[7]};
    *plan = P;
    return GNN_OK;
}

extern "C" void gnn_plan_destroy(gnn_plan_t* plan) { delete plan; }

extern "C" gnn_status_t gnn_csr_validate(int32_t n, int64_t nnz, const int32_t* rowptr, const int32_t* colidx,
                                         void* scratch, gnn_stream_t stream) {
    if (n < 1 || nnz < 0 || nnz >= (1ll << 31) || !rowptr || (!colidx && nnz > 0) || !scratch || ((uintptr_t)scratch & 15)) {
        set_error("gnn_csr_validate: need n >= 1, 0 <= nnz < 2^31, non-NULL pointers and a 16-byte aligned scratch");
        return GNN_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long init[2] = {(unsigned long long)n, (unsigned long long)nnz}, got[2];
    int32_t ends[2] = {0, 0};
    cudaError_t e = cudaMemcpyAsync(scratch, init, sizeof(init), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) {
        const long long work = nnz > n ? nnz : n;
        csr_validate_kernel<<<(unsigned)((work + 255) / 256), 256, 0, st>>>(rowptr, colidx, n, nnz, (unsigned long long*)scratch);
        count_launch();
        e = cudaMemcpyAsync(got, scratch, sizeof(got), cudaMemcpyDeviceToHost, st);
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(&ends[0], rowptr, sizeof(int32_t), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&ends[1], rowptr + n, sizeof(int32_t), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { set_error("gnn_csr_validate: CUDA error: %s", cudaGetErrorString(e)); return GNN_ECUDA; }
    if (ends[0] != 0 || ends[1] != nnz) {
        set_error("gnn_csr_validate: rowptr[0] = %d (want 0), rowptr[n] = %d (want nnz = %lld)", ends[0], ends[1], (long long)nnz);
        return GNN_EINVAL;
    }
    if (got[0] != (unsigned long long)n) {
        set_error("gnn_csr_validate: rowptr decreases after row %llu", got[0]);
        return GNN_EINVAL;
    }
    if (got[1] != (unsigned long long)nnz) {
        set_error("gnn_csr_validate: colidx[%llu] is outside [0, n)", got[1]);
        return GNN_EINVAL;
    }
    return GNN_OK;
}

extern "C" const int32_t* gnn_plan_rowptr_t(const gnn_plan_t* plan) { return plan ? plan->rowptr_t : nullptr; }
extern "C" const int32_t* gnn_plan_colidx_t(const gnn_plan_t* plan) { return plan ? plan->colidx_t : nullptr; }

extern "C" gnn_status_t gnn_plan_export(const gnn_plan_t* P, int what, void* host_dst, size_t* bytes) {
    if (!P || !bytes) { set_error("gnn_plan_export: NULL plan or bytes"); return GNN_EINVAL; }
    const void* src = nullptr;
    size_t need = 0;
    int32_t counts[8] = {P->fwd.n_hub, P->fwd.n_cta, P->fwd.n_group, P->fwd.n_chunks,
                         P->tr.n_hub, P->tr.n_cta, P->tr.n_group, P->tr.n_chunks};
    const bool T = P->opts.build_transpose != 0;
    const int32_t flags[2] = {P->rows_sorted, P->opts.build_transpose == GNN_TRANSPOSE_UNDIRECTED ? 1 : 0};
    const int32_t wsbinfo[6] = {P->has_wsb, (P->n + 15) / 16, P->wsb.n_tcb, P->wsb.n_dup, P->wsb_t.n_tcb, P->wsb_t.n_dup};
    switch (what) {
        case GNN_PLAN_FLAGS: src = flags; need = sizeof(flags); break;
        case GNN_PLAN_COUNTS: need = sizeof(counts); break;
        case GNN_PLAN_PERM: src = P->fwd.perm; need = 4 * (size_t)P->n; break;
        case GNN_PLAN_CHUNKS: src = P->fwd.chunks; need = 16 * (size_t)P->fwd.n_chunks; break;
        case GNN_PLAN_CHUNK_PTR: src = P->fwd.chunk_ptr; need = 4 * ((size_t)P->fwd.n_hub + 1); break;
        case GNN_PLAN_ROWPTR_T: if (T) { src = P->rowptr_t; need = 4 * ((size_t)P->n + 1); } break;
        case GNN_PLAN_COLIDX_T: if (T) { src = P->colidx_t; need = 4 * (size_t)P->nnz; } break;
        case GNN_PLAN_PERM_T: if (T) { src = P->tr.perm; need = 4 * (size_t)P->n; } break;
        case GNN_PLAN_CHUNKS_T: if (T) { src = P->tr.chunks; need = 16 * (size_t)P->tr.n_chunks; } break;
        case GNN_PLAN_CHUNK_PTR_T: if (T) { src = P->tr.chunk_ptr; need = 4 * ((size_t)P->tr.n_hub + 1); } break;
        case GNN_PLAN_WSB_INFO: need = sizeof(wsbinfo); break;
        case GNN_PLAN_WSB_ROW_OFFSET: if (P->has_wsb) { src = P->wsb.row_offset; need = 4 * ((size_t)(P->n + 15) / 16 + 1); } break;
        case GNN_PLAN_WSB_COLS: if (P->has_wsb) { src = P->wsb.cols; need = 32 * (size_t)P->wsb.n_tcb; } break;
        case GNN_PLAN_WSB_BITMAP: if (P->has_wsb) { src = P->wsb.bitmap; need = 16 * (size_t)P->wsb.n_tcb; } break;
        case GNN_PLAN_WSB_ROW_OFFSET_T: if (P->has_wsb && T) { src = P->wsb_t.row_offset; need = 4 * ((size_t)(P->n + 15) / 16 + 1); } break;
        case GNN_PLAN_WSB_COLS_T: if (P->has_wsb && T) { src = P->wsb_t.cols; need = 32 * (size_t)P->wsb_t.n_tcb; } break;
        case GNN_PLAN_WSB_BITMAP_T: if (P->has_wsb && T) { src = P->wsb_t.bitmap; need = 16 * (size_t)P->wsb_t.n_tcb; } break;
        case GNN_PLAN_BLOCK_REM_ROWPTR_T: if (P->rem_rowptr_t) { src = P->rem_rowptr_t; need = 4 * ((size_t)P->n + 1); } break;
        case GNN_PLAN_BLOCK_REM_COLIDX_T: if (P->rem_rowptr_t) { src = P->rem_colidx_t; need = 4 * (size_t)P->rem_nnz; } break;
        case GNN_PLAN_BLOCK_BITMAP: if (P->blk_bitmap) { src = P->blk_bitmap; need = 2 * 16 * (size_t)P->n_windows; } break;
        case GNN_PLAN_BLOCK_REM_ROWPTR: if (P->blk_bitmap) { src = P->blk_rem_rowptr; need = 4 * ((size_t)P->n + 1); } break;
        case GNN_PLAN_BLOCK_REM_COLIDX: if (P->blk_bitmap) { src = P->blk_rem_colidx; need = 4 * (size_t)P->rem_nnz; } break;
        default: break;
    }
    if (what == GNN_PLAN_BLOCK_REM_COLIDX && P->blk_bitmap && P->rem_nnz == 0) { *bytes = 0; return GNN_OK; }
    if (what == GNN_PLAN_BLOCK_REM_COLIDX_T && P->rem_rowptr_t && P->rem_nnz == 0) { *bytes = 0; return GNN_OK; }
    if (what == GNN_PLAN_WSB_INFO) {
        const size_t cap0 = *bytes;
        *bytes = need;
        if (!host_dst) return GNN_OK;
        if (cap0 < need) { set_error("gnn_plan_export: buffer too small (%zu < %zu)", cap0, need); return GNN_EWORKSPACE; }
        memcpy(host_dst, wsbinfo, need);
        return GNN_OK;
    }
    if ((what == GNN_PLAN_WSB_COLS || what == GNN_PLAN_WSB_BITMAP) && P->has_wsb && P->wsb.n_tcb == 0) { *bytes = 0; return GNN_OK; }
    if ((what == GNN_PLAN_WSB_COLS_T || what == GNN_PLAN_WSB_BITMAP_T) && P->has_wsb && T && P->wsb_t.n_tcb == 0) { *bytes = 0; return GNN_OK; }
    if (what != GNN_PLAN_COUNTS && !src) {
        set_error("gnn_plan_export: item %d is not part of this plan", what);
        return GNN_EINVAL;
    }
    const size_t cap = *bytes;
    *bytes = need;
    if (!host_dst) return GNN_OK;
    if (cap < need) { set_error("gnn_plan_export: buffer too small (%zu < %zu)", cap, need); return GNN_EWORKSPACE; }
    if (what == GNN_PLAN_COUNTS) { memcpy(host_dst, counts, need); return GNN_OK; }
    if (what == GNN_PLAN_FLAGS) { memcpy(host_dst, flags, need); return GNN_OK; }
    if (need == 0) return GNN_OK;
    cudaError_t e = cudaMemcpy(host_dst, src, need, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) { set_error("gnn_plan_export: CUDA error: %s", cudaGetErrorString(e)); return GNN_ECUDA; }
    return GNN_OK;
}
