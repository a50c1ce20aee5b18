// ops_agg.cuh - degree-aware min / max aggregation with argmin.
//   out[i,c] = min over stored in-neighbours j of x[j,c],  arg[i,c] = the j that attains it (ties: smaller j).
// The paper runs light rows one block per node and splits heavy rows over a 2-D grid whose chunks meet in a packed
// 64-bit (order-preserving key, index) atomicMin followed by an unpack pass.  Here the pass rides on the
// same degree bins as attention: a lane keeps (value, index) per channel in registers, CTA rows and hub chunks are
// merged by the lexicographic (value, index) minimum in shared memory / the hub merge kernel - no atomics, no
// packed intermediate, no unpack pass.  `sign` = +1 (min) or -1 (max: the minimum of -x, negated on store).
#pragma once
#include "kernels.cuh"
#include "ops_gt.cuh"

namespace gnn {

// SORTED: every CSR row lists its sources in ascending order (plan flag).  A lane then meets its candidates in
// ascending index order, so "first strict minimum wins" is the tie rule and the per-channel update is one compare and
// two selects; the merges across lane groups and hub chunks always use the full lexicographic order.
template <typename T, int CB_, int G_, int KU_, bool SORTED> struct MinFwdT : OpBase<T, CB_, G_, KU_, 1, 0> {
    static constexpr const char* kName = "seg_minmax_fwd";
    static constexpr int kMinBlocks = GNN_FWD_MINB;
    static constexpr bool kDoubleBuffer = false;
    using B = OpBase<T, CB_, G_, KU_, 1, 0>;
    using typename B::GeoT;
    using typename B::Ck;
    using typename B::Src;
    static constexpr int CH = B::kCH, KU = KU_;
    static constexpr int NA = 2, NS = 0;   // acc[0] = signed value, acc[1] = source index (int bits)
    static constexpr bool SOFTMAX = false, HAS_DA = false, MINARG = true;
    using St = State<NA, NS, CH>;
    struct Params {
        const T* x;
        T* out;
        int32_t* arg;
        float sign;
    };
    struct Own {};

    __device__ __forceinline__ static void init_state(St& st) {
#pragma unroll
        for (int c = 0; c < CH; ++c) {
            st.acc[0][c] = __int_as_float(0x7fc00000);   // NaN: "no candidate yet", loses every less-than-or-unordered test
            st.acc[1][c] = __int_as_float(-1);
        }
    }
    __device__ __forceinline__ static void load_own(Own&, const Params&, const Shape&, int, bool, const GeoT&) {}
    __device__ __forceinline__ static void gather(const Params& p, const Shape& sh, const int (&nbr)[KU], const GeoT& g,
                                                  Src& src) {
#pragma unroll
        for (int u = 0; u < KU; ++u)
            src.c[u][0].load_global(p.x, (size_t)(nbr[u] < 0 ? 0 : nbr[u]) * sh.ld + g.eoff, nbr[u] >= 0 && g.act);
    }
    __device__ __forceinline__ static void prefetch(const Params& p, const Shape& sh, int nbr) {
        prefetch_row_l2(p.x + (size_t)nbr * sh.ld, sh.rowe * (int)sizeof(T));
    }
    __device__ __forceinline__ static void compute(St& st, const Own&, const Params& p, const Shape&,
                                                   const int (&nbr)[KU], const GeoT&, const Src& src) {
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const Ck& xc = src.c[u][0];
            const int j = nbr[u];
            const bool valid = j >= 0;
            const float jf = __int_as_float(j);
            // branch-free lexicographic update (bitwise predicate logic keeps the compiler from short-circuit branches).
            // The state starts at (NaN, -1) and the test is "less than or unordered" (!(v >= bv), one FSETP.LTU), so
            // the first valid candidate always wins - also a signed value of +inf (x = +inf for min, -inf for max) -
            // and afterwards it is the plain IEEE `<`.  NaN inputs are outside the contract (include/gnn_attn.h).
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                const float v = p.sign * xc.get(c);
                const float bv = st.acc[0][c];
                const bool b = SORTED ? (valid & !(v >= bv))
                                      : (valid & (!(v >= bv) | ((v == bv) & (j < __float_as_int(st.acc[1][c])))));
                st.acc[0][c] = b ? v : bv;
                st.acc[1][c] = b ? jf : st.acc[1][c];
            }
        }
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&)[CH]) {
        float o[CH], a[CH];
#pragma unroll
        for (int c = 0; c < CH; ++c) {
            const bool has = __float_as_int(st.acc[1][c]) >= 0;
            o[c] = has ? p.sign * st.acc[0][c] : 0.f;   // rows without in-neighbours: 0 / -1 (A20)
            a[c] = st.acc[1][c];
        }
        if (g.act) {
            store_feat<CH>(p.out, (size_t)row * sh.ld + g.eoff, o);
            store_f32<CH>(reinterpret_cast<float*>(p.arg), (size_t)row * sh.ld + g.eoff, a);   // bit copies
        }
    }
};

template <typename T, int CB_, int G_, int KU_> using MinFwd = MinFwdT<T, CB_, G_, KU_, false>;
template <typename T, int CB_, int G_, int KU_> using MinFwdSorted = MinFwdT<T, CB_, G_, KU_, true>;

}  // namespace gnn
