// ops_gt.cuh - Graph Transformer passes (PAPER.md:76; kernels PAPER.md:484-494; identities :539, :563).
// Scores are carried in the log2 domain: s' = <q,k> * log2(e)/sqrt(d), alpha = 2^(s' - L*log2(e)).
//
// Every Op splits a batch of KU edges into gather() - the lane's 128/256-bit loads of its chunk of each gathered
// row, kept raw in registers - and compute(), so the engine can issue batch t+1 before computing batch t.
#pragma once
#include "engine.cuh"

namespace gnn {

// T: feature dtype; CB: bytes per lane per row (16|32|64); G: lanes per row; KU: edges per batch;
// NT: gathered feature rows per edge; NSC: gathered per-(node, head) scalars per edge
template <typename T, int CB_, int G_, int KU_, int NT_, int NSC_> struct OpBase {
    static constexpr int kG = G_, kCB = CB_, kU = KU_, kCH = CB_ / (int)sizeof(T), kNT = NT_, kNSC = NSC_;
    using GeoT = Geo<G_>;
    using Ck = Chunk<T, CB_>;
    // states are sums merged by addition unless an Op says otherwise: MINARG = pairs (value in acc[0], source index
    // bits in acc[1]) that start at (+inf, -1) and are merged by the lexicographic minimum (ops_agg.cuh)
    static constexpr bool MINARG = false;
    // the gathered operands of one batch of KU edges, raw (unconverted) in registers
    struct Src {
        Ck c[KU_][NT_];
        float s[KU_][NSC_ > 0 ? NSC_ : 1];
    };
};

// online-softmax update with KU new scores: fills p[u], updates (m, l), returns the rescale
template <int KU> __device__ __forceinline__ float softmax_step(float& m, float& l, const float (&s)[KU], float (&pw)[KU]) {
    float mx = m;
#pragma unroll
    for (int u = 0; u < KU; ++u) mx = fmaxf(mx, s[u]);
    const float ms = (mx == -INFINITY) ? 0.f : mx;
    const float corr = ex2(m - ms);
    float sum = 0.f;
#pragma unroll
    for (int u = 0; u < KU; ++u) {
        pw[u] = ex2(s[u] - ms);
        sum += pw[u];
    }
    l = l * corr + sum;
    m = mx;
    return corr;
}

// ------------------------------------------------------------------------------------- GT forward
template <typename T, int CB_, int G_, int KU_> struct GtFwd : OpBase<T, CB_, G_, KU_, 2, 0> {
    static constexpr const char* kName = "gt_fwd";
    static constexpr int kMinBlocks = GNN_FWD_MINB;  // resident CTAs per SM the register budget is held to
    static constexpr bool kDoubleBuffer = GNN_FWD_DB != 0;
    using B = OpBase<T, CB_, G_, KU_, 2, 0>;
    using typename B::GeoT;
    using typename B::Ck;
    using typename B::Src;
    static constexpr int CH = B::kCH, KU = KU_;
    static constexpr int NA = 1, NS = 1;
    static constexpr bool SOFTMAX = true, HAS_DA = false;
    using St = State<NA, NS, CH>;
    struct Params {
        const T *q, *k, *v;
        T* out;
        float* lse;
        float qscale;  // log2(e) / sqrt(d)
    };
    struct Own { Ck q; };

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
        o.q.load_global(p.q, (size_t)row * sh.ld + g.eoff, valid && g.act);
    }
    __device__ __forceinline__ static void gather(const Params& p, const Shape& sh, const int (&nbr)[KU], const GeoT& g,
                                                  Src& src) {
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const bool pr = nbr[u] >= 0 && g.act;
            const size_t off = (size_t)(nbr[u] < 0 ? 0 : nbr[u]) * sh.ld + g.eoff;
            src.c[u][0].load_global(p.k, off, pr);
            src.c[u][1].load_global(p.v, off, pr);
        }
    }
    // this lane's neighbour of the NEXT edge block: its K and V rows into L2 (see run_edges)
    __device__ __forceinline__ static void prefetch(const Params& p, const Shape& sh, int nbr) {
        prefetch_row_l2(p.k + (size_t)nbr * sh.ld, sh.rowe * (int)sizeof(T));
        prefetch_row_l2(p.v + (size_t)nbr * sh.ld, sh.rowe * (int)sizeof(T));
    }
    __device__ __forceinline__ static void compute(St& st, const Own& o, const Params& p, const Shape&,
                                                   const int (&nbr)[KU], const GeoT& g, const Src& src) {
        float s[KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const Ck& kc = src.c[u][0];
            s[u] = dot(o.q, kc);
        }
        head_reduce(s, g.lpl);
        float pw[KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) s[u] = nbr[u] < 0 ? -INFINITY : s[u] * p.qscale;
        const float corr = softmax_step<KU>(st.m, st.sc[0], s, pw);
        scale<CH>(st.acc[0], corr);
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            float vf[CH];
            src.c[u][1].to_float(vf);
            axpy<CH>(st.acc[0], pw[u], vf);
        }
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&)[CH]) {
        const float l = st.sc[0];
        const float inv = l > 0.f ? 1.f / l : 0.f;
        float o[CH];
#pragma unroll
        for (int c = 0; c < CH; ++c) o[c] = st.acc[0][c] * inv;
        if (g.act) store_feat<CH>(p.out, (size_t)row * sh.ld + g.eoff, o);
        if (g.lead) p.lse[(size_t)row * sh.ldh + g.hd] = l > 0.f ? (st.m + lg2(l)) * kLn2 : -INFINITY;
    }
};

// ------------------------------------------------------------------- GT backward, dst pass (CSR)
// One sweep, no O needed: A = sum alpha dP k, B = sum alpha k, Delta = sum alpha dP;
// dQ = (A - Delta B)/sqrt(d)   (== sum_j alpha (dP - Delta) k_j / sqrt(d))
template <typename T, int CB_, int G_, int KU_> struct GtBwdDst : OpBase<T, CB_, G_, KU_, 2, 0> {
    static constexpr const char* kName = "gt_bwd_dst";
    static constexpr int kMinBlocks = GNN_BWD_MINB;  // resident CTAs per SM the register budget is held to
    static constexpr bool kDoubleBuffer = GNN_BWD_DB != 0;
    using B = OpBase<T, CB_, G_, KU_, 2, 0>;
    using typename B::GeoT;
    using typename B::Ck;
    using typename B::Src;
    static constexpr int CH = B::kCH, KU = KU_;
    static constexpr int NA = 2, NS = 1;
    static constexpr bool SOFTMAX = false, HAS_DA = false;
    using St = State<NA, NS, CH>;
    struct Params {
        const T *q, *k, *v, *dout;
        const float* lse;
        float *dq, *delta;
        float2* stat2;
        float qscale, inv_sqrt_d;
    };
    struct Own { Ck q, go; float lp; };

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
        const bool pr = valid && g.act;
        o.q.load_global(p.q, (size_t)row * sh.ld + g.eoff, pr);
        o.go.load_global(p.dout, (size_t)row * sh.ld + g.eoff, pr);
        o.lp = pr ? __ldg(p.lse + (size_t)row * sh.ldh + g.hd) * kLog2e : 0.f;
    }
    __device__ __forceinline__ static void gather(const Params& p, const Shape& sh, const int (&nbr)[KU], const GeoT& g,
                                                  Src& src) {
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const bool pr = nbr[u] >= 0 && g.act;
            const size_t off = (size_t)(nbr[u] < 0 ? 0 : nbr[u]) * sh.ld + g.eoff;
            src.c[u][0].load_global(p.k, off, pr);
            src.c[u][1].load_global(p.v, off, pr);
        }
    }
    __device__ __forceinline__ static void prefetch(const Params& p, const Shape& sh, int nbr) {
        prefetch_row_l2(p.k + (size_t)nbr * sh.ld, sh.rowe * (int)sizeof(T));
        prefetch_row_l2(p.v + (size_t)nbr * sh.ld, sh.rowe * (int)sizeof(T));
    }
    __device__ __forceinline__ static void compute(St& st, const Own& o, const Params& p, const Shape&,
                                                   const int (&nbr)[KU], const GeoT& g, const Src& src) {
        float r[2 * KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const Ck &kc = src.c[u][0], &vc = src.c[u][1];
            r[2 * u] = dot(o.q, kc);
            r[2 * u + 1] = dot(o.go, vc);
        }
        head_reduce(r, g.lpl);
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const float alpha = nbr[u] < 0 ? 0.f : ex2(r[2 * u] * p.qscale - o.lp);
            const float w = alpha * r[2 * u + 1];
            float kf[CH];
            src.c[u][0].to_float(kf);
            axpy<CH>(st.acc[0], w, kf);
            axpy<CH>(st.acc[1], alpha, kf);
            st.sc[0] += w;
        }
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&)[CH]) {
        const float dl = st.sc[0];
        float o[CH];
#pragma unroll
        for (int c = 0; c < CH; ++c) o[c] = (st.acc[0][c] - dl * st.acc[1][c]) * p.inv_sqrt_d;
        if (g.act) store_f32<CH>(p.dq, (size_t)row * sh.ld + g.eoff, o);
        if (g.lead) {
            p.delta[(size_t)row * sh.ldh + g.hd] = dl;
            p.stat2[(size_t)row * sh.ldh + g.hd] = make_float2(__ldg(p.lse + (size_t)row * sh.ldh + g.hd) * kLog2e, dl);
        }
    }
};

// ------------------------------------------------------------------ GT backward, src pass (CSR^T)
// rows are SOURCES j, entries the destinations i they feed; dK_j, dV_j accumulate in registers in
// CSR^T order: deterministic, no atomics (the paper uses atomicAdd here).
template <typename T, int CB_, int G_, int KU_> struct GtBwdSrc : OpBase<T, CB_, G_, KU_, 2, 2> {
    static constexpr const char* kName = "gt_bwd_src";
    static constexpr int kMinBlocks = GNN_BWD_MINB;  // resident CTAs per SM the register budget is held to
    static constexpr bool kDoubleBuffer = GNN_BWD_DB != 0;
    using B = OpBase<T, CB_, G_, KU_, 2, 2>;
    using typename B::GeoT;
    using typename B::Ck;
    using typename B::Src;
    static constexpr int CH = B::kCH, KU = KU_;
    static constexpr int NA = 2, NS = 0;
    static constexpr bool SOFTMAX = false, HAS_DA = false;
    using St = State<NA, NS, CH>;
    struct Params {
        const T *q, *k, *v, *dout;
        const float2* stat2;   // (L * log2(e), Delta) per (node, head), written by the dst pass
        float *dk, *dv;
        float kscale, inv_sqrt_d;
        int accumulate;        // 1: dk / dv already hold a partial result (the tile-local part of the block backward): add to it
    };
    struct Own { Ck k, v; };

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
        const bool pr = valid && g.act;
        o.k.load_global(p.k, (size_t)row * sh.ld + g.eoff, pr);
        o.v.load_global(p.v, (size_t)row * sh.ld + g.eoff, pr);
    }
    __device__ __forceinline__ static void gather(const Params& p, const Shape& sh, const int (&nbr)[KU], const GeoT& g,
                                                  Src& src) {
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const bool pr = nbr[u] >= 0 && g.act;
            const size_t i = (size_t)(nbr[u] < 0 ? 0 : nbr[u]);
            src.c[u][0].load_global(p.q, i * sh.ld + g.eoff, pr);
            src.c[u][1].load_global(p.dout, i * sh.ld + g.eoff, pr);
            const float2 t = pr ? __ldg(p.stat2 + i * sh.ldh + g.hd) : make_float2(0.f, 0.f);
            src.s[u][0] = t.x;
            src.s[u][1] = t.y;
        }
    }
    __device__ __forceinline__ static void prefetch(const Params& p, const Shape& sh, int nbr) {
        prefetch_row_l2(p.q + (size_t)nbr * sh.ld, sh.rowe * (int)sizeof(T));
        prefetch_row_l2(p.dout + (size_t)nbr * sh.ld, sh.rowe * (int)sizeof(T));
        prefetch_row_l2(p.stat2 + (size_t)nbr * sh.ldh, sh.H * (int)sizeof(float2));
    }
    __device__ __forceinline__ static void compute(St& st, const Own& o, const Params& p, const Shape&,
                                                   const int (&nbr)[KU], const GeoT& g, const Src& src) {
        float r[2 * KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const Ck &qc = src.c[u][0], &gc = src.c[u][1];
            r[2 * u] = dot(qc, o.k);
            r[2 * u + 1] = dot(gc, o.v);
        }
        head_reduce(r, g.lpl);
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const float li = src.s[u][0], di = src.s[u][1];
            const float alpha = nbr[u] < 0 ? 0.f : ex2(r[2 * u] * p.kscale - li);
            const float ds = alpha * (r[2 * u + 1] - di);
            float xf[CH];
            src.c[u][0].to_float(xf);
            axpy<CH>(st.acc[0], ds, xf);
            src.c[u][1].to_float(xf);
            axpy<CH>(st.acc[1], alpha, xf);
        }
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&)[CH]) {
        float o[CH], o2[CH];
#pragma unroll
        for (int c = 0; c < CH; ++c) { o[c] = st.acc[0][c] * p.inv_sqrt_d; o2[c] = st.acc[1][c]; }
        if (p.accumulate) {      // fixed order (partial already stored + this row's sum): still deterministic, one writer
            float a[CH], b[CH];
            load_f32<CH>(p.dk, (size_t)row * sh.ld + g.eoff, g.act, a);
            load_f32<CH>(p.dv, (size_t)row * sh.ld + g.eoff, g.act, b);
#pragma unroll
            for (int c = 0; c < CH; ++c) { o[c] += a[c]; o2[c] += b[c]; }
        }
        if (g.act) {
            store_f32<CH>(p.dk, (size_t)row * sh.ld + g.eoff, o);
            store_f32<CH>(p.dv, (size_t)row * sh.ld + g.eoff, o2);
        }
    }
};

}  // namespace gnn
