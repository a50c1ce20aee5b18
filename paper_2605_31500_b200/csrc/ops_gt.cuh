// ops_gt.cuh - Graph Transformer passes (PAPER.md:76; kernels PAPER.md:484-494; identities :539, :563).
// Scores are carried in the log2 domain: s' = <q,k> * log2(e)/sqrt(d), alpha = 2^(s' - L*log2(e)).
#pragma once
#include "engine.cuh"

namespace gnn {

// T: feature dtype; VB: bytes per load (16|32); NV: loads per lane; G: lanes per row; KU: edges per batch
template <typename T, int VB_, int NV_, int G_, int KU_> struct OpBase {
    static constexpr int kG = G_, kVB = VB_, kNV = NV_, kU = KU_, kCH = NV_ * VB_ / (int)sizeof(T);
    using GeoT = Geo<G_>;
    using Ck = Chunk<T, VB_, NV_>;
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
template <typename T, int VB_, int NV_, int G_, int KU_> struct GtFwd : OpBase<T, VB_, NV_, G_, KU_> {
    static constexpr const char* kName = "gt_fwd";
    using B = OpBase<T, VB_, NV_, G_, KU_>;
    using typename B::GeoT;
    using typename B::Ck;
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
    struct Own { float q[CH]; };

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
        Ck c;
        c.load(p.q, (size_t)row * sh.rowe + g.eoff, valid && g.act);
#pragma unroll
        for (int i = 0; i < CH; ++i) o.q[i] = c.get(i) * p.qscale;
    }
    __device__ __forceinline__ static void batch(St& st, const Own& o, const Params& p, const Shape& sh,
                                                 const int (&nbr)[KU], const GeoT& g) {
        Ck kr[KU], vr[KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const bool pr = nbr[u] >= 0 && g.act;
            const size_t off = (size_t)(nbr[u] < 0 ? 0 : nbr[u]) * sh.rowe + g.eoff;
            kr[u].load(p.k, off, pr);
            vr[u].load(p.v, off, pr);
        }
        float s[KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            float a0 = 0.f, a1 = 0.f;
#pragma unroll
            for (int c = 0; c < CH; c += 2) {
                a0 = fmaf(o.q[c], kr[u].get(c), a0);
                a1 = fmaf(o.q[c + 1], kr[u].get(c + 1), a1);
            }
            s[u] = a0 + a1;
        }
        head_reduce(s, g.lpl);
        float pw[KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) s[u] = nbr[u] < 0 ? -INFINITY : s[u];
        const float corr = softmax_step<KU>(st.m, st.sc[0], s, pw);
#pragma unroll
        for (int c = 0; c < CH; ++c) st.acc[0][c] *= corr;
#pragma unroll
        for (int u = 0; u < KU; ++u) {
#pragma unroll
            for (int c = 0; c < CH; ++c) st.acc[0][c] = fmaf(pw[u], vr[u].get(c), st.acc[0][c]);
        }
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&)[CH]) {
        const float l = st.sc[0];
        const float inv = l > 0.f ? 1.f / l : 0.f;
        float o[CH];
#pragma unroll
        for (int c = 0; c < CH; ++c) o[c] = st.acc[0][c] * inv;
        if (g.act) store_feat<CH>(p.out, (size_t)row * sh.rowe + g.eoff, o);
        if (g.lead) p.lse[(size_t)row * sh.H + g.hd] = l > 0.f ? (st.m + lg2(l)) * kLn2 : -INFINITY;
    }
};

// ------------------------------------------------------------------- GT backward, dst pass (CSR)
// One sweep, no O needed: A = sum alpha dP k, B = sum alpha k, Delta = sum alpha dP;
// dQ = (A - Delta B)/sqrt(d)   (== sum_j alpha (dP - Delta) k_j / sqrt(d))
template <typename T, int VB_, int NV_, int G_, int KU_> struct GtBwdDst : OpBase<T, VB_, NV_, G_, KU_> {
    static constexpr const char* kName = "gt_bwd_dst";
    using B = OpBase<T, VB_, NV_, G_, KU_>;
    using typename B::GeoT;
    using typename B::Ck;
    static constexpr int CH = B::kCH, KU = KU_;
    static constexpr int NA = 2, NS = 1;
    static constexpr bool SOFTMAX = false, HAS_DA = false;
    using St = State<NA, NS, CH>;
    struct Params {
        const T *q, *k, *v, *dout;
        const float* lse;
        float *dq, *delta;
        float qscale, inv_sqrt_d;
    };
    struct Own { float q[CH], go[CH], lp; };

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
        const bool pr = valid && g.act;
        Ck a, b;
        a.load(p.q, (size_t)row * sh.rowe + g.eoff, pr);
        b.load(p.dout, (size_t)row * sh.rowe + g.eoff, pr);
#pragma unroll
        for (int i = 0; i < CH; ++i) {
            o.q[i] = a.get(i) * p.qscale;
            o.go[i] = b.get(i);
        }
        o.lp = pr ? __ldg(p.lse + (size_t)row * sh.H + g.hd) * kLog2e : 0.f;
    }
    __device__ __forceinline__ static void batch(St& st, const Own& o, const Params& p, const Shape& sh,
                                                 const int (&nbr)[KU], const GeoT& g) {
        Ck kr[KU], vr[KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const bool pr = nbr[u] >= 0 && g.act;
            const size_t off = (size_t)(nbr[u] < 0 ? 0 : nbr[u]) * sh.rowe + g.eoff;
            kr[u].load(p.k, off, pr);
            vr[u].load(p.v, off, pr);
        }
        float r[2 * KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            float a = 0.f, b = 0.f;
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                a = fmaf(o.q[c], kr[u].get(c), a);
                b = fmaf(o.go[c], vr[u].get(c), b);
            }
            r[2 * u] = a;
            r[2 * u + 1] = b;
        }
        head_reduce(r, g.lpl);
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const float alpha = nbr[u] < 0 ? 0.f : ex2(r[2 * u] - o.lp);
            const float w = alpha * r[2 * u + 1];
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                const float kf = kr[u].get(c);
                st.acc[0][c] = fmaf(w, kf, st.acc[0][c]);
                st.acc[1][c] = fmaf(alpha, kf, st.acc[1][c]);
            }
            st.sc[0] += w;
        }
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&)[CH]) {
        const float dl = st.sc[0];
        float o[CH];
#pragma unroll
        for (int c = 0; c < CH; ++c) o[c] = (st.acc[0][c] - dl * st.acc[1][c]) * p.inv_sqrt_d;
        if (g.act) store_f32<CH>(p.dq, (size_t)row * sh.rowe + g.eoff, o);
        if (g.lead) p.delta[(size_t)row * sh.H + g.hd] = dl;
    }
};

// ------------------------------------------------------------------ GT backward, src pass (CSR^T)
// rows are SOURCES j, entries the destinations i they feed; dK_j, dV_j accumulate in registers in
// CSR^T order: deterministic, no atomics (the paper uses atomicAdd here).
template <typename T, int VB_, int NV_, int G_, int KU_> struct GtBwdSrc : OpBase<T, VB_, NV_, G_, KU_> {
    static constexpr const char* kName = "gt_bwd_src";
    using B = OpBase<T, VB_, NV_, G_, KU_>;
    using typename B::GeoT;
    using typename B::Ck;
    static constexpr int CH = B::kCH, KU = KU_;
    static constexpr int NA = 2, NS = 0;
    static constexpr bool SOFTMAX = false, HAS_DA = false;
    using St = State<NA, NS, CH>;
    struct Params {
        const T *q, *k, *v, *dout;
        const float *lse, *delta;
        float *dk, *dv;
        float kscale, inv_sqrt_d;
    };
    struct Own { float k[CH], v[CH]; };

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
        const bool pr = valid && g.act;
        Ck a, b;
        a.load(p.k, (size_t)row * sh.rowe + g.eoff, pr);
        b.load(p.v, (size_t)row * sh.rowe + g.eoff, pr);
#pragma unroll
        for (int i = 0; i < CH; ++i) {
            o.k[i] = a.get(i) * p.kscale;
            o.v[i] = b.get(i);
        }
    }
    __device__ __forceinline__ static void batch(St& st, const Own& o, const Params& p, const Shape& sh,
                                                 const int (&nbr)[KU], const GeoT& g) {
        Ck qr[KU], gr[KU];
        float li[KU], di[KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const bool pr = nbr[u] >= 0 && g.act;
            const size_t i = (size_t)(nbr[u] < 0 ? 0 : nbr[u]);
            qr[u].load(p.q, i * sh.rowe + g.eoff, pr);
            gr[u].load(p.dout, i * sh.rowe + g.eoff, pr);
            li[u] = pr ? __ldg(p.lse + i * sh.H + g.hd) : 0.f;
            di[u] = pr ? __ldg(p.delta + i * sh.H + g.hd) : 0.f;
        }
        float r[2 * KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            float a = 0.f, b = 0.f;
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                a = fmaf(qr[u].get(c), o.k[c], a);
                b = fmaf(gr[u].get(c), o.v[c], b);
            }
            r[2 * u] = a;
            r[2 * u + 1] = b;
        }
        head_reduce(r, g.lpl);
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const float alpha = nbr[u] < 0 ? 0.f : ex2(r[2 * u] - li[u] * kLog2e);
            const float ds = alpha * (r[2 * u + 1] - di[u]);
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                st.acc[0][c] = fmaf(ds, qr[u].get(c), st.acc[0][c]);
                st.acc[1][c] = fmaf(alpha, gr[u].get(c), st.acc[1][c]);
            }
        }
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&)[CH]) {
        float o[CH];
#pragma unroll
        for (int c = 0; c < CH; ++c) o[c] = st.acc[0][c] * p.inv_sqrt_d;
        if (g.act) {
            store_f32<CH>(p.dk, (size_t)row * sh.rowe + g.eoff, o);
            store_f32<CH>(p.dv, (size_t)row * sh.rowe + g.eoff, st.acc[1]);
        }
    }
};

}  // namespace gnn
