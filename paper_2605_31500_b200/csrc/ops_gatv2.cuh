// ops_gatv2.cuh - GATv2 passes (PAPER.md:74; kernels PAPER.md:488, :496-500; identities :539).
// e_ij = a^T LeakyReLU(xl_i + xr_j); the single gathered row xr_j is both score input and value.
#pragma once
#include "ops_gt.cuh"

namespace gnn {

__device__ __forceinline__ float lrelu(float z, float slope) { return fmaxf(z, 0.f) + slope * fminf(z, 0.f); }

// ------------------------------------------------------------------------------------ GATv2 forward
template <typename T, int CB_, int G_, int KU_> struct GatFwd : OpBase<T, CB_, G_, KU_, 1, 0> {
    static constexpr const char* kName = "gatv2_fwd";
    static constexpr int kMinBlocks = GNN_FWD_MINB;  // resident CTAs per SM the register budget is held to
    static constexpr bool kDoubleBuffer = GNN_FWD_DB != 0;
    using B = OpBase<T, CB_, G_, KU_, 1, 0>;
    using typename B::GeoT;
    using typename B::Ck;
    using typename B::Src;
    static constexpr int CH = B::kCH, KU = KU_;
    static constexpr int NA = 1, NS = 1;
    static constexpr bool SOFTMAX = true, HAS_DA = false;
    using St = State<NA, NS, CH>;
    struct Params {
        const T *xl, *xr;
        const float* a;
        T* out;
        float* lse;
        float slope;
    };
    struct Own { float xl[CH], a[CH]; };  // a pre-multiplied by log2(e)

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
        Ck c;
        c.load_global(p.xl, (size_t)row * sh.rowe + g.eoff, valid && g.act);
        c.to_float(o.xl);
        load_f32<CH>(p.a, g.eoff, g.act, o.a);
#pragma unroll
        for (int i = 0; i < CH; ++i) o.a[i] *= kLog2e;
    }
    __device__ __forceinline__ static void gather(const Params& p, const Shape& sh, const int (&nbr)[KU], const GeoT& g,
                                                  Src& src) {
#pragma unroll
        for (int u = 0; u < KU; ++u)
            src.c[u][0].load_global(p.xr, (size_t)(nbr[u] < 0 ? 0 : nbr[u]) * sh.rowe + g.eoff, nbr[u] >= 0 && g.act);
    }
    __device__ __forceinline__ static void compute(St& st, const Own& o, const Params& p, const Shape&,
                                                   const int (&nbr)[KU], const GeoT& g, const Src& src) {
        float s[KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const Ck& xc = src.c[u][0];
            float z[CH];
            add_chunk(xc, o.xl, z);
            float a0 = 0.f, a1 = 0.f;
#pragma unroll
            for (int c = 0; c < CH; c += 2) {
                a0 = fmaf(o.a[c], lrelu(z[c], p.slope), a0);
                a1 = fmaf(o.a[c + 1], lrelu(z[c + 1], p.slope), a1);
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
            const Ck& xc = src.c[u][0];
#pragma unroll
            for (int c = 0; c < CH; ++c) st.acc[0][c] = fmaf(pw[u], xc.get(c), st.acc[0][c]);
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

// ------------------------------------------------------------- GATv2 backward, dst pass ("AL" kernel)
// With s' = LeakyReLU'(z) in {1, slope} and LeakyReLU(z) = z s'(z), z = xl_i + xr_j, de_ij = alpha_ij (dP_ij - G_i):
//   dxl_i = a . S_i,              S_i = sum_j de_ij s'_ij                       (this pass)
//   dxr_j = V_j + a . U_j,        V_j = sum_i alpha_ij dO_i,  U_j = sum_i de_ij s'_ij   (src pass)
//   da    = sum_ij de_ij z_ij s'_ij = sum_i xl_i . S_i + sum_j xr_j . U_j
// so the attention-vector gradient needs no accumulators of its own: each pass adds (own row) . (its s'-weighted
// sum) to the per-lane da partial.  One sweep over the row (G_i is only known at its end):
//   A = sum w s', B = sum alpha s', G = sum w  with w = alpha dP;  S_i = A - G B.
template <typename T, int CB_, int G_, int KU_> struct GatBwdDst : OpBase<T, CB_, G_, KU_, 1, 0> {
    static constexpr const char* kName = "gatv2_bwd_dst";
    static constexpr int kMinBlocks = GNN_GAT_DST_MINB;  // resident CTAs per SM the register budget is held to
    static constexpr bool kDoubleBuffer = false;
    using B = OpBase<T, CB_, G_, KU_, 1, 0>;
    using typename B::GeoT;
    using typename B::Ck;
    using typename B::Src;
    static constexpr int CH = B::kCH, KU = KU_;
    static constexpr int NA = 2, NS = 1;
    static constexpr bool SOFTMAX = false, HAS_DA = true;
    using St = State<NA, NS, CH>;
    struct Params {
        const T *xl, *xr, *dout;
        const float *a, *lse;
        float *dxl, *g;
        float slope;
    };
    struct Own { float xl[CH], a[CH], lp; Ck go; };

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
        const bool pr = valid && g.act;
        Ck c0;
        c0.load_global(p.xl, (size_t)row * sh.rowe + g.eoff, pr);
        c0.to_float(o.xl);
        o.go.load_global(p.dout, (size_t)row * sh.rowe + g.eoff, pr);
        load_f32<CH>(p.a, g.eoff, g.act, o.a);
        o.lp = pr ? __ldg(p.lse + (size_t)row * sh.H + g.hd) * kLog2e : 0.f;
    }
    __device__ __forceinline__ static void gather(const Params& p, const Shape& sh, const int (&nbr)[KU], const GeoT& g,
                                                  Src& src) {
#pragma unroll
        for (int u = 0; u < KU; ++u)
            src.c[u][0].load_global(p.xr, (size_t)(nbr[u] < 0 ? 0 : nbr[u]) * sh.rowe + g.eoff, nbr[u] >= 0 && g.act);
    }
    __device__ __forceinline__ static void compute(St& st, const Own& o, const Params& p, const Shape&,
                                                   const int (&nbr)[KU], const GeoT& g, const Src& src) {
        float r[2 * KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const Ck& xc = src.c[u][0];
            float z[CH];
            add_chunk(xc, o.xl, z);
            float a0 = 0.f;
#pragma unroll
            for (int c = 0; c < CH; ++c) a0 = fmaf(o.a[c], lrelu(z[c], p.slope), a0);
            r[2 * u] = a0;
            r[2 * u + 1] = dot(o.go, xc);
        }
        head_reduce(r, g.lpl);
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const float alpha = nbr[u] < 0 ? 0.f : ex2(r[2 * u] * kLog2e - o.lp);
            const float w = alpha * r[2 * u + 1];
            const float ws = w * p.slope, as = alpha * p.slope;
            const Ck& xc = src.c[u][0];
            float z[CH];
            add_chunk(xc, o.xl, z);
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                const bool pos = z[c] > 0.f;
                st.acc[0][c] += pos ? w : ws;
                st.acc[1][c] += pos ? alpha : as;
            }
            st.sc[0] += w;
        }
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&da)[CH]) {
        const float gg = st.sc[0];
        float xl[CH], a[CH], o[CH];
        Ck c0;
        c0.load_global(p.xl, (size_t)row * sh.rowe + g.eoff, g.act);
        c0.to_float(xl);
        load_f32<CH>(p.a, g.eoff, g.act, a);
#pragma unroll
        for (int c = 0; c < CH; ++c) {
            const float sdash = st.acc[0][c] - gg * st.acc[1][c];   // S_i
            o[c] = a[c] * sdash;
            da[c] = fmaf(xl[c], sdash, da[c]);
        }
        if (g.act) store_f32<CH>(p.dxl, (size_t)row * sh.rowe + g.eoff, o);
        if (g.lead) p.g[(size_t)row * sh.H + g.hd] = gg;
    }
};

// ----------------------------------------------------- GATv2 backward, src pass over CSR^T ("R" kernel)
// V_j = sum_i alpha_ij dO_i and U_j = sum_i de_ij s'_ij accumulate in registers in CSR^T order (deterministic, no
// atomics); dxr_j = V_j + a . U_j and xr_j . U_j goes to the da partial (see the dst pass for the identities).
template <typename T, int CB_, int G_, int KU_> struct GatBwdSrc : OpBase<T, CB_, G_, KU_, 2, 2> {
    static constexpr const char* kName = "gatv2_bwd_src";
    static constexpr int kMinBlocks = GNN_GAT_SRC_MINB;  // resident CTAs per SM the register budget is held to
    static constexpr bool kDoubleBuffer = false;
    using B = OpBase<T, CB_, G_, KU_, 2, 2>;
    using typename B::GeoT;
    using typename B::Ck;
    using typename B::Src;
    static constexpr int CH = B::kCH, KU = KU_;
    static constexpr int NA = 2, NS = 0;
    static constexpr bool SOFTMAX = false, HAS_DA = true;
    using St = State<NA, NS, CH>;
    struct Params {
        const T *xl, *xr, *dout;
        const float *a, *lse, *g;
        float* dxr;
        float slope;
    };
    struct Own { Ck xr; float xrf[CH], a[CH]; };

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
        o.xr.load_global(p.xr, (size_t)row * sh.rowe + g.eoff, valid && g.act);
        o.xr.to_float(o.xrf);
        load_f32<CH>(p.a, g.eoff, g.act, o.a);
    }
    __device__ __forceinline__ static void gather(const Params& p, const Shape& sh, const int (&nbr)[KU], const GeoT& g,
                                                  Src& src) {
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const bool pr = nbr[u] >= 0 && g.act;
            const size_t i = (size_t)(nbr[u] < 0 ? 0 : nbr[u]);
            src.c[u][0].load_global(p.xl, i * sh.rowe + g.eoff, pr);
            src.c[u][1].load_global(p.dout, i * sh.rowe + g.eoff, pr);
            src.s[u][0] = pr ? __ldg(p.lse + i * sh.H + g.hd) : 0.f;
            src.s[u][1] = pr ? __ldg(p.g + i * sh.H + g.hd) : 0.f;
        }
    }
    __device__ __forceinline__ static void compute(St& st, const Own& o, const Params& p, const Shape&,
                                                   const int (&nbr)[KU], const GeoT& g, const Src& src) {
        float r[2 * KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const Ck &lc = src.c[u][0], &gc = src.c[u][1];
            float z[CH];
            add_chunk(lc, o.xrf, z);
            float a0 = 0.f;
#pragma unroll
            for (int c = 0; c < CH; ++c) a0 = fmaf(o.a[c], lrelu(z[c], p.slope), a0);
            r[2 * u] = a0;
            r[2 * u + 1] = dot(gc, o.xr);
        }
        head_reduce(r, g.lpl);
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const float li = src.s[u][0], gi = src.s[u][1];
            const float alpha = nbr[u] < 0 ? 0.f : ex2((r[2 * u] - li) * kLog2e);
            const float de = alpha * (r[2 * u + 1] - gi);
            const float des = de * p.slope;
            const Ck &lc = src.c[u][0], &gc = src.c[u][1];
            float z[CH];
            add_chunk(lc, o.xrf, z);
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                st.acc[0][c] = fmaf(alpha, gc.get(c), st.acc[0][c]);
                st.acc[1][c] += z[c] > 0.f ? de : des;
            }
        }
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&da)[CH]) {
        float xr[CH], a[CH], o[CH];
        Ck c0;
        c0.load_global(p.xr, (size_t)row * sh.rowe + g.eoff, g.act);
        c0.to_float(xr);
        load_f32<CH>(p.a, g.eoff, g.act, a);
#pragma unroll
        for (int c = 0; c < CH; ++c) {
            o[c] = fmaf(a[c], st.acc[1][c], st.acc[0][c]);
            da[c] = fmaf(xr[c], st.acc[1][c], da[c]);
        }
        if (g.act) store_f32<CH>(p.dxr, (size_t)row * sh.rowe + g.eoff, o);
    }
};

}  // namespace gnn
