// ops_gatv2.cuh - GATv2 passes (PAPER.md:74; kernels PAPER.md:488, :496-500; identities :539).
// e_ij = a^T LeakyReLU(xl_i + xr_j); the single gathered row xr_j is both score input and value.
#pragma once
#include "ops_gt.cuh"

namespace gnn {

// LeakyReLU(z) = c1 z + c2 |z| with c1 = (1 + slope) / 2, c2 = (1 - slope) / 2, so with a' = a c1 and k = c2 / c1
// (|k| <= 1 for slope >= 0, which the entry points require)
//   sum_c a_c LeakyReLU(z_c) = sum_c a'_c (z_c + k |z_c|):
// two FFMAs per channel (|z| is an operand modifier) instead of max, min and two FFMAs.
struct LreluK {
    float c1, k;
    __device__ __forceinline__ explicit LreluK(float slope) : c1(0.5f * (1.f + slope)), k((1.f - slope) / (1.f + slope)) {}
};
__device__ __forceinline__ float lrelu_dot_step(float a1, float z, float k, float acc) {
    return fmaf(a1, fmaf(k, fabsf(z), z), acc);
}

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
    struct Own { float xl[CH], a[CH], k; };  // a pre-multiplied by log2(e) (1 + slope) / 2, k = (1 - slope) / (1 + slope)

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
        Ck c;
        c.load_global(p.xl, (size_t)row * sh.ld + g.eoff, valid && g.act);
        c.to_float(o.xl);
        load_f32<CH>(p.a, g.eoff, g.act, o.a);
        const LreluK lk(p.slope);
        o.k = lk.k;
#pragma unroll
        for (int i = 0; i < CH; ++i) o.a[i] *= kLog2e * lk.c1;
    }
    __device__ __forceinline__ static void gather(const Params& p, const Shape& sh, const int (&nbr)[KU], const GeoT& g,
                                                  Src& src) {
#pragma unroll
        for (int u = 0; u < KU; ++u)
            src.c[u][0].load_global(p.xr, (size_t)(nbr[u] < 0 ? 0 : nbr[u]) * sh.ld + g.eoff, nbr[u] >= 0 && g.act);
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
                a0 = lrelu_dot_step(o.a[c], z[c], o.k, a0);
                a1 = lrelu_dot_step(o.a[c + 1], z[c + 1], o.k, a1);
            }
            s[u] = a0 + a1;
        }
        head_reduce(s, g.lpl);
        float pw[KU];
#pragma unroll
        for (int u = 0; u < KU; ++u) s[u] = nbr[u] < 0 ? -INFINITY : s[u];
        const float corr = softmax_step<KU>(st.m, st.sc[0], s, pw);
        scale<CH>(st.acc[0], corr);
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            float xf[CH];
            src.c[u][0].to_float(xf);
            axpy<CH>(st.acc[0], pw[u], xf);
        }
    }
    __device__ __forceinline__ static void prefetch(const Params& p, const Shape& sh, int nbr) {
        prefetch_row_l2(p.xr + (size_t)nbr * sh.ld, sh.rowe * (int)sizeof(T));
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

// ------------------------------------------------------------- GATv2 backward, dst pass ("AL" kernel)
// With s' = LeakyReLU'(z) in {1, slope} and LeakyReLU(z) = z s'(z), z = xl_i + xr_j, de_ij = alpha_ij (dP_ij - G_i):
//   dxl_i = a . S_i,              S_i = sum_j de_ij s'_ij                       (this pass)
//   dxr_j = V_j + a . U_j,        V_j = sum_i alpha_ij dO_i,  U_j = sum_i de_ij s'_ij   (src pass)
//   da    = sum_ij de_ij z_ij s'_ij = sum_i xl_i . S_i + sum_j xr_j . U_j
// so the attention-vector gradient needs no accumulators of its own: each pass adds (own row) . (its s'-weighted
// sum) to the per-lane da partial.  One sweep over the row (G_i is only known at its end):
//   A = sum w s', B = sum alpha s', G = sum w  with w = alpha dP;  S_i = A - G B.
// s' takes two values, so A = slope G + (1 - slope) A+ with A+ = sum over {z > 0} of w (likewise B from B+ and
// sum alpha): the sweep keeps A+, B+ per channel (a compare and two predicated adds) and G, sum alpha per head.
template <typename T, int CB_, int G_, int KU_> struct GatBwdDst : OpBase<T, CB_, G_, KU_, 1, 0> {
    static constexpr const char* kName = "gatv2_bwd_dst";
    static constexpr int kMinBlocks = GNN_GAT_DST_MINB;  // resident CTAs per SM the register budget is held to
    static constexpr bool kDoubleBuffer = false;
    using B = OpBase<T, CB_, G_, KU_, 1, 0>;
    using typename B::GeoT;
    using typename B::Ck;
    using typename B::Src;
    static constexpr int CH = B::kCH, KU = KU_;
    static constexpr int NA = 2, NS = 2;
    static constexpr bool SOFTMAX = false, HAS_DA = true;
    using St = State<NA, NS, CH>;
    struct Params {
        const T *xl, *xr, *dout;
        const float *a, *lse;
        float *dxl, *g;
        float slope;
    };
    struct Own { float xl[CH], a[CH], lp, k; Ck go; };  // a pre-multiplied by log2(e) (1 + slope) / 2

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
        const bool pr = valid && g.act;
        Ck c0;
        c0.load_global(p.xl, (size_t)row * sh.ld + g.eoff, pr);
        c0.to_float(o.xl);
        o.go.load_global(p.dout, (size_t)row * sh.ld + g.eoff, pr);
        load_f32<CH>(p.a, g.eoff, g.act, o.a);
        const LreluK lk(p.slope);
        o.k = lk.k;
#pragma unroll
        for (int i = 0; i < CH; ++i) o.a[i] *= kLog2e * lk.c1;
        o.lp = pr ? __ldg(p.lse + (size_t)row * sh.ldh + g.hd) * kLog2e : 0.f;
    }
    __device__ __forceinline__ static void gather(const Params& p, const Shape& sh, const int (&nbr)[KU], const GeoT& g,
                                                  Src& src) {
#pragma unroll
        for (int u = 0; u < KU; ++u)
            src.c[u][0].load_global(p.xr, (size_t)(nbr[u] < 0 ? 0 : nbr[u]) * sh.ld + g.eoff, nbr[u] >= 0 && g.act);
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
            for (int c = 0; c < CH; ++c) a0 = lrelu_dot_step(o.a[c], z[c], o.k, a0);
            r[2 * u] = a0;
            r[2 * u + 1] = dot(o.go, xc);
        }
        head_reduce(r, g.lpl);
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const float alpha = nbr[u] < 0 ? 0.f : ex2(r[2 * u] - o.lp);
            const float w = alpha * r[2 * u + 1];
            const Ck& xc = src.c[u][0];
            float z[CH];
            add_chunk(xc, o.xl, z);
#pragma unroll
            for (int c = 0; c < CH; ++c) add2_if(z[c] > 0.f, st.acc[0][c], st.acc[1][c], w, alpha);   // (A+, B+) += (w, alpha)
            st.sc[0] += w;
            st.sc[1] += alpha;
        }
    }
    __device__ __forceinline__ static void prefetch(const Params& p, const Shape& sh, int nbr) {
        prefetch_row_l2(p.xr + (size_t)nbr * sh.ld, sh.rowe * (int)sizeof(T));
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&da)[CH]) {
        const float gg = st.sc[0], om = 1.f - p.slope;
        const float gs = p.slope * gg, as = p.slope * st.sc[1];
        float xl[CH], a[CH], o[CH];
        Ck c0;
        c0.load_global(p.xl, (size_t)row * sh.ld + g.eoff, g.act);
        c0.to_float(xl);
        load_f32<CH>(p.a, g.eoff, g.act, a);
#pragma unroll
        for (int c = 0; c < CH; ++c) {
            const float sdash = fmaf(om, st.acc[0][c], gs) - gg * fmaf(om, st.acc[1][c], as);   // S_i = A - G B
            o[c] = a[c] * sdash;
            da[c] = fmaf(xl[c], sdash, da[c]);
        }
        if (g.act) store_f32<CH>(p.dxl, (size_t)row * sh.ld + g.eoff, o);
        if (g.lead) p.g[(size_t)row * sh.ldh + g.hd] = gg;
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
    static constexpr int NA = 2, NS = 1;   // acc[1] = U+ (sum of de over {z > 0}), sc[0] = sum of de: U = slope sc + (1 - slope) U+
    static constexpr bool SOFTMAX = false, HAS_DA = true;
    using St = State<NA, NS, CH>;
    struct Params {
        const T *xl, *xr, *dout;
        const float *a, *lse, *g;
        float* dxr;
        float slope;
    };
    struct Own { Ck xr; float xrf[CH], a[CH], k; };  // a pre-multiplied by log2(e) (1 + slope) / 2

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
        o.xr.load_global(p.xr, (size_t)row * sh.ld + g.eoff, valid && g.act);
        o.xr.to_float(o.xrf);
        load_f32<CH>(p.a, g.eoff, g.act, o.a);
        const LreluK lk(p.slope);
        o.k = lk.k;
#pragma unroll
        for (int i = 0; i < CH; ++i) o.a[i] *= kLog2e * lk.c1;
    }
    __device__ __forceinline__ static void gather(const Params& p, const Shape& sh, const int (&nbr)[KU], const GeoT& g,
                                                  Src& src) {
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const bool pr = nbr[u] >= 0 && g.act;
            const size_t i = (size_t)(nbr[u] < 0 ? 0 : nbr[u]);
            src.c[u][0].load_global(p.xl, i * sh.ld + g.eoff, pr);
            src.c[u][1].load_global(p.dout, i * sh.ld + g.eoff, pr);
            src.s[u][0] = pr ? __ldg(p.lse + i * sh.ldh + g.hd) : 0.f;
            src.s[u][1] = pr ? __ldg(p.g + i * sh.ldh + g.hd) : 0.f;
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
            for (int c = 0; c < CH; ++c) a0 = lrelu_dot_step(o.a[c], z[c], o.k, a0);
            r[2 * u] = a0;
            r[2 * u + 1] = dot(gc, o.xr);
        }
        head_reduce(r, g.lpl);
#pragma unroll
        for (int u = 0; u < KU; ++u) {
            const float li = src.s[u][0], gi = src.s[u][1];
            const float alpha = nbr[u] < 0 ? 0.f : ex2(fmaf(-li, kLog2e, r[2 * u]));
            const float de = alpha * (r[2 * u + 1] - gi);
            const Ck &lc = src.c[u][0], &gc = src.c[u][1];
            float z[CH];
            add_chunk(lc, o.xrf, z);
            float gf[CH];
            gc.to_float(gf);
            axpy<CH>(st.acc[0], alpha, gf);
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                if (z[c] > 0.f) st.acc[1][c] += de;
            }
            st.sc[0] += de;
        }
    }
    __device__ __forceinline__ static void prefetch(const Params& p, const Shape& sh, int nbr) {
        prefetch_row_l2(p.xl + (size_t)nbr * sh.ld, sh.rowe * (int)sizeof(T));
        prefetch_row_l2(p.dout + (size_t)nbr * sh.ld, sh.rowe * (int)sizeof(T));
        prefetch_row_l2(p.lse + (size_t)nbr * sh.ldh, sh.H * (int)sizeof(float));
        prefetch_row_l2(p.g + (size_t)nbr * sh.ldh, sh.H * (int)sizeof(float));
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&da)[CH]) {
        float xr[CH], a[CH], o[CH];
        Ck c0;
        c0.load_global(p.xr, (size_t)row * sh.ld + g.eoff, g.act);
        c0.to_float(xr);
        load_f32<CH>(p.a, g.eoff, g.act, a);
        const float om = 1.f - p.slope, ds = p.slope * st.sc[0];
#pragma unroll
        for (int c = 0; c < CH; ++c) {
            const float u = fmaf(om, st.acc[1][c], ds);   // U_j
            o[c] = fmaf(a[c], u, st.acc[0][c]);
            da[c] = fmaf(xr[c], u, da[c]);
        }
        if (g.act) store_f32<CH>(p.dxr, (size_t)row * sh.ld + g.eoff, o);
    }
};

}  // namespace gnn
