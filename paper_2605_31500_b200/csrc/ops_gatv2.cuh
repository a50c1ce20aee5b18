// ops_gatv2.cuh - GATv2 passes (PAPER.md:74; kernels PAPER.md:488, :496-500; identities :539).
// e_ij = a^T LeakyReLU(xl_i + xr_j); the single gathered row xr_j is both score input and value.
#pragma once
#include "ops_gt.cuh"

namespace gnn {

// ------------------------------------------------------------------------------------ GATv2 forward
template <typename T, int G_, int NV_> struct GatFwd : OpBase<T, G_, NV_> {
    static constexpr const char* kName = "gatv2_fwd";
    using B = OpBase<T, G_, NV_>;
    using typename B::GeoT;
    static constexpr int NV = NV_, VEC = B::kVEC;
    static constexpr int NA = 1, NS = 1;
    static constexpr bool SOFTMAX = true, HAS_DA = false;
    using St = State<NA, NS, NV, VEC>;
    struct Params {
        const T *xl, *xr;
        const float* a;
        T* out;
        float* lse;
        float slope;
    };
    struct Own { float xl[NV][VEC], a[NV][VEC]; };  // a pre-multiplied by log2(e)

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
#pragma unroll
        for (int t = 0; t < NV; ++t) {
            load_vec(p.xl, (size_t)row * sh.rowe + g.eoff[t], valid && g.act[t], o.xl[t]);
            load_f32<VEC>(p.a, g.eoff[t], g.act[t], o.a[t]);
#pragma unroll
            for (int c = 0; c < VEC; ++c) o.a[t][c] *= kLog2e;
        }
    }
    __device__ __forceinline__ static void batch(St& st, const Own& o, const Params& p, const Shape& sh,
                                                 const int (&nbr)[kU], const GeoT& g) {
        uint4 xr[kU][NV];
#pragma unroll
        for (int u = 0; u < kU; ++u)
#pragma unroll
            for (int t = 0; t < NV; ++t)
                xr[u][t] = load_raw(p.xr, (size_t)(nbr[u] < 0 ? 0 : nbr[u]) * sh.rowe + g.eoff[t],
                                    nbr[u] >= 0 && g.act[t]);
        float s[NV * kU];
#pragma unroll
        for (int u = 0; u < kU; ++u)
#pragma unroll
            for (int t = 0; t < NV; ++t) {
                float f[VEC];
                unpack(xr[u][t], f, (const T*)nullptr);
                float a = 0.f;
#pragma unroll
                for (int c = 0; c < VEC; ++c) {
                    const float z = o.xl[t][c] + f[c];
                    a = fmaf(o.a[t][c], z > 0.f ? z : p.slope * z, a);
                }
                s[t * kU + u] = a;
            }
        head_reduce(s, g.lph);
#pragma unroll
        for (int t = 0; t < NV; ++t) {
            float sv[kU], pw[kU];
#pragma unroll
            for (int u = 0; u < kU; ++u) sv[u] = nbr[u] < 0 ? -INFINITY : s[t * kU + u];
            const float corr = softmax_step(st.m[t], st.sc[0][t], sv, pw);
#pragma unroll
            for (int c = 0; c < VEC; ++c) st.acc[0][t][c] *= corr;
#pragma unroll
            for (int u = 0; u < kU; ++u) {
                float f[VEC];
                unpack(xr[u][t], f, (const T*)nullptr);
#pragma unroll
                for (int c = 0; c < VEC; ++c) st.acc[0][t][c] = fmaf(pw[u], f[c], st.acc[0][t][c]);
            }
        }
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&)[NV][VEC]) {
#pragma unroll
        for (int t = 0; t < NV; ++t) {
            const float l = st.sc[0][t];
            const float inv = l > 0.f ? 1.f / l : 0.f;
            float o[VEC];
#pragma unroll
            for (int c = 0; c < VEC; ++c) o[c] = st.acc[0][t][c] * inv;
            if (g.act[t]) store_vec(p.out, (size_t)row * sh.rowe + g.eoff[t], o);
            if (g.lead[t]) p.lse[(size_t)row * sh.H + g.hd[t]] = l > 0.f ? (st.m[t] + lg2(l)) * kLn2 : -INFINITY;
        }
    }
};

// ------------------------------------------------------------- GATv2 backward, dst pass ("AL" kernel)
// One sweep: with as = a . LeakyReLU'(z), sg = LeakyReLU(z), w = alpha dP:
//   A1 = sum w as, B1 = sum alpha as, A2 = sum w sg, B2 = sum alpha sg, G = sum w
//   dxl_i = A1 - G B1;  this row's share of da = A2 - G B2      (== sum_j de_ij ...)
template <typename T, int G_, int NV_> struct GatBwdDst : OpBase<T, G_, NV_> {
    static constexpr const char* kName = "gatv2_bwd_dst";
    using B = OpBase<T, G_, NV_>;
    using typename B::GeoT;
    static constexpr int NV = NV_, VEC = B::kVEC;
    static constexpr int NA = 4, NS = 1;
    static constexpr bool SOFTMAX = false, HAS_DA = true;
    using St = State<NA, NS, NV, VEC>;
    struct Params {
        const T *xl, *xr, *dout;
        const float *a, *lse;
        float *dxl, *g;
        float slope;
    };
    struct Own { float xl[NV][VEC], go[NV][VEC], a[NV][VEC], lp[NV]; };

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
#pragma unroll
        for (int t = 0; t < NV; ++t) {
            const bool pr = valid && g.act[t];
            load_vec(p.xl, (size_t)row * sh.rowe + g.eoff[t], pr, o.xl[t]);
            load_vec(p.dout, (size_t)row * sh.rowe + g.eoff[t], pr, o.go[t]);
            load_f32<VEC>(p.a, g.eoff[t], g.act[t], o.a[t]);
            o.lp[t] = pr ? __ldg(p.lse + (size_t)row * sh.H + g.hd[t]) * kLog2e : 0.f;
        }
    }
    __device__ __forceinline__ static void batch(St& st, const Own& o, const Params& p, const Shape& sh,
                                                 const int (&nbr)[kU], const GeoT& g) {
        uint4 xr[kU][NV];
#pragma unroll
        for (int u = 0; u < kU; ++u)
#pragma unroll
            for (int t = 0; t < NV; ++t)
                xr[u][t] = load_raw(p.xr, (size_t)(nbr[u] < 0 ? 0 : nbr[u]) * sh.rowe + g.eoff[t],
                                    nbr[u] >= 0 && g.act[t]);
        float r[2 * NV * kU];
#pragma unroll
        for (int u = 0; u < kU; ++u)
#pragma unroll
            for (int t = 0; t < NV; ++t) {
                float f[VEC];
                unpack(xr[u][t], f, (const T*)nullptr);
                float a = 0.f, b = 0.f;
#pragma unroll
                for (int c = 0; c < VEC; ++c) {
                    const float z = o.xl[t][c] + f[c];
                    a = fmaf(o.a[t][c], z > 0.f ? z : p.slope * z, a);
                    b = fmaf(o.go[t][c], f[c], b);
                }
                r[2 * (t * kU + u)] = a;
                r[2 * (t * kU + u) + 1] = b;
            }
        head_reduce(r, g.lph);
#pragma unroll
        for (int t = 0; t < NV; ++t)
#pragma unroll
            for (int u = 0; u < kU; ++u) {
                const float alpha = nbr[u] < 0 ? 0.f : ex2(r[2 * (t * kU + u)] * kLog2e - o.lp[t]);
                const float w = alpha * r[2 * (t * kU + u) + 1];
                float f[VEC];
                unpack(xr[u][t], f, (const T*)nullptr);
#pragma unroll
                for (int c = 0; c < VEC; ++c) {
                    const float z = o.xl[t][c] + f[c];
                    const bool pos = z > 0.f;
                    const float sg = pos ? z : p.slope * z;
                    const float as = pos ? o.a[t][c] : p.slope * o.a[t][c];
                    st.acc[0][t][c] = fmaf(w, as, st.acc[0][t][c]);
                    st.acc[1][t][c] = fmaf(alpha, as, st.acc[1][t][c]);
                    st.acc[2][t][c] = fmaf(w, sg, st.acc[2][t][c]);
                    st.acc[3][t][c] = fmaf(alpha, sg, st.acc[3][t][c]);
                }
                st.sc[0][t] += w;
            }
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&da)[NV][VEC]) {
#pragma unroll
        for (int t = 0; t < NV; ++t) {
            const float gg = st.sc[0][t];
            float o[VEC];
#pragma unroll
            for (int c = 0; c < VEC; ++c) {
                o[c] = st.acc[0][t][c] - gg * st.acc[1][t][c];
                da[t][c] += st.acc[2][t][c] - gg * st.acc[3][t][c];
            }
            if (g.act[t]) store_f32<VEC>(p.dxl, (size_t)row * sh.rowe + g.eoff[t], o);
            if (g.lead[t]) p.g[(size_t)row * sh.H + g.hd[t]] = gg;
        }
    }
};

// ----------------------------------------------------- GATv2 backward, src pass over CSR^T ("R" kernel)
template <typename T, int G_, int NV_> struct GatBwdSrc : OpBase<T, G_, NV_> {
    static constexpr const char* kName = "gatv2_bwd_src";
    using B = OpBase<T, G_, NV_>;
    using typename B::GeoT;
    static constexpr int NV = NV_, VEC = B::kVEC;
    static constexpr int NA = 1, NS = 0;
    static constexpr bool SOFTMAX = false, HAS_DA = false;
    using St = State<NA, NS, NV, VEC>;
    struct Params {
        const T *xl, *xr, *dout;
        const float *a, *lse, *g;
        float* dxr;
        float slope;
    };
    struct Own { float xr[NV][VEC], a[NV][VEC]; };

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
#pragma unroll
        for (int t = 0; t < NV; ++t) {
            load_vec(p.xr, (size_t)row * sh.rowe + g.eoff[t], valid && g.act[t], o.xr[t]);
            load_f32<VEC>(p.a, g.eoff[t], g.act[t], o.a[t]);
        }
    }
    __device__ __forceinline__ static void batch(St& st, const Own& o, const Params& p, const Shape& sh,
                                                 const int (&nbr)[kU], const GeoT& g) {
        uint4 lr[kU][NV], gr[kU][NV];
        float li[kU][NV], gi[kU][NV];
#pragma unroll
        for (int u = 0; u < kU; ++u)
#pragma unroll
            for (int t = 0; t < NV; ++t) {
                const bool pr = nbr[u] >= 0 && g.act[t];
                const size_t i = (size_t)(nbr[u] < 0 ? 0 : nbr[u]);
                lr[u][t] = load_raw(p.xl, i * sh.rowe + g.eoff[t], pr);
                gr[u][t] = load_raw(p.dout, i * sh.rowe + g.eoff[t], pr);
                li[u][t] = pr ? __ldg(p.lse + i * sh.H + g.hd[t]) : 0.f;
                gi[u][t] = pr ? __ldg(p.g + i * sh.H + g.hd[t]) : 0.f;
            }
        float r[2 * NV * kU];
#pragma unroll
        for (int u = 0; u < kU; ++u)
#pragma unroll
            for (int t = 0; t < NV; ++t) {
                float lf[VEC], gf[VEC];
                unpack(lr[u][t], lf, (const T*)nullptr);
                unpack(gr[u][t], gf, (const T*)nullptr);
                float a = 0.f, b = 0.f;
#pragma unroll
                for (int c = 0; c < VEC; ++c) {
                    const float z = lf[c] + o.xr[t][c];
                    a = fmaf(o.a[t][c], z > 0.f ? z : p.slope * z, a);
                    b = fmaf(gf[c], o.xr[t][c], b);
                }
                r[2 * (t * kU + u)] = a;
                r[2 * (t * kU + u) + 1] = b;
            }
        head_reduce(r, g.lph);
#pragma unroll
        for (int t = 0; t < NV; ++t)
#pragma unroll
            for (int u = 0; u < kU; ++u) {
                const float alpha = nbr[u] < 0 ? 0.f : ex2((r[2 * (t * kU + u)] - li[u][t]) * kLog2e);
                const float de = alpha * (r[2 * (t * kU + u) + 1] - gi[u][t]);
                float lf[VEC], gf[VEC];
                unpack(lr[u][t], lf, (const T*)nullptr);
                unpack(gr[u][t], gf, (const T*)nullptr);
#pragma unroll
                for (int c = 0; c < VEC; ++c) {
                    const float z = lf[c] + o.xr[t][c];
                    const float as = z > 0.f ? o.a[t][c] : p.slope * o.a[t][c];
                    st.acc[0][t][c] = fmaf(alpha, gf[c], fmaf(de, as, st.acc[0][t][c]));
                }
            }
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&)[NV][VEC]) {
#pragma unroll
        for (int t = 0; t < NV; ++t)
            if (g.act[t]) store_f32<VEC>(p.dxr, (size_t)row * sh.rowe + g.eoff[t], st.acc[0][t]);
    }
};

}  // namespace gnn
