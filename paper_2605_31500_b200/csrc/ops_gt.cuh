// ops_gt.cuh - Graph Transformer passes (PAPER.md:76; kernels PAPER.md:484-494; identities :539, :563).
// Scores are carried in the log2 domain: s' = <q,k> * log2(e)/sqrt(d), alpha = 2^(s' - L*log2(e)).
#pragma once
#include "engine.cuh"

namespace gnn {

template <typename T, int G_, int NV_> struct OpBase {
    static constexpr int kG = G_, kNV = NV_, kVEC = Elt<T>::VEC;
    using GeoT = Geo<G_, NV_, Elt<T>::VEC>;
};

// raw 16-byte gather kept unconverted until use (keeps the in-flight loads at 4 registers each)
template <typename T> __device__ __forceinline__ uint4 load_raw(const T* base, size_t elt, bool pred) {
    uint4 r = make_uint4(0u, 0u, 0u, 0u);
    if (pred) r = __ldg(reinterpret_cast<const uint4*>(base + elt));
    return r;
}
__device__ __forceinline__ void unpack(const uint4& r, float (&o)[4], const float*) {
    o[0] = __uint_as_float(r.x); o[1] = __uint_as_float(r.y); o[2] = __uint_as_float(r.z); o[3] = __uint_as_float(r.w);
}
__device__ __forceinline__ void unpack(const uint4& r, float (&o)[8], const __nv_bfloat16*) {
    o[0] = __uint_as_float(r.x << 16); o[1] = __uint_as_float(r.x & 0xffff0000u);
    o[2] = __uint_as_float(r.y << 16); o[3] = __uint_as_float(r.y & 0xffff0000u);
    o[4] = __uint_as_float(r.z << 16); o[5] = __uint_as_float(r.z & 0xffff0000u);
    o[6] = __uint_as_float(r.w << 16); o[7] = __uint_as_float(r.w & 0xffff0000u);
}

// online-softmax update for one vector slot with kU new scores: returns p[u], rescales l
__device__ __forceinline__ float softmax_step(float& m, float& l, const float (&s)[kU], float (&pw)[kU]) {
    float mx = m;
#pragma unroll
    for (int u = 0; u < kU; ++u) mx = fmaxf(mx, s[u]);
    const float ms = (mx == -INFINITY) ? 0.f : mx;
    const float corr = ex2(m - ms);
    float sum = 0.f;
#pragma unroll
    for (int u = 0; u < kU; ++u) {
        pw[u] = ex2(s[u] - ms);
        sum += pw[u];
    }
    l = l * corr + sum;
    m = mx;
    return corr;
}

// ------------------------------------------------------------------------------------- GT forward
template <typename T, int G_, int NV_> struct GtFwd : OpBase<T, G_, NV_> {
    static constexpr const char* kName = "gt_fwd";
    using B = OpBase<T, G_, NV_>;
    using typename B::GeoT;
    static constexpr int NV = NV_, VEC = B::kVEC;
    static constexpr int NA = 1, NS = 1;
    static constexpr bool SOFTMAX = true, HAS_DA = false;
    using St = State<NA, NS, NV, VEC>;
    struct Params {
        const T *q, *k, *v;
        T* out;
        float* lse;
        float qscale;  // log2(e) / sqrt(d)
    };
    struct Own { float q[NV][VEC]; };

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
#pragma unroll
        for (int t = 0; t < NV; ++t) {
            load_vec(p.q, (size_t)row * sh.rowe + g.eoff[t], valid && g.act[t], o.q[t]);
#pragma unroll
            for (int c = 0; c < VEC; ++c) o.q[t][c] *= p.qscale;
        }
    }
    __device__ __forceinline__ static void batch(St& st, const Own& o, const Params& p, const Shape& sh,
                                                 const int (&nbr)[kU], const GeoT& g) {
        uint4 kr[kU][NV], vr[kU][NV];
#pragma unroll
        for (int u = 0; u < kU; ++u)
#pragma unroll
            for (int t = 0; t < NV; ++t) {
                const bool pr = nbr[u] >= 0 && g.act[t];
                const size_t off = (size_t)(nbr[u] < 0 ? 0 : nbr[u]) * sh.rowe + g.eoff[t];
                kr[u][t] = load_raw(p.k, off, pr);
                vr[u][t] = load_raw(p.v, off, pr);
            }
        float s[NV * kU];
#pragma unroll
        for (int u = 0; u < kU; ++u)
#pragma unroll
            for (int t = 0; t < NV; ++t) {
                float f[VEC];
                unpack(kr[u][t], f, (const T*)nullptr);
                float a = 0.f;
#pragma unroll
                for (int c = 0; c < VEC; ++c) a = fmaf(o.q[t][c], f[c], a);
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
                unpack(vr[u][t], f, (const T*)nullptr);
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

// ------------------------------------------------------------------- GT backward, dst pass (CSR)
// One sweep, no O needed: A = sum alpha dP k, B = sum alpha k, Delta = sum alpha dP;
// dQ = (A - Delta B)/sqrt(d)   (== sum_j alpha (dP - Delta) k_j / sqrt(d))
template <typename T, int G_, int NV_> struct GtBwdDst : OpBase<T, G_, NV_> {
    static constexpr const char* kName = "gt_bwd_dst";
    using B = OpBase<T, G_, NV_>;
    using typename B::GeoT;
    static constexpr int NV = NV_, VEC = B::kVEC;
    static constexpr int NA = 2, NS = 1;
    static constexpr bool SOFTMAX = false, HAS_DA = false;
    using St = State<NA, NS, NV, VEC>;
    struct Params {
        const T *q, *k, *v, *dout;
        const float* lse;
        float *dq, *delta;
        float qscale, inv_sqrt_d;
    };
    struct Own { float q[NV][VEC], go[NV][VEC], lp[NV]; };

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
#pragma unroll
        for (int t = 0; t < NV; ++t) {
            const bool pr = valid && g.act[t];
            load_vec(p.q, (size_t)row * sh.rowe + g.eoff[t], pr, o.q[t]);
            load_vec(p.dout, (size_t)row * sh.rowe + g.eoff[t], pr, o.go[t]);
#pragma unroll
            for (int c = 0; c < VEC; ++c) o.q[t][c] *= p.qscale;
            o.lp[t] = pr ? __ldg(p.lse + (size_t)row * sh.H + g.hd[t]) * kLog2e : 0.f;
        }
    }
    __device__ __forceinline__ static void batch(St& st, const Own& o, const Params& p, const Shape& sh,
                                                 const int (&nbr)[kU], const GeoT& g) {
        uint4 kr[kU][NV], vr[kU][NV];
#pragma unroll
        for (int u = 0; u < kU; ++u)
#pragma unroll
            for (int t = 0; t < NV; ++t) {
                const bool pr = nbr[u] >= 0 && g.act[t];
                const size_t off = (size_t)(nbr[u] < 0 ? 0 : nbr[u]) * sh.rowe + g.eoff[t];
                kr[u][t] = load_raw(p.k, off, pr);
                vr[u][t] = load_raw(p.v, off, pr);
            }
        float r[2 * NV * kU];
#pragma unroll
        for (int u = 0; u < kU; ++u)
#pragma unroll
            for (int t = 0; t < NV; ++t) {
                float kf[VEC], vf[VEC];
                unpack(kr[u][t], kf, (const T*)nullptr);
                unpack(vr[u][t], vf, (const T*)nullptr);
                float a = 0.f, b = 0.f;
#pragma unroll
                for (int c = 0; c < VEC; ++c) {
                    a = fmaf(o.q[t][c], kf[c], a);
                    b = fmaf(o.go[t][c], vf[c], b);
                }
                r[2 * (t * kU + u)] = a;
                r[2 * (t * kU + u) + 1] = b;
            }
        head_reduce(r, g.lph);
#pragma unroll
        for (int t = 0; t < NV; ++t)
#pragma unroll
            for (int u = 0; u < kU; ++u) {
                const float alpha = nbr[u] < 0 ? 0.f : ex2(r[2 * (t * kU + u)] - o.lp[t]);
                const float w = alpha * r[2 * (t * kU + u) + 1];
                float kf[VEC];
                unpack(kr[u][t], kf, (const T*)nullptr);
#pragma unroll
                for (int c = 0; c < VEC; ++c) {
                    st.acc[0][t][c] = fmaf(w, kf[c], st.acc[0][t][c]);
                    st.acc[1][t][c] = fmaf(alpha, kf[c], st.acc[1][t][c]);
                }
                st.sc[0][t] += w;
            }
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&)[NV][VEC]) {
#pragma unroll
        for (int t = 0; t < NV; ++t) {
            const float dl = st.sc[0][t];
            float o[VEC];
#pragma unroll
            for (int c = 0; c < VEC; ++c) o[c] = (st.acc[0][t][c] - dl * st.acc[1][t][c]) * p.inv_sqrt_d;
            if (g.act[t]) store_f32<VEC>(p.dq, (size_t)row * sh.rowe + g.eoff[t], o);
            if (g.lead[t]) p.delta[(size_t)row * sh.H + g.hd[t]] = dl;
        }
    }
};

// ------------------------------------------------------------------ GT backward, src pass (CSR^T)
// rows are SOURCES j, entries the destinations i they feed; dK_j, dV_j accumulate in registers in
// CSR^T order: deterministic, no atomics (the paper uses atomicAdd here).
template <typename T, int G_, int NV_> struct GtBwdSrc : OpBase<T, G_, NV_> {
    static constexpr const char* kName = "gt_bwd_src";
    using B = OpBase<T, G_, NV_>;
    using typename B::GeoT;
    static constexpr int NV = NV_, VEC = B::kVEC;
    static constexpr int NA = 2, NS = 0;
    static constexpr bool SOFTMAX = false, HAS_DA = false;
    using St = State<NA, NS, NV, VEC>;
    struct Params {
        const T *q, *k, *v, *dout;
        const float *lse, *delta;
        float *dk, *dv;
        float kscale, inv_sqrt_d;
    };
    struct Own { float k[NV][VEC], v[NV][VEC]; };

    __device__ __forceinline__ static void load_own(Own& o, const Params& p, const Shape& sh, int row, bool valid,
                                                    const GeoT& g) {
#pragma unroll
        for (int t = 0; t < NV; ++t) {
            const bool pr = valid && g.act[t];
            load_vec(p.k, (size_t)row * sh.rowe + g.eoff[t], pr, o.k[t]);
            load_vec(p.v, (size_t)row * sh.rowe + g.eoff[t], pr, o.v[t]);
#pragma unroll
            for (int c = 0; c < VEC; ++c) o.k[t][c] *= p.kscale;
        }
    }
    __device__ __forceinline__ static void batch(St& st, const Own& o, const Params& p, const Shape& sh,
                                                 const int (&nbr)[kU], const GeoT& g) {
        uint4 qr[kU][NV], gr[kU][NV];
        float li[kU][NV], di[kU][NV];
#pragma unroll
        for (int u = 0; u < kU; ++u)
#pragma unroll
            for (int t = 0; t < NV; ++t) {
                const bool pr = nbr[u] >= 0 && g.act[t];
                const size_t i = (size_t)(nbr[u] < 0 ? 0 : nbr[u]);
                qr[u][t] = load_raw(p.q, i * sh.rowe + g.eoff[t], pr);
                gr[u][t] = load_raw(p.dout, i * sh.rowe + g.eoff[t], pr);
                li[u][t] = pr ? __ldg(p.lse + i * sh.H + g.hd[t]) : 0.f;
                di[u][t] = pr ? __ldg(p.delta + i * sh.H + g.hd[t]) : 0.f;
            }
        float r[2 * NV * kU];
#pragma unroll
        for (int u = 0; u < kU; ++u)
#pragma unroll
            for (int t = 0; t < NV; ++t) {
                float qf[VEC], gf[VEC];
                unpack(qr[u][t], qf, (const T*)nullptr);
                unpack(gr[u][t], gf, (const T*)nullptr);
                float a = 0.f, b = 0.f;
#pragma unroll
                for (int c = 0; c < VEC; ++c) {
                    a = fmaf(qf[c], o.k[t][c], a);
                    b = fmaf(gf[c], o.v[t][c], b);
                }
                r[2 * (t * kU + u)] = a;
                r[2 * (t * kU + u) + 1] = b;
            }
        head_reduce(r, g.lph);
#pragma unroll
        for (int t = 0; t < NV; ++t)
#pragma unroll
            for (int u = 0; u < kU; ++u) {
                const float alpha = nbr[u] < 0 ? 0.f : ex2(r[2 * (t * kU + u)] - li[u][t] * kLog2e);
                const float ds = alpha * (r[2 * (t * kU + u) + 1] - di[u][t]);
                float qf[VEC], gf[VEC];
                unpack(qr[u][t], qf, (const T*)nullptr);
                unpack(gr[u][t], gf, (const T*)nullptr);
#pragma unroll
                for (int c = 0; c < VEC; ++c) {
                    st.acc[0][t][c] = fmaf(ds, qf[c], st.acc[0][t][c]);
                    st.acc[1][t][c] = fmaf(alpha, gf[c], st.acc[1][t][c]);
                }
            }
    }
    __device__ __forceinline__ static void finalize(const St& st, const Params& p, const Shape& sh, int row,
                                                    const GeoT& g, float (&)[NV][VEC]) {
#pragma unroll
        for (int t = 0; t < NV; ++t) {
            float o[VEC];
#pragma unroll
            for (int c = 0; c < VEC; ++c) o[c] = st.acc[0][t][c] * p.inv_sqrt_d;
            if (g.act[t]) {
                store_f32<VEC>(p.dk, (size_t)row * sh.rowe + g.eoff[t], o);
                store_f32<VEC>(p.dv, (size_t)row * sh.rowe + g.eoff[t], st.acc[1][t]);
            }
        }
    }
};

}  // namespace gnn
