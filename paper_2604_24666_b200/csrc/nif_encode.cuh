// nif_encode.cuh -- device functions for steps (a2) map back and (a3) encode, shared by the
// scalar-FMA engine and the tcgen05 fused kernel.  PAPER.md:41 (inverse deformation)
// Eq. 1 (psi = phi o gamma), readings R2-R6 of DESIGN.md section 3.
#pragma once

#include "nif_common.cuh"

// (a2) inverse deformation of a deformed-space point, fp32: twist^-1(bend^-1(P)) (R7)
__device__ __forceinline__ void nif_inverse_deform(float theta_max, float k, float X, float Y, float Z,
                                                   float& x, float& y, float& z)
{
    float bx = X, by = Y, bz = Z;
    if (fabsf(k) >= 1e-6f) {
        float dx = k * X;
        float dy = 1.0f - k * Y;
        float r = sqrtf(dx * dx + dy * dy);
        bx = atan2f(dx, dy) / k;
        by = (2.0f * Y - k * (X * X + Y * Y)) / (1.0f + r);
    }
    float a = -theta_max * (by + 1.0f) * 0.5f;
    float sa, ca;
    sincosf(a, &sa, &ca);
    x = bx * ca + bz * sa;
    y = by;
    z = -bx * sa + bz * ca;
}

// rest-space point -> normalised grid coordinate in [0,1] ("normalized query point")
__device__ __forceinline__ float nif_normalise(float p) { return __saturatef((p + 1.0f) * 0.5f); }

// sample s of gamma(x_n) for one coordinate: s = 0 -> x; s = 1+2k -> (sin(2^k x)+1)/2;
// s = 2+2k -> (cos(2^k x)+1)/2  (Eq. 1 literal, no pi; R3, R4)
__device__ __forceinline__ float nif_pe_sample(float xn, int s)
{
    if (s == 0) return xn;
    const int k = (s - 1) >> 1;
    const float arg = ldexpf(1.0f, k) * xn;
    const float v = ((s - 1) & 1) ? cosf(arg) : sinf(arg);
    return (v + 1.0f) * 0.5f;
}

// NIF_ENC_CONCAT: scalar j of gamma(x_n) handed to the MLP as it is: j < 3 -> x; then per band k:
// sin(2^k x) of the three axes, cos(2^k x) of the three axes (raw values, no pi); 0 beyond 3 + 6B
__device__ __forceinline__ float nif_pe_scalar(const float* __restrict__ xn, int j, int bands)
{
    if (j < 3) return xn[j];
    const int jj = j - 3, k = jj / 6, r = jj - 6 * k;
    if (k >= bands) return 0.0f;
    const float arg = ldexpf(1.0f, k) * xn[r >= 3 ? r - 3 : r];
    return r >= 3 ? cosf(arg) : sinf(arg);
}

template <typename T, int F> struct NifEntry;
template <> struct NifEntry<float, 1> {
    static __device__ __forceinline__ void load(const float* t, uint32_t i, float* v) { v[0] = __ldg(t + i); }
};
template <> struct NifEntry<float, 2> {
    static __device__ __forceinline__ void load(const float* t, uint32_t i, float* v)
    { float2 a = __ldg(reinterpret_cast<const float2*>(t) + i); v[0] = a.x; v[1] = a.y; }
};
template <> struct NifEntry<float, 4> {
    static __device__ __forceinline__ void load(const float* t, uint32_t i, float* v)
    { float4 a = __ldg(reinterpret_cast<const float4*>(t) + i); v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; }
};
template <> struct NifEntry<__half, 1> {
    static __device__ __forceinline__ void load(const __half* t, uint32_t i, float* v)
    { v[0] = __half2float(__ldg(t + i)); }
};
template <> struct NifEntry<__half, 2> {
    static __device__ __forceinline__ void load(const __half* t, uint32_t i, float* v)
    { float2 a = __half22float2(__ldg(reinterpret_cast<const __half2*>(t) + i)); v[0] = a.x; v[1] = a.y; }
};
template <> struct NifEntry<__half, 4> {
    static __device__ __forceinline__ void load(const __half* t, uint32_t i, float* v)
    {
        uint2 raw = __ldg(reinterpret_cast<const uint2*>(t) + i);
        float2 a = __half22float2(*reinterpret_cast<__half2*>(&raw.x));
        float2 b = __half22float2(*reinterpret_cast<__half2*>(&raw.y));
        v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
    }
};

// phi_l(p): trilinear interpolation of the 8 surrounding table entries of one level
// (index rule R6: dense i + (N+1)(j + (N+1)k) if (N+1)^3 <= T else the [MESK22] hash).
// Corner order (dx,dy,dz) = 000,100,010,110,001,101,011,111; fp32 accumulate.
template <typename T, int F>
__device__ __forceinline__ void nif_level_features(const T* __restrict__ level_table, int N, bool dense,
                                                   uint32_t t_mask, float px, float py, float pz,
                                                   float* __restrict__ feat)
{
    const float fn = (float)N, top = (float)(N - 1);
    const float posx = px * fn, posy = py * fn, posz = pz * fn;
    const float flx = fmaxf(fminf(floorf(posx), top), 0.0f);
    const float fly = fmaxf(fminf(floorf(posy), top), 0.0f);
    const float flz = fmaxf(fminf(floorf(posz), top), 0.0f);
    const float wx = posx - flx, wy = posy - fly, wz = posz - flz;
    const uint32_t cx = (uint32_t)flx, cy = (uint32_t)fly, cz = (uint32_t)flz;
    uint32_t idx[8];
    if (dense) {
        const uint32_t np1 = (uint32_t)N + 1u;
        const uint32_t b = cx + np1 * (cy + np1 * cz);
#pragma unroll
        for (int c = 0; c < 8; ++c)
            idx[c] = b + (uint32_t)(c & 1) + np1 * ((uint32_t)((c >> 1) & 1) + np1 * (uint32_t)(c >> 2));
    } else {
        const uint32_t hx0 = cx, hx1 = cx + 1u;
        const uint32_t hy0 = cy * 2654435761u, hy1 = (cy + 1u) * 2654435761u;
        const uint32_t hz0 = cz * 805459861u, hz1 = (cz + 1u) * 805459861u;
#pragma unroll
        for (int c = 0; c < 8; ++c)
            idx[c] = (((c & 1) ? hx1 : hx0) ^ (((c >> 1) & 1) ? hy1 : hy0) ^ ((c >> 2) ? hz1 : hz0)) & t_mask;
    }
    float v[8][F];
#pragma unroll
    for (int c = 0; c < 8; ++c) NifEntry<T, F>::load(level_table, idx[c], v[c]);
#pragma unroll
    for (int f = 0; f < F; ++f) feat[f] = 0.0f;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const float w = (((c & 1) ? wx : 1.0f - wx) * (((c >> 1) & 1) ? wy : 1.0f - wy)) * ((c >> 2) ? wz : 1.0f - wz);
#pragma unroll
        for (int f = 0; f < F; ++f) feat[f] = fmaf(w, v[c][f], feat[f]);
    }
}

// (a5) heads from the 12 logits (B:7; R13, R16, R17)
__device__ __forceinline__ float nif_sigmoid(float z) { return 1.0f / (1.0f + expf(-z)); }

// what the optional hit-position outputs need beyond the logits
struct NifDecodeCtx {
    const float* origin;
    const float* dir;
    float theta_max, bend_k;
};

__device__ __forceinline__ void nif_decode_store(const float* __restrict__ z, float t_in, float t_out,
                                                 long long ray, const nif_query_out& out, unsigned flags,
                                                 const NifDecodeCtx& ctx)
{
    out.occlusion[ray] = nif_sigmoid(z[0]);
    if (flags & NIF_OCCLUSION_ONLY) {
        if (out.raw_logits) {
            out.raw_logits[NIF_N_OUT * ray] = z[0];
#pragma unroll
            for (int a = 1; a < NIF_N_OUT; ++a) out.raw_logits[NIF_N_OUT * ray + a] = 0.0f;
        }
        return;
    }
    const float ell = t_out - t_in;
    float d, D;
    if (flags & NIF_DIST_LOG) {                  // P:87, R24: ReLU output = log(1 + accumulated distance)
        D = expm1f(fmaxf(z[1], 0.0f));
        d = D - t_in;
    } else {                                     // P:59-61, R14: local distance in [0, l], D = t_in + d
        d = nif_sigmoid(z[1]) * ell;
        D = t_in + d;
    }
    out.distance[ray] = d;
    out.dist_total[ray] = D;
    const float nn = z[2] * z[2] + z[3] * z[3] + z[4] * z[4];
    const float inv = rsqrtf(fmaxf(nn, 1e-24f));
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        out.normal[3 * ray + a] = z[2 + a] * inv;
        out.albedo[3 * ray + a] = nif_sigmoid(z[5 + a]);
    }
#pragma unroll
    for (int a = 0; a < 4; ++a) out.material_logits[4 * ray + a] = z[8 + a];
    if (out.raw_logits) {
#pragma unroll
        for (int a = 0; a < NIF_N_OUT; ++a) out.raw_logits[NIF_N_OUT * ray + a] = z[a];
    }
    if (out.hit_position || out.hit_position_rest) {
        const float ox = ctx.origin[3 * ray], oy = ctx.origin[3 * ray + 1], oz = ctx.origin[3 * ray + 2];
        const float dx = ctx.dir[3 * ray], dy = ctx.dir[3 * ray + 1], dz = ctx.dir[3 * ray + 2];
        if (out.hit_position) {
            out.hit_position[3 * ray] = fmaf(D, dx, ox);
            out.hit_position[3 * ray + 1] = fmaf(D, dy, oy);
            out.hit_position[3 * ray + 2] = fmaf(D, dz, oz);
        }
        if (out.hit_position_rest) {
            float ix, iy, iz, ex, ey, ez;
            nif_inverse_deform(ctx.theta_max, ctx.bend_k, fmaf(t_in, dx, ox), fmaf(t_in, dy, oy), fmaf(t_in, dz, oz), ix, iy, iz);
            nif_inverse_deform(ctx.theta_max, ctx.bend_k, fmaf(t_out, dx, ox), fmaf(t_out, dy, oy), fmaf(t_out, dz, oz), ex, ey, ez);
            const float u = ell > 0.0f ? __saturatef(d / ell) : 0.0f;
            out.hit_position_rest[3 * ray] = fmaf(u, ex - ix, ix);
            out.hit_position_rest[3 * ray + 1] = fmaf(u, ey - iy, iy);
            out.hit_position_rest[3 * ray + 2] = fmaf(u, ez - iz, iz);
        }
    }
}
