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

// (a2) for a deformation given as a corner lattice (R27): voxel-local inverse of the trilinear
// interpolant of the voxel's 8 deformed corners, Newton from the voxel centre, NIF_NEWTON_ITERS iterations,
// Cramer's rule, fp32.  `q` = the 8 corners (c = dx + 2 dy + 4 dz).
#define NIF_NEWTON_ITERS 5
__device__ __forceinline__ void nif_load_voxel_corners(const float4* __restrict__ lat, int nv, int32_t id, float (&q)[8][3],
                                                       int (&cell)[3])
{
    const uint32_t unv = (uint32_t)nv, uid = (uint32_t)id;
    const uint32_t ix = uid % unv, iy = (uid / unv) % unv, iz = uid / (unv * unv);
    cell[0] = (int)ix; cell[1] = (int)iy; cell[2] = (int)iz;
    const size_t np1 = (size_t)nv + 1;
    const float4* base = lat + (size_t)ix + np1 * ((size_t)iy + np1 * (size_t)iz);
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const float4 v = __ldg(base + (c & 1) + np1 * (size_t)((c >> 1) & 1) + np1 * np1 * (size_t)(c >> 2));
        q[c][0] = v.x; q[c][1] = v.y; q[c][2] = v.z;
    }
}
__device__ __forceinline__ void nif_inverse_trilinear(const float (&q)[8][3], const int (&cell)[3], int nv,
                                                      float X, float Y, float Z, float& x, float& y, float& z)
{
    // Shape-function form (written independently of the oracle's nested-lerp form): T = sum_c N_c q_c with
    // N_c = a_c(u) b_c(v) g_c(w), a = (1-u, u) etc.; the Jacobian columns are sum_c (dN_c/du) q_c, ...; the
    // Newton step solves J d = P - T with the adjugate (cofactor) inverse.
    float u = 0.5f, v = 0.5f, w = 0.5f;
    for (int it = 0; it < NIF_NEWTON_ITERS; ++it) {
        const float au[2] = {1.0f - u, u}, bv[2] = {1.0f - v, v}, gw[2] = {1.0f - w, w};
        float T[3] = {0.f, 0.f, 0.f}, J[3][3] = {{0.f, 0.f, 0.f}, {0.f, 0.f, 0.f}, {0.f, 0.f, 0.f}};   // J[row = axis][col = u,v,w]
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const int i = c & 1, j = (c >> 1) & 1, k = c >> 2;
            const float n = au[i] * bv[j] * gw[k];
            const float du = (i ? 1.0f : -1.0f) * bv[j] * gw[k];
            const float dv = au[i] * (j ? 1.0f : -1.0f) * gw[k];
            const float dw = au[i] * bv[j] * (k ? 1.0f : -1.0f);
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                T[a] = fmaf(n, q[c][a], T[a]);
                J[a][0] = fmaf(du, q[c][a], J[a][0]); J[a][1] = fmaf(dv, q[c][a], J[a][1]); J[a][2] = fmaf(dw, q[c][a], J[a][2]);
            }
        }
        const float r0 = X - T[0], r1 = Y - T[1], r2 = Z - T[2];
        // cofactors of J
        const float c00 = J[1][1] * J[2][2] - J[1][2] * J[2][1], c01 = J[1][2] * J[2][0] - J[1][0] * J[2][2], c02 = J[1][0] * J[2][1] - J[1][1] * J[2][0];
        const float det = J[0][0] * c00 + J[0][1] * c01 + J[0][2] * c02;
        if (det == 0.0f) break;
        const float c10 = J[0][2] * J[2][1] - J[0][1] * J[2][2], c11 = J[0][0] * J[2][2] - J[0][2] * J[2][0], c12 = J[0][1] * J[2][0] - J[0][0] * J[2][1];
        const float c20 = J[0][1] * J[1][2] - J[0][2] * J[1][1], c21 = J[0][2] * J[1][0] - J[0][0] * J[1][2], c22 = J[0][0] * J[1][1] - J[0][1] * J[1][0];
        const float inv = 1.0f / det;
        // d = J^-1 r = adj(J) r / det, adj(J)[i][j] = cofactor[j][i]
        u += (c00 * r0 + c10 * r1 + c20 * r2) * inv;
        v += (c01 * r0 + c11 * r1 + c21 * r2) * inv;
        w += (c02 * r0 + c12 * r1 + c22 * r2) * inv;
    }
    const float fnv = (float)nv;
    x = (2.0f * ((float)cell[0] + u) - fnv) / fnv;
    y = (2.0f * ((float)cell[1] + v) - fnv) / fnv;
    z = (2.0f * ((float)cell[2] + w) - fnv) / fnv;
}

// what step (a2) needs: the closed-form pose, or the lattice for the voxel-local inverse
struct NifMapCtx {
    float theta_max, bend_k;
    const float4* lat;        // deformed corner lattice
    int nv;
    int local;                // 1: the BVH was built from a user lattice -> voxel-local inverse (R27)
};

// nif_query_poses: the pose of this ray (closed-form parameters, or its lattice) replaces the batch-wide one
__device__ __forceinline__ NifMapCtx nif_ray_map(const NifMapCtx& base, const NifPoseBatch& b, long long ray)
{
    NifMapCtx m = base;
    if (b.pose_id) {
        const NifPoseDesc* pd = b.poses + b.pose_id[ray];
        m.theta_max = pd->theta_max; m.bend_k = pd->bend_k; m.lat = pd->lat;
    }
    return m;
}

// rest images of a ray's entry and exit points (both lie in voxel `vid`)
template <bool LOCAL>
__device__ __forceinline__ void nif_map_back_pair(const NifMapCtx& m, int32_t vid, const float* __restrict__ o,
                                                  const float* __restrict__ d, float t_in, float t_out, float (&ri)[3], float (&ro)[3])
{
    const float Xi = fmaf(t_in, d[0], o[0]), Yi = fmaf(t_in, d[1], o[1]), Zi = fmaf(t_in, d[2], o[2]);
    const float Xo = fmaf(t_out, d[0], o[0]), Yo = fmaf(t_out, d[1], o[1]), Zo = fmaf(t_out, d[2], o[2]);
    if constexpr (LOCAL) {
        float q[8][3]; int cell[3];
        nif_load_voxel_corners(m.lat, m.nv, vid, q, cell);
        nif_inverse_trilinear(q, cell, m.nv, Xi, Yi, Zi, ri[0], ri[1], ri[2]);
        nif_inverse_trilinear(q, cell, m.nv, Xo, Yo, Zo, ro[0], ro[1], ro[2]);
    } else {
        nif_inverse_deform(m.theta_max, m.bend_k, Xi, Yi, Zi, ri[0], ri[1], ri[2]);
        nif_inverse_deform(m.theta_max, m.bend_k, Xo, Yo, Zo, ro[0], ro[1], ro[2]);
    }
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
    NifMapCtx map;
    NifPoseBatch batch;
};

template <bool LOCAL>
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
            const float oo[3] = {ox, oy, oz}, dd[3] = {dx, dy, dz};
            float ri[3], ro[3];
            nif_map_back_pair<LOCAL>(nif_ray_map(ctx.map, ctx.batch, ray), LOCAL ? out.voxel_id[ray] : 0, oo, dd, t_in, t_out, ri, ro);
            const float u = ell > 0.0f ? __saturatef(d / ell) : 0.0f;
            out.hit_position_rest[3 * ray] = fmaf(u, ro[0] - ri[0], ri[0]);
            out.hit_position_rest[3 * ray + 1] = fmaf(u, ro[1] - ri[1], ri[1]);
            out.hit_position_rest[3 * ray + 2] = fmaf(u, ro[2] - ri[2], ri[2]);
        }
    }
}
