// nif_traverse.cu -- step (a1): nearest deformed voxel with entry/exit parameters.
// PAPER.md:41 "trace rays directly in this domain, where rays remain straight lines. Each
// ray-voxel intersection produces a hit point"; "intersecting the ray with the occupied
// deformed voxels using a simple BVH. The first intersection point defines the starting voxel".
//
// Result definition (R9-R12): arg-min over ALL occupied voxels of
// (t_in, id), where a voxel's [t_in, t_out] comes from its exact-AABB slab interval and its 12
// triangles under a fixed fp32 operation sequence.  Every arithmetic step below is an explicit
// round-to-nearest intrinsic so that nvcc can neither contract nor reassociate it: the ids must
// be bit-exact against an independent implementation.  The hierarchy only prunes: its boxes
// nest exactly, rounding is monotone, so pruning never changes the arg-min.
#include "nif_common.cuh"

namespace {

struct Ray {
    float ox, oy, oz, dx, dy, dz, ix, iy, iz;
};

__device__ __forceinline__ void axis_interval(float lo, float hi, float o, float inv, float& tn, float& tf)
{
    float t0 = __fmul_rn(__fsub_rn(lo, o), inv);
    float t1 = __fmul_rn(__fsub_rn(hi, o), inv);
    tn = fminf(t0, t1);
    tf = fmaxf(t0, t1);
    if (t0 != t0 || t1 != t1) { tn = -INFINITY; tf = INFINITY; }   // 0*inf: ray inside a face plane
}

// slab interval of box [lo,hi]; returns hit, bn = max(tmin,0), bf = tmax
__device__ __forceinline__ bool slab(float lx, float ly, float lz, float hx, float hy, float hz,
                                     const Ray& r, float& bn, float& bf)
{
    float nx, fx, ny, fy, nz, fz;
    axis_interval(lx, hx, r.ox, r.ix, nx, fx);
    axis_interval(ly, hy, r.oy, r.iy, ny, fy);
    axis_interval(lz, hz, r.oz, r.iz, nz, fz);
    float tmin = fmaxf(fmaxf(nx, ny), nz);
    float tmax = fminf(fminf(fx, fy), fz);
    bn = fmaxf(tmin, 0.0f);
    bf = tmax;
    return (tmin <= tmax) && (tmax >= 0.0f);
}

struct V3 { float x, y, z; };

__device__ __forceinline__ V3 vsub(V3 a, V3 b)
{
    return V3{__fsub_rn(a.x, b.x), __fsub_rn(a.y, b.y), __fsub_rn(a.z, b.z)};
}
__device__ __forceinline__ V3 vcross(V3 p, V3 q)
{
    return V3{__fmaf_rn(p.y, q.z, -__fmul_rn(p.z, q.y)),
              __fmaf_rn(p.z, q.x, -__fmul_rn(p.x, q.z)),
              __fmaf_rn(p.x, q.y, -__fmul_rn(p.y, q.x))};
}
__device__ __forceinline__ float vdot(V3 p, V3 q)
{
    return __fmaf_rn(p.z, q.z, __fmaf_rn(p.y, q.y, __fmul_rn(p.x, q.x)));
}

// Moeller-Trumbore, two-sided, infinite line (R9).  Updates tlo/thi on acceptance.
__device__ __forceinline__ void tri(V3 o, V3 d, V3 v0, V3 v1, V3 v2, float& tlo, float& thi, bool& any)
{
    V3 e1 = vsub(v1, v0);
    V3 e2 = vsub(v2, v0);
    V3 pv = vcross(d, e2);
    float det = vdot(e1, pv);
    if (det == 0.0f) return;
    float inv = __fdiv_rn(1.0f, det);
    V3 sv = vsub(o, v0);
    float u = __fmul_rn(vdot(sv, pv), inv);
    V3 qv = vcross(sv, e1);
    float v = __fmul_rn(vdot(d, qv), inv);
    if (!((u >= 0.0f) && (v >= 0.0f) && (__fadd_rn(u, v) <= 1.0f))) return;
    float t = __fmul_rn(vdot(e2, qv), inv);
    if ((__float_as_uint(t) & 0x7f800000u) == 0x7f800000u) return;   // inf or NaN
    tlo = fminf(tlo, t);
    thi = fmaxf(thi, t);
    any = true;
}

// one deformed voxel: 8 lattice corners, exact AABB, slab, 12 triangles (R8-R11)
__device__ __forceinline__ bool voxel_hit(const float4* __restrict__ lat, int nv, uint32_t id,
                                          const Ray& r, float& t_in, float& t_out)
{
    const uint32_t unv = (uint32_t)nv;
    const uint32_t ix = id % unv, iy = (id / unv) % unv, iz = id / (unv * unv);
    const size_t np1 = (size_t)nv + 1;
    const float4* base = lat + (size_t)ix + np1 * ((size_t)iy + np1 * (size_t)iz);
    V3 q[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        float4 p = __ldg(base + (c & 1) + np1 * (size_t)((c >> 1) & 1) + np1 * np1 * (size_t)(c >> 2));
        q[c] = V3{p.x, p.y, p.z};
    }
    float lx = q[0].x, ly = q[0].y, lz = q[0].z, hx = lx, hy = ly, hz = lz;
#pragma unroll
    for (int c = 1; c < 8; ++c) {
        lx = fminf(lx, q[c].x); hx = fmaxf(hx, q[c].x);
        ly = fminf(ly, q[c].y); hy = fmaxf(hy, q[c].y);
        lz = fminf(lz, q[c].z); hz = fmaxf(hz, q[c].z);
    }
    float bn, bf;
    if (!slab(lx, ly, lz, hx, hy, hz, r, bn, bf)) return false;
    const V3 o{r.ox, r.oy, r.oz}, d{r.dx, r.dy, r.dz};
    float tlo = INFINITY, thi = -INFINITY;
    bool any = false;
    // face (axis a, side s): q_uv = corner with offset s on a, u on b, v on c, (b,c) cyclic after a.
    // corner index = dx + 2 dy + 4 dz.  Triangles (q00,q10,q11), (q00,q11,q01).
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        // a = x: u on y, v on z
        tri(o, d, q[s], q[s + 2], q[s + 6], tlo, thi, any);
        tri(o, d, q[s], q[s + 6], q[s + 4], tlo, thi, any);
        // a = y: u on z, v on x
        tri(o, d, q[2 * s], q[2 * s + 4], q[2 * s + 5], tlo, thi, any);
        tri(o, d, q[2 * s], q[2 * s + 5], q[2 * s + 1], tlo, thi, any);
        // a = z: u on x, v on y
        tri(o, d, q[4 * s], q[4 * s + 1], q[4 * s + 3], tlo, thi, any);
        tri(o, d, q[4 * s], q[4 * s + 3], q[4 * s + 2], tlo, thi, any);
    }
    if (!any || !(thi >= 0.0f)) return false;
    float ti = fminf(fmaxf(tlo, bn), bf);
    t_in = ti;
    t_out = fmaxf(fminf(thi, bf), ti);
    return true;
}

constexpr int TRAV_BLOCK = 128;
constexpr int STACK_MAX = 96;                 // 7 pushes per level net, <= 10 levels
constexpr uint32_t LEAF_FLAG = 0x80000000u;

__global__ void __launch_bounds__(TRAV_BLOCK)
k_traverse(const NifNode* __restrict__ nodes, const float4* __restrict__ lat, int nv, int root,
           float rlx, float rly, float rlz, float rhx, float rhy, float rhz,
           long long n, const float* __restrict__ origin, const float* __restrict__ dir,
           nif_query_out out, uint32_t* __restrict__ bin_count, uint32_t* __restrict__ rank,
           int bin_shift, int nvb, unsigned flags)
{
    const long long ray = (long long)blockIdx.x * TRAV_BLOCK + threadIdx.x;
    const bool active = ray < n;
    Ray r;
    int32_t best_id = -1;
    float best_in = INFINITY, best_out = INFINITY;
    if (active) {
        r.ox = origin[3 * ray]; r.oy = origin[3 * ray + 1]; r.oz = origin[3 * ray + 2];
        r.dx = dir[3 * ray]; r.dy = dir[3 * ray + 1]; r.dz = dir[3 * ray + 2];
        r.ix = __fdiv_rn(1.0f, r.dx); r.iy = __fdiv_rn(1.0f, r.dy); r.iz = __fdiv_rn(1.0f, r.dz);
        uint2 stack[STACK_MAX];
        int sp = 0;
        float bn, bf;
        if (root >= 0 && slab(rlx, rly, rlz, rhx, rhy, rhz, r, bn, bf)) {
            stack[sp++] = make_uint2((uint32_t)root, __float_as_uint(bn));
        }
        while (sp > 0) {
            const uint2 e = stack[--sp];
            if (__uint_as_float(e.y) > best_in) continue;          // strictly later: cannot win a tie either
            if (e.x & LEAF_FLAG) {
                const uint32_t id = e.x & ~LEAF_FLAG;
                float ti, to;
                if (voxel_hit(lat, nv, id, r, ti, to)) {
                    if (ti < best_in || (ti == best_in && (int32_t)id < best_id)) {
                        best_id = (int32_t)id; best_in = ti; best_out = to;
                    }
                }
                continue;
            }
            const NifNode* nd = nodes + e.x;
            const float4* f4 = reinterpret_cast<const float4*>(nd);
            float lo[3][8], hi[3][8];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                float4 l0 = __ldg(f4 + 2 * a), l1 = __ldg(f4 + 2 * a + 1);
                float4 h0 = __ldg(f4 + 6 + 2 * a), h1 = __ldg(f4 + 6 + 2 * a + 1);
                lo[a][0] = l0.x; lo[a][1] = l0.y; lo[a][2] = l0.z; lo[a][3] = l0.w;
                lo[a][4] = l1.x; lo[a][5] = l1.y; lo[a][6] = l1.z; lo[a][7] = l1.w;
                hi[a][0] = h0.x; hi[a][1] = h0.y; hi[a][2] = h0.z; hi[a][3] = h0.w;
                hi[a][4] = h1.x; hi[a][5] = h1.y; hi[a][6] = h1.z; hi[a][7] = h1.w;
            }
            const uint4 c0 = __ldg(reinterpret_cast<const uint4*>(nd->child));
            const uint4 c1 = __ldg(reinterpret_cast<const uint4*>(nd->child) + 1);
            const uint2 meta = __ldg(reinterpret_cast<const uint2*>(&nd->mask));
            const uint32_t child[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
            const uint32_t leaf = meta.y ? LEAF_FLAG : 0u;
            const int sp0 = sp;
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                if (!((meta.x >> c) & 1u)) continue;
                float cn, cf;
                if (slab(lo[0][c], lo[1][c], lo[2][c], hi[0][c], hi[1][c], hi[2][c], r, cn, cf) &&
                    !(cn > best_in) && sp < STACK_MAX) {
                    // insertion sort of the new entries, farthest first (nearest ends on top)
                    int p = sp++;
                    while (p > sp0 && __uint_as_float(stack[p - 1].y) < cn) { stack[p] = stack[p - 1]; --p; }
                    stack[p] = make_uint2(child[c] | leaf, __float_as_uint(cn));
                }
            }
        }
        out.voxel_id[ray] = best_id;
        out.t_in[ray] = best_in;
        out.t_out[ray] = best_out;
    }
    const bool hit = active && best_id >= 0;
    if (flags & NIF_TRAVERSE_ONLY) return;
    if (active && !hit) {                              // miss: every head output is 0 (R18)
        out.occlusion[ray] = 0.0f;
        if (!(flags & NIF_OCCLUSION_ONLY)) {
            out.distance[ray] = 0.0f; out.dist_total[ray] = 0.0f;
#pragma unroll
            for (int a = 0; a < 3; ++a) { out.normal[3 * ray + a] = 0.0f; out.albedo[3 * ray + a] = 0.0f; }
#pragma unroll
            for (int a = 0; a < 4; ++a) out.material_logits[4 * ray + a] = 0.0f;
        }
        if (out.raw_logits) {
#pragma unroll
            for (int a = 0; a < NIF_N_OUT; ++a) out.raw_logits[NIF_N_OUT * ray + a] = 0.0f;
        }
    }
    // hit rays are counted into the bin of the voxel they hit; the returned count is the ray's rank
    // inside its bin (k_bin_offsets / k_scatter_hits below turn ranks into positions in hit_list)
    if (hit) {
        const uint32_t unv = (uint32_t)nv, id = (uint32_t)best_id;
        const uint32_t ix = id % unv, iy = (id / unv) % unv, iz = id / (unv * unv);
        const uint32_t bin = (ix >> bin_shift) + (uint32_t)nvb * ((iy >> bin_shift) + (uint32_t)nvb * (iz >> bin_shift));
        rank[ray] = atomicAdd(&bin_count[bin], 1u);
    }
}

// bin_count[b] -> start of bin b in hit_list.  Each block scans 1024 consecutive bins and takes one
// contiguous range from the global cursor (scratch->n_hit): bins of a block stay in order, blocks
// land in arrival order -- enough locality for the encode kernel's tiles, no multi-pass scan.
__global__ void __launch_bounds__(1024)
k_bin_offsets(uint32_t* __restrict__ bin_count, uint32_t n_bins, NifQueryScratch* __restrict__ scratch)
{
    __shared__ uint32_t warp_sum[32];
    __shared__ unsigned long long block_base;
    const uint32_t b = blockIdx.x * 1024u + threadIdx.x;
    const uint32_t c = b < n_bins ? bin_count[b] : 0u;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t inc = c;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    if (lane == 31) warp_sum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        uint32_t v = warp_sum[lane];
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, v, d);
            if (lane >= d) v += t;
        }
        warp_sum[lane] = v;                                             // inclusive over warps
        if (lane == 31) block_base = v ? atomicAdd(&scratch->n_hit, (unsigned long long)v) : 0ull;
    }
    __syncthreads();
    if (b < n_bins) bin_count[b] = (uint32_t)block_base + (wid ? warp_sum[wid - 1] : 0u) + inc - c;
}

__global__ void __launch_bounds__(256)
k_scatter_hits(long long n, int nv, int bin_shift, int nvb, const int32_t* __restrict__ voxel_id,
               const uint32_t* __restrict__ bin_start, const uint32_t* __restrict__ rank,
               int32_t* __restrict__ hit_list)
{
    const long long ray = (long long)blockIdx.x * 256 + threadIdx.x;
    if (ray >= n) return;
    const int32_t vid = voxel_id[ray];
    if (vid < 0) return;
    const uint32_t unv = (uint32_t)nv, id = (uint32_t)vid;
    const uint32_t ix = id % unv, iy = (id / unv) % unv, iz = id / (unv * unv);
    const uint32_t bin = (ix >> bin_shift) + (uint32_t)nvb * ((iy >> bin_shift) + (uint32_t)nvb * (iz >> bin_shift));
    hit_list[bin_start[bin] + rank[ray]] = (int32_t)ray;
}

}  // namespace

int nif_launch_traverse(const nif_bvh* bvh, const nif_ray_batch* rays, const nif_query_out* out,
                        const NifQueryWs* ws, unsigned flags, cudaStream_t stream)
{
    if (rays->n == 0) return NIF_OK;
    const long long blocks = (rays->n + TRAV_BLOCK - 1) / TRAV_BLOCK;
    k_traverse<<<(unsigned)blocks, TRAV_BLOCK, 0, stream>>>(
        bvh->nodes, bvh->lattice, bvh->nv, bvh->root, bvh->lo[0], bvh->lo[1], bvh->lo[2],
        bvh->hi[0], bvh->hi[1], bvh->hi[2], (long long)rays->n, rays->origin, rays->dir, *out,
        ws->bin_count, ws->rank, ws->bin_shift, ws->nvb, flags);
    nif_count_launch(1);
    NIF_CUDA_TRY(cudaGetLastError());
    return NIF_OK;
}

int nif_launch_bin_hits(const nif_bvh* bvh, const nif_ray_batch* rays, const nif_query_out* out,
                        const NifQueryWs* ws, cudaStream_t stream)
{
    if (rays->n == 0) return NIF_OK;
    k_bin_offsets<<<(ws->n_bins + 1023u) / 1024u, 1024, 0, stream>>>(ws->bin_count, ws->n_bins, ws->scratch);
    k_scatter_hits<<<(unsigned)((rays->n + 255) / 256), 256, 0, stream>>>(
        (long long)rays->n, bvh->nv, ws->bin_shift, ws->nvb, out->voxel_id, ws->bin_count, ws->rank, ws->hit_list);
    nif_count_launch(2);
    NIF_CUDA_TRY(cudaGetLastError());
    return NIF_OK;
}
