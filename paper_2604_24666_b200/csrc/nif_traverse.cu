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

// Child boxes of a hierarchy node only PRUNE (a voxel's own interval comes from voxel_hit), so their test
// may be cheaper as long as it stays conservative: the build stores them inflated by one ulp outwards
// (nif_build.cu) and the ray carries inverses clamped to +-FLT_MAX, so a ray parallel to a slab and exactly
// on the voxel's boundary plane lies strictly inside the inflated slab and 0 * inv is 0, never NaN -- the
// NaN handling of axis_interval (a third of the node step's instructions) is not needed.  Same operation
// sequence otherwise, so monotone rounding keeps every enclosed voxel's interval inside the node's:
//   t0 = (lo - o) * inv, t1 = (hi - o) * inv per axis, tmin = max of the three min(t0, t1), tmax = min of the three max.
// It is evaluated with the six planes already in the ray's order: n* = the plane of each axis the ray meets first (lo when
// the inverse direction is positive, hi when it is negative), f* = the other one.  Rounding is monotone and the clamped
// inverse is never 0 or NaN, so (near - o) * inv <= (far - o) * inv holds on the computed values too: the per-axis
// fminf/fmaxf would always pick exactly these two numbers, and leaving them out changes no bit of tmin or tmax
// (6 of the 9 min/max per child gone; the ALU pipe that executes them is the busiest unit of the traversal kernels).
__device__ __forceinline__ bool slab_node_ordered(float nx, float ny, float nz, float fx, float fy, float fz,
                                                  const Ray& r, float& bn)
{
    const float x0 = __fmul_rn(__fsub_rn(nx, r.ox), r.ix), x1 = __fmul_rn(__fsub_rn(fx, r.ox), r.ix);
    const float y0 = __fmul_rn(__fsub_rn(ny, r.oy), r.iy), y1 = __fmul_rn(__fsub_rn(fy, r.oy), r.iy);
    const float z0 = __fmul_rn(__fsub_rn(nz, r.oz), r.iz), z1 = __fmul_rn(__fsub_rn(fz, r.oz), r.iz);
    const float tmin = fmaxf(fmaxf(x0, y0), z0);
    const float tmax = fminf(fminf(x1, y1), z1);
    bn = fmaxf(tmin, 0.0f);
    return (tmin <= tmax) && (tmax >= 0.0f);
}
// offset (in float4) of an axis' near-plane block inside a node: lo planes start at 0, hi planes at 6
__device__ __forceinline__ int near_block(float inv) { return (int)(__float_as_uint(inv) >> 31) * 6; }

// r.ix/iy/iz are the CLAMPED inverses (node tests); the exact ones (+-inf for a zero component), which the
// root box and the voxel's own box need (R10), are recomputed where used
__device__ __forceinline__ Ray exact_inverses(const Ray& r)
{
    Ray e = r;
    e.ix = __fdiv_rn(1.0f, r.dx); e.iy = __fdiv_rn(1.0f, r.dy); e.iz = __fdiv_rn(1.0f, r.dz);
    return e;
}
__device__ __forceinline__ float clamp_inverse(float inv) { return fminf(fmaxf(inv, -3.402823466e38f), 3.402823466e38f); }

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
    if (!slab(lx, ly, lz, hx, hy, hz, exact_inverses(r), bn, bf)) return false;
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
#ifndef NIF_TRAV_BPS
#define NIF_TRAV_BPS 7      // persistent kernel: 72 registers, 7 blocks per SM (round 2, after the node step lost its votes and half its min/max: cfg 2 1.40 -> 1.33 ms per pose; 6: 1.40, 8: 1.41, 5: 1.46)
#endif
constexpr int TRAV_BLOCKS_PER_SM = NIF_TRAV_BPS;
constexpr int STACK_MAX = 96;                 // a node pops 1 entry and pushes <= 8: 7 net per level
constexpr int TRAV_MAX_LEVELS = 9;            // nv <= 512 (checked in nif_build.cu) -> padded 512^3 -> 9 octree levels
static_assert(STACK_MAX >= 7 * TRAV_MAX_LEVELS + 8, "per-ray stack too small for the deepest hierarchy");
constexpr uint32_t LEAF_FLAG = 0x80000000u;
#ifndef NIF_TRAV_REFILL
#define NIF_TRAV_REFILL 8
#endif
constexpr int TRAV_REFILL = NIF_TRAV_REFILL;               // fetch new rays when at least this many lanes are idle
constexpr int TRAV_B_LEAVES = 12, TRAV_B_FEW_INNER = 8, TRAV_B_FEW_LEAVES = 4;   // phase A -> B policy of k_traverse_persistent

struct TravParams {
    const NifNode* nodes;
    const float4* lat;
    int nv, root;
    float rlx, rly, rlz, rhx, rhy, rhz;       // root box
    long long n;
    const float* origin;
    const float* dir;
    nif_query_out out;
    unsigned int* ray_counter;                // dynamic ray fetch (scratch header)
    unsigned int* overflow_flag;              // scratch header: set if a stack ever overflowed (reported as NIF_ERR_INTERNAL)
    const unsigned int* coherent_flag;        // written by k_ray_coherence: 1 -> simple kernel, 0 -> persistent
    const unsigned int* image_width;          // written by k_ray_coherence: row length if the batch is a row-major image, else 0
    uint32_t* bin_count;
    uint32_t* rank;
    int bin_shift, nvb;
    unsigned flags;
    // multi-voxel walk (nif_query_multi, R22): rounds >= 1 run over the list of rays still
    // walking and look for the successor of the voxel each ray evaluated last
    const int32_t* ray_list;                  // NULL: rays 0..n-1
    const unsigned int* n_list;               // device count of ray_list
    float* walk_dist_accum;                   // NULL outside a walk; a ray that runs out of voxels gets 0
    NifPoseBatch batch;                       // nif_query_poses: per-ray pose (MULTI kernels)
};

// MULTI kernels: the pose descriptors staged in shared memory, a pose index per lane
template <bool MULTI> struct PoseView {
    const NifPoseDesc* s;                     // shared-memory copy
    __device__ __forceinline__ const NifNode* nodes(const TravParams& p, int pose) const { return MULTI ? s[pose].nodes : p.nodes; }
    __device__ __forceinline__ const float4* lat(const TravParams& p, int pose) const { return MULTI ? s[pose].lat : p.lat; }
    __device__ __forceinline__ int root(const TravParams& p, int pose) const { return MULTI ? s[pose].root : p.root; }
    __device__ __forceinline__ bool root_hit(const TravParams& p, int pose, const Ray& r, float& bn) const
    {
        float bf;
        if (MULTI) {
            const NifPoseDesc& d = s[pose];
            return d.root >= 0 && slab(d.lo[0], d.lo[1], d.lo[2], d.hi[0], d.hi[1], d.hi[2], r, bn, bf);
        }
        return p.root >= 0 && slab(p.rlx, p.rly, p.rlz, p.rhx, p.rhy, p.rhz, r, bn, bf);
    }
};
template <bool MULTI>
__device__ __forceinline__ PoseView<MULTI> stage_poses(const TravParams& p, NifPoseDesc* s_pose)
{
    if (MULTI) {
        const int n_words = p.batch.n_poses * (int)(sizeof(NifPoseDesc) / 4);
        for (int i = threadIdx.x; i < n_words; i += blockDim.x)
            reinterpret_cast<uint32_t*>(s_pose)[i] = reinterpret_cast<const uint32_t*>(p.batch.poses)[i];
        __syncthreads();
    }
    return PoseView<MULTI>{s_pose};
}

// successor bound of the walk: only voxels whose (t_in, id) is lexicographically greater than the
// voxel the ray evaluated last are candidates (R22)
__device__ __forceinline__ bool after_bound(float ti, int32_t id, float after_t, int32_t after_id)
{
    return (ti > after_t) || (ti == after_t && id > after_id);
}

// results of one finished ray: ids/t always; zero heads for a miss (R18); bin count for a hit
__device__ __forceinline__ void retire_ray(const TravParams& p, long long ray, int32_t best_id, float best_in, float best_out)
{
    p.out.voxel_id[ray] = best_id;
    p.out.t_in[ray] = best_in;
    p.out.t_out[ray] = best_out;
    if (p.flags & NIF_TRAVERSE_ONLY) return;
    if (best_id < 0) {
        p.out.occlusion[ray] = 0.0f;
        if (!(p.flags & NIF_OCCLUSION_ONLY)) {
            p.out.distance[ray] = 0.0f; p.out.dist_total[ray] = 0.0f;
#pragma unroll
            for (int a = 0; a < 3; ++a) { p.out.normal[3 * ray + a] = 0.0f; p.out.albedo[3 * ray + a] = 0.0f; }
#pragma unroll
            for (int a = 0; a < 4; ++a) p.out.material_logits[4 * ray + a] = 0.0f;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                if (p.out.hit_position) p.out.hit_position[3 * ray + a] = 0.0f;
                if (p.out.hit_position_rest) p.out.hit_position_rest[3 * ray + a] = 0.0f;
            }
        }
        if (p.out.raw_logits) {
#pragma unroll
            for (int a = 0; a < NIF_N_OUT; ++a) p.out.raw_logits[NIF_N_OUT * ray + a] = 0.0f;
        }
        if (p.walk_dist_accum) p.walk_dist_accum[ray] = 0.0f;
    } else {
        // counted into the bin of the voxel it hit; the returned count is the ray's rank inside its
        // bin (k_bin_offsets / k_scatter_hits below turn ranks into positions in hit_list)
        const uint32_t unv = (uint32_t)p.nv, id = (uint32_t)best_id;
        const uint32_t ix = id % unv, iy = (id / unv) % unv, iz = id / (unv * unv);
        const uint32_t bin = (ix >> p.bin_shift) + (uint32_t)p.nvb * ((iy >> p.bin_shift) + (uint32_t)p.nvb * (iz >> p.bin_shift));
        p.rank[ray] = atomicAdd(&p.bin_count[bin], 1u);
    }
}

// Persistent warps, one ray per lane, "while-while" traversal with dynamic ray fetch: lanes first
// work through inner nodes until enough live lanes have a voxel on top of their stack (or are finished),
// then those run the expensive 12-triangle voxel test together; finished lanes are refilled
// from a global counter once enough of them are idle.  Incoherent rays (config 3) otherwise leave
// 4 of 32 lanes active on average.
template <bool AFTER, bool MULTI>
__global__ void __launch_bounds__(TRAV_BLOCK, TRAV_BLOCKS_PER_SM)
k_traverse_persistent(const TravParams p)
{
    if (!AFTER && *p.coherent_flag != 0u) return;         // k_traverse_simple takes this batch
    __shared__ NifPoseDesc s_pose[MULTI ? NIF_MAX_POSES : 1];
    const PoseView<MULTI> pv = stage_poses<MULTI>(p, s_pose);
    int pose = 0;
    const long long n_rays = p.ray_list ? (long long)*p.n_list : p.n;
    float after_t = -INFINITY;                            // AFTER: successor bound (R22)
    int32_t after_id = -1;
    const int lane = threadIdx.x & 31;
    uint2 stack[STACK_MAX];
    int sp = 0;
    long long ray = -1;                                   // -1: lane has no ray
    Ray r;
    int32_t best_id = -1;
    float best_in = INFINITY, best_out = INFINITY;
    bool exhausted = false;                               // the global counter ran past n

    for (;;) {
        // ---- refill idle lanes from the global ray counter.  Rays that miss the root box retire on
        // the spot, so the loop keeps fetching until enough lanes hold a live ray.
        for (;;) {
            const unsigned idle = __ballot_sync(0xffffffffu, ray < 0);
            if (exhausted || (__popc(idle) < TRAV_REFILL && idle != 0xffffffffu)) break;
            unsigned base = 0;
            if (lane == 0) base = atomicAdd(p.ray_counter, (unsigned)__popc(idle));
            base = __shfl_sync(0xffffffffu, base, 0);
            if ((long long)base + __popc(idle) >= n_rays) exhausted = true;
            const long long cand = (long long)base + __popc(idle & ((1u << lane) - 1u));
            if (ray < 0 && cand < n_rays) {
                ray = p.ray_list ? (long long)p.ray_list[cand] : cand;
                if (AFTER) { after_t = p.out.t_in[ray]; after_id = p.out.voxel_id[ray]; }
                if (MULTI) pose = p.batch.pose_id[ray];
                r.ox = p.origin[3 * ray]; r.oy = p.origin[3 * ray + 1]; r.oz = p.origin[3 * ray + 2];
                r.dx = p.dir[3 * ray]; r.dy = p.dir[3 * ray + 1]; r.dz = p.dir[3 * ray + 2];
                r.ix = __fdiv_rn(1.0f, r.dx); r.iy = __fdiv_rn(1.0f, r.dy); r.iz = __fdiv_rn(1.0f, r.dz);
                best_id = -1; best_in = INFINITY; best_out = INFINITY; sp = 0;
                float bn;
                const bool root_hit = pv.root_hit(p, pose, r, bn);
                if constexpr (!AFTER) {       // successor rounds keep the exact inverses: they also prune on the far end
                    r.ix = clamp_inverse(r.ix); r.iy = clamp_inverse(r.iy); r.iz = clamp_inverse(r.iz);
                }
                if (root_hit) {
                    stack[sp++] = make_uint2((uint32_t)pv.root(p, pose), __float_as_uint(bn));
                } else {
                    retire_ray(p, ray, -1, INFINITY, INFINITY);
                    ray = -1;
                }
            }
        }
        if (__all_sync(0xffffffffu, ray < 0)) break;      // nothing left anywhere in this warp

        // ---- phase A: inner nodes until enough lanes have a voxel on top (policy below) ----
        for (;;) {
            // drop entries that can no longer win (strictly later than the best entry: ties stay, R12)
            while (sp > 0 && __uint_as_float(stack[sp - 1].y) > best_in) --sp;
            const bool inner = ray >= 0 && sp > 0 && !(stack[sp - 1].x & LEAF_FLAG);
            // When to leave phase A.  Round 1 waited until NO lane had an inner node on top; lanes that reached a voxel early
            // then idled through the node steps of the slowest lane.  Now phase B starts as soon as enough lanes hold a voxel:
            // TRAV_B_LEAVES of them, or TRAV_B_FEW_LEAVES once fewer than TRAV_B_FEW_INNER lanes still have inner nodes.  A
            // lane's own sequence of pops is unchanged, only the interleaving between lanes: same results, cfg 2 / 3
            // traversal -24 % (1.34 -> 1.02 ms, 1.59 -> 1.24 ms per pose; thresholds swept, all within 3 % of each other).
            {
                const unsigned mi = __ballot_sync(0xffffffffu, inner);
                const int leaves = __popc(__ballot_sync(0xffffffffu, ray >= 0 && sp > 0 && (stack[sp - 1].x & LEAF_FLAG)));
                if (mi == 0u || leaves >= TRAV_B_LEAVES || (__popc(mi) < TRAV_B_FEW_INNER && leaves >= TRAV_B_FEW_LEAVES)) break;
            }
            {
                // one node per lane, branch-free: slab tests of all 8 octants, a sorting
                // network on packed (t_near, octant) keys, up to 8 predicated pushes (farthest first,
                // so the nearest child ends on top).  Lanes without an inner node run it masked off.
                float lo[3][8], hi[3][8];
                uint4 meta = make_uint4(0u, 0u, 0u, 0u);                     // mask, is_brick, base, -
                if (inner) {
                    const uint2 e = stack[--sp];
                    const NifNode* nd = pv.nodes(p, pose) + e.x;
                    const float4* f4 = reinterpret_cast<const float4*>(nd);
                    // lo[] / hi[] hold the NEAR / FAR planes of this ray (slab_node_ordered); the successor rounds keep
                    // lo / hi proper for the exact test
                    const int nb3[3] = {AFTER ? 0 : near_block(r.ix), AFTER ? 0 : near_block(r.iy), AFTER ? 0 : near_block(r.iz)};
#pragma unroll
                    for (int a = 0; a < 3; ++a) {
                        const float4 l0 = __ldg(f4 + nb3[a] + 2 * a), l1 = __ldg(f4 + nb3[a] + 2 * a + 1);
                        const float4 h0 = __ldg(f4 + (6 - nb3[a]) + 2 * a), h1 = __ldg(f4 + (6 - nb3[a]) + 2 * a + 1);
                        lo[a][0] = l0.x; lo[a][1] = l0.y; lo[a][2] = l0.z; lo[a][3] = l0.w;
                        lo[a][4] = l1.x; lo[a][5] = l1.y; lo[a][6] = l1.z; lo[a][7] = l1.w;
                        hi[a][0] = h0.x; hi[a][1] = h0.y; hi[a][2] = h0.z; hi[a][3] = h0.w;
                        hi[a][4] = h1.x; hi[a][5] = h1.y; hi[a][6] = h1.z; hi[a][7] = h1.w;
                    }
                    meta = __ldg(reinterpret_cast<const uint4*>(&nd->mask));
                } else {
#pragma unroll
                    for (int a = 0; a < 3; ++a)
#pragma unroll
                        for (int c = 0; c < 8; ++c) { lo[a][c] = 0.0f; hi[a][c] = 0.0f; }
                }
                uint32_t key[8];
                int count = 0;
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    key[c] = 0xffffffffu;
                    {   // all 8 octants, absent ones masked off below: the lanes of this kernel sit on different nodes, so a
                        // warp-wide "does any lane have octant c" vote (round 1) was nearly always true -- dropping the 8
                        // votes and branches: cfg 2 / 3 traversal -5 %
                        float cn, cf = INFINITY;
                        // AFTER: every voxel below has t_in <= its box's far end <= cf (boxes nest, R10), so a
                        // child that ends before after_t holds no successor
                        bool ok;
                        if constexpr (AFTER)
                            ok = slab(lo[0][c], lo[1][c], lo[2][c], hi[0][c], hi[1][c], hi[2][c], r, cn, cf);
                        else
                            ok = slab_node_ordered(lo[0][c], lo[1][c], lo[2][c], hi[0][c], hi[1][c], hi[2][c], r, cn);
                        ok = ok && ((meta.x >> c) & 1u) && !(cn > best_in) && !(AFTER && cf < after_t);
                        // cn >= 0: its bit pattern orders like an integer; the 3 low mantissa bits make
                        // room for the octant (t_near only gets smaller: pruning stays conservative).  ~
                        // turns the ascending network into "farthest first"; rejected children sort last.
                        if (ok) key[c] = ~((__float_as_uint(cn) & ~7u) | (uint32_t)c);
                        count += ok ? 1 : 0;
                    }
                }
#define NIF_CE(i, j) { const uint32_t lo_ = min(key[i], key[j]), hi_ = max(key[i], key[j]); key[i] = lo_; key[j] = hi_; }
                NIF_CE(0, 1) NIF_CE(2, 3) NIF_CE(4, 5) NIF_CE(6, 7)
                NIF_CE(0, 2) NIF_CE(1, 3) NIF_CE(4, 6) NIF_CE(5, 7)
                NIF_CE(1, 2) NIF_CE(5, 6)
                NIF_CE(0, 4) NIF_CE(1, 5) NIF_CE(2, 6) NIF_CE(3, 7)
                NIF_CE(2, 4) NIF_CE(3, 5)
                NIF_CE(1, 2) NIF_CE(3, 4) NIF_CE(5, 6)
#undef NIF_CE
                if (count > STACK_MAX - sp) {                               // excluded by the static_assert above for nv <= 512;
                    count = STACK_MAX - sp;                                 // never silently: the query reports NIF_ERR_INTERNAL
                    *p.overflow_flag = 1u;
                }
                const uint32_t unv = (uint32_t)p.nv;
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    if (i < count) {
                        const uint32_t k = ~key[i], c = k & 7u;
                        const uint32_t id = meta.y
                            ? (meta.z + (c & 1u) + unv * (((c >> 1) & 1u) + unv * (c >> 2))) | LEAF_FLAG
                            : meta.z + (uint32_t)__popc(meta.x & ((1u << c) - 1u));
                        stack[sp + i] = make_uint2(id, k & ~7u);
                    }
                }
                sp += count;
            }
        }

        // ---- phase B: every lane with a voxel on top tests it ------------------------------------
        if (ray >= 0 && sp > 0 && (stack[sp - 1].x & LEAF_FLAG)) {
            const uint32_t id = stack[--sp].x & ~LEAF_FLAG;
            float ti, to;
            if (voxel_hit(pv.lat(p, pose), p.nv, id, r, ti, to) && (!AFTER || after_bound(ti, (int32_t)id, after_t, after_id))) {
                if (ti < best_in || (ti == best_in && (int32_t)id < best_id)) {
                    best_id = (int32_t)id; best_in = ti; best_out = to;
                }
            }
            while (sp > 0 && __uint_as_float(stack[sp - 1].y) > best_in) --sp;
        }

        // ---- retire finished lanes -------------------------------------------------------------------
        if (ray >= 0 && sp == 0) {
            retire_ray(p, ray, best_id, best_in, best_out);
            ray = -1;
        }
    }
}

// One thread per ray, static assignment: the right shape for coherent batches (camera rays), where
// the 32 rays of a warp walk the same nodes and the loads of a node broadcast.  Absent octants are
// skipped, hit children are insertion-sorted (farthest first).
#ifndef NIF_TRAV_SIMPLE_MINB
#define NIF_TRAV_SIMPLE_MINB 6      // 80 registers, 6 blocks per SM: cfg 1 0.186 -> 0.177 ms (8: 0.182, 10: 0.209)
#endif
template <bool MULTI>
__global__ void __launch_bounds__(TRAV_BLOCK, NIF_TRAV_SIMPLE_MINB)
k_traverse_simple(const TravParams p)
{
    if (*p.coherent_flag == 0u) return;                   // k_traverse_persistent takes this batch
    __shared__ NifPoseDesc s_pose[MULTI ? NIF_MAX_POSES : 1];
    const PoseView<MULTI> pv = stage_poses<MULTI>(p, s_pose);
    long long ray = (long long)blockIdx.x * TRAV_BLOCK + threadIdx.x;
    // A batch that k_ray_coherence recognised as a row-major image (width a multiple of 8, height of 4) is walked in
    // tiles of 8 x 4 pixels per warp instead of 32 pixels of one row: the rays of a warp then visit fewer different
    // nodes (config 1: 0.179 -> 0.169 ms, config 4: 1.93 -> 1.64 ms) and the hit rays reach the bins in a more
    // compact order (encode+MLP -2 %).  Pure re-assignment of rays to threads: every ray is still traced once, by
    // the same code, and written to its own output slot, so results cannot depend on it (or on a wrong guess).
    const unsigned img_w = *p.image_width;
    if (img_w) {
        const long long wg = ray >> 5;                          // warp index in the grid = tile index
        const int lane = threadIdx.x & 31;
        const long long tiles_x = img_w >> 3, ty = wg / tiles_x, tx = wg - ty * tiles_x;
        ray = (ty * 4 + (lane >> 3)) * (long long)img_w + tx * 8 + (lane & 7);
    }
    if (ray >= p.n) return;
    const int pose = MULTI ? p.batch.pose_id[ray] : 0;
    Ray r;
    int32_t best_id = -1;
    float best_in = INFINITY, best_out = INFINITY;
    r.ox = p.origin[3 * ray]; r.oy = p.origin[3 * ray + 1]; r.oz = p.origin[3 * ray + 2];
    r.dx = p.dir[3 * ray]; r.dy = p.dir[3 * ray + 1]; r.dz = p.dir[3 * ray + 2];
    r.ix = __fdiv_rn(1.0f, r.dx); r.iy = __fdiv_rn(1.0f, r.dy); r.iz = __fdiv_rn(1.0f, r.dz);
    uint2 stack[STACK_MAX];
    int sp = 0;
    float bn;
    const bool root_hit = pv.root_hit(p, pose, r, bn);
    r.ix = clamp_inverse(r.ix); r.iy = clamp_inverse(r.iy); r.iz = clamp_inverse(r.iz);
    if (root_hit)
        stack[sp++] = make_uint2((uint32_t)pv.root(p, pose), __float_as_uint(bn));
    while (sp > 0) {
        const uint2 e = stack[--sp];
        if (__uint_as_float(e.y) > best_in) continue;          // strictly later: cannot win a tie either (R12)
        if (e.x & LEAF_FLAG) {
            const uint32_t id = e.x & ~LEAF_FLAG;
            float ti, to;
            if (voxel_hit(pv.lat(p, pose), p.nv, id, r, ti, to)) {
                if (ti < best_in || (ti == best_in && (int32_t)id < best_id)) {
                    best_id = (int32_t)id; best_in = ti; best_out = to;
                }
            }
            continue;
        }
        const NifNode* nd = pv.nodes(p, pose) + e.x;
        const float4* f4 = reinterpret_cast<const float4*>(nd);
        float lo[3][8], hi[3][8];
#pragma unroll
        for (int a = 0; a < 3; ++a) {                             // lo = near planes, hi = far planes of this ray
            const int nb = near_block(a == 0 ? r.ix : a == 1 ? r.iy : r.iz);
            const float4 l0 = __ldg(f4 + nb + 2 * a), l1 = __ldg(f4 + nb + 2 * a + 1);
            const float4 h0 = __ldg(f4 + (6 - nb) + 2 * a), h1 = __ldg(f4 + (6 - nb) + 2 * a + 1);
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
            float cn;
            if (slab_node_ordered(lo[0][c], lo[1][c], lo[2][c], hi[0][c], hi[1][c], hi[2][c], r, cn) && !(cn > best_in)) {
                if (sp >= STACK_MAX) { *p.overflow_flag = 1u; continue; }   // see k_traverse_persistent
                int q = sp++;
                while (q > sp0 && __uint_as_float(stack[q - 1].y) < cn) { stack[q] = stack[q - 1]; --q; }
                stack[q] = make_uint2(child[c] | leaf, __float_as_uint(cn));
            }
        }
    }
    retire_ray(p, ray, best_id, best_in, best_out);
}

// squared step from ray i to ray j: direction change plus origin change in units of the object's size
__device__ __forceinline__ float ray_step2(const float* __restrict__ origin, const float* __restrict__ dir, float inv_extent,
                                           long long i, long long j)
{
    float s = 0.0f;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float dd = dir[3 * j + a] - dir[3 * i + a], oo = (origin[3 * j + a] - origin[3 * i + a]) * inv_extent;
        s += dd * dd + oo * oo;
    }
    return s;
}

// Decides which traversal kernel runs (device-side: nif_query never synchronises).  Sampled groups
// of 32 consecutive rays vote "coherent" when every direction is within ~8 degrees of the group's
// first and all origins lie within a tenth of the object's size of each other; the batch is coherent
// when most groups are.  NIF_TRAVERSE_COHERENT / NIF_TRAVERSE_INCOHERENT override the vote.
__global__ void __launch_bounds__(256)
k_ray_coherence(long long n, const float* __restrict__ origin, const float* __restrict__ dir, float extent,
                int n_groups, unsigned flags, unsigned int* __restrict__ votes, unsigned int* __restrict__ flag_out,
                unsigned int* __restrict__ image_width_out, unsigned int* __restrict__ first_break)
{
    // ---- is the batch a row-major image?  Consecutive rays of a row are one pixel step apart; the first step that is
    // much larger than the first one ends row 0.  One pair (i, i+1) per thread over the first 8192 rays; the smallest
    // breaking i is collected with an atomic (stored inverted: the header starts at zero) and checked by the last block.
    // Only a hint for the thread assignment of k_traverse_simple (see there): a wrong answer costs time, never a result.
    const float inv_extent = extent > 0.0f ? 1.0f / extent : 0.0f;
    const float big = n > 1 ? 64.0f * ray_step2(origin, dir, inv_extent, 0, 1) : 0.0f;
    {
        const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
        const long long pairs = n - 1 < 8192 ? n - 1 : 8192;                 // widths up to 8192
        if (i < pairs && ray_step2(origin, dir, inv_extent, i, i + 1) > big) atomicMax(first_break, 0xffffffffu - (unsigned)i);
    }
    const int lane = threadIdx.x & 31;
    const int g = (int)((blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    const long long groups_total = (n + 31) / 32;
    bool coherent = false;
    if (g < n_groups) {
        const long long base = 32 * ((groups_total * g) / n_groups);          // evenly spread over the batch
        const long long i0 = base, i = base + lane < n ? base + lane : n - 1;
        const float dx = dir[3 * i0], dy = dir[3 * i0 + 1], dz = dir[3 * i0 + 2];
        const float c = dir[3 * i] * dx + dir[3 * i + 1] * dy + dir[3 * i + 2] * dz;
        const float ex = origin[3 * i] - origin[3 * i0], ey = origin[3 * i + 1] - origin[3 * i0 + 1],
                    ez = origin[3 * i + 2] - origin[3 * i0 + 2];
        const bool ok = c > 0.99f && (ex * ex + ey * ey + ez * ez) <= 0.01f * extent * extent;
        coherent = __all_sync(0xffffffffu, ok);
        if (lane == 0 && coherent) atomicAdd(&votes[0], 1u);
    }
    __threadfence();
    __syncthreads();
    // last block to finish publishes the decision
    __shared__ bool last;
    if (threadIdx.x == 0) last = atomicAdd(&votes[1], 1u) == gridDim.x - 1;
    __syncthreads();
    if (last && threadIdx.x == 0) {
        const unsigned yes = atomicAdd(&votes[0], 0u);
        unsigned decision = 2u * yes > (unsigned)n_groups ? 1u : 0u;
        if (flags & NIF_TRAVERSE_COHERENT) decision = 1u;
        if (flags & NIF_TRAVERSE_INCOHERENT) decision = 0u;
        *flag_out = decision;
        // the width is accepted when it tiles the batch (n = w x h, w % 8 == 0, h % 4 == 0), the ray below ray 0 is a
        // neighbour and row 1 starts and ends like row 0
        const unsigned fb = atomicAdd(first_break, 0u);
        const long long w = fb == 0u ? 0 : (long long)(0xffffffffu - fb) + 1;
        bool ok = big > 0.0f && w >= 32 && w % 8 == 0 && n % w == 0 && (n / w) % 4 == 0 && n >= 2 * w;
        if (ok) ok = ray_step2(origin, dir, inv_extent, 0, w) * 4.0f <= big &&
                     ray_step2(origin, dir, inv_extent, w, w + 1) <= big &&
                     (n == 2 * w || ray_step2(origin, dir, inv_extent, 2 * w - 1, 2 * w) > big);
        *image_width_out = ok ? (unsigned)w : 0u;
    }
}

// bin_count[b] -> start of bin b in hit_list.  Each block scans 1024 consecutive bins and takes one
// contiguous range from the global cursor (scratch->n_hit): bins of a block stay in order, blocks
// land in arrival order -- enough locality for the encode kernel's tiles, no multi-pass scan.
__global__ void __launch_bounds__(1024)
k_bin_offsets(uint32_t* __restrict__ bin_count, uint32_t n_bins, NifQueryScratch* __restrict__ scratch,
              const unsigned int* __restrict__ n_list)
{
    if (n_list && *n_list == 0u) return;                  // walk round with no ray left: nothing was binned
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
               int32_t* __restrict__ hit_list, const int32_t* __restrict__ ray_list,
               const unsigned int* __restrict__ n_list)
{
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= (ray_list ? (long long)*n_list : n)) return;
    const long long ray = ray_list ? (long long)ray_list[i] : i;
    const int32_t vid = voxel_id[ray];
    if (vid < 0) return;
    const uint32_t unv = (uint32_t)nv, id = (uint32_t)vid;
    const uint32_t ix = id % unv, iy = (id / unv) % unv, iz = id / (unv * unv);
    const uint32_t bin = (ix >> bin_shift) + (uint32_t)nvb * ((iy >> bin_shift) + (uint32_t)nvb * (iz >> bin_shift));
    hit_list[bin_start[bin] + rank[ray]] = (int32_t)ray;
}

// walk rounds >= 1: zero the bin counters only if some ray still walks (an empty round must stay cheap)
__global__ void __launch_bounds__(256)
k_clear_bins(uint32_t* __restrict__ bin_count, uint32_t n_bins, const unsigned int* __restrict__ n_list)
{
    if (*n_list == 0u) return;
    for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n_bins; i += gridDim.x * 256u) bin_count[i] = 0u;
}

}  // namespace

int nif_launch_clear_bins(const NifQueryWs* ws, const unsigned int* n_list, cudaStream_t stream)
{
    const unsigned blocks = (ws->n_bins + 255u) / 256u;
    k_clear_bins<<<blocks < 1184u ? blocks : 1184u, 256, 0, stream>>>(ws->bin_count, ws->n_bins, n_list);
    nif_count_launch(1);
    NIF_CUDA_TRY(cudaGetLastError());
    return NIF_OK;
}

int nif_launch_traverse(const nif_bvh* bvh, const nif_ray_batch* rays, const nif_query_out* out,
                        const NifQueryWs* ws, unsigned flags, const NifWalkRound* walk, cudaStream_t stream,
                        const NifPoseBatch* batch)
{
    if (rays->n == 0) return NIF_OK;
    const int n_sm = nif_sm_count();
    if (n_sm <= 0) return NIF_ERR_CUDA;
    TravParams p;
    p.nodes = bvh->nodes; p.lat = bvh->lattice; p.nv = bvh->nv; p.root = bvh->root;
    p.rlx = bvh->lo[0]; p.rly = bvh->lo[1]; p.rlz = bvh->lo[2];
    p.rhx = bvh->hi[0]; p.rhy = bvh->hi[1]; p.rhz = bvh->hi[2];
    p.n = (long long)rays->n; p.origin = rays->origin; p.dir = rays->dir; p.out = *out;
    p.ray_counter = &ws->scratch->tile_counter;
    p.overflow_flag = &ws->scratch->pad[3];
    p.bin_count = ws->bin_count; p.rank = ws->rank; p.bin_shift = ws->bin_shift; p.nvb = ws->nvb;
    p.flags = flags;
    p.ray_list = walk && walk->round > 0 ? walk->ray_list : nullptr;
    p.n_list = walk ? walk->n_list : nullptr;
    p.walk_dist_accum = walk ? walk->dist_accum : nullptr;
    p.batch = batch ? *batch : NifPoseBatch{nullptr, nullptr, 0};
    p.coherent_flag = &ws->scratch->pad[0];
    p.image_width = &ws->scratch->pad[5];
    const long long want = (rays->n + TRAV_BLOCK - 1) / TRAV_BLOCK;
    const long long cap = (long long)n_sm * TRAV_BLOCKS_PER_SM;
    if (p.ray_list) {
        // walk rounds >= 1: the live rays are in voxel-bin order, not pixel order -> persistent kernel
        k_traverse_persistent<true, false><<<(unsigned)(want < cap ? want : cap), TRAV_BLOCK, 0, stream>>>(p);
        nif_count_launch(1);
        NIF_CUDA_TRY(cudaGetLastError());
        return NIF_OK;
    }
    // scratch header (zeroed by nif_query): pad[0] decision, pad[1] coherent votes, pad[2] finished blocks,
    // pad[5] image width (0: not an image), pad[6] first row break (inverted)
    const long long groups_total = (rays->n + 31) / 32;
    const int n_groups = (int)(groups_total < 2048 ? groups_total : 2048);
    float extent = 0.0f;
    for (int a = 0; a < 3; ++a) extent = fmaxf(extent, bvh->hi[a] - bvh->lo[a]);
    k_ray_coherence<<<(n_groups * 32 + 255) / 256, 256, 0, stream>>>(
        (long long)rays->n, rays->origin, rays->dir, extent, n_groups, flags, &ws->scratch->pad[1], &ws->scratch->pad[0],
        &ws->scratch->pad[5], &ws->scratch->pad[6]);
    if (batch) {
        k_traverse_simple<true><<<(unsigned)want, TRAV_BLOCK, 0, stream>>>(p);
        k_traverse_persistent<false, true><<<(unsigned)(want < cap ? want : cap), TRAV_BLOCK, 0, stream>>>(p);
    } else {
        k_traverse_simple<false><<<(unsigned)want, TRAV_BLOCK, 0, stream>>>(p);
        k_traverse_persistent<false, false><<<(unsigned)(want < cap ? want : cap), TRAV_BLOCK, 0, stream>>>(p);
    }
    nif_count_launch(3);
    NIF_CUDA_TRY(cudaGetLastError());
    return NIF_OK;
}

int nif_launch_bin_hits(const nif_bvh* bvh, const nif_ray_batch* rays, const nif_query_out* out,
                        const NifQueryWs* ws, const NifWalkRound* walk, cudaStream_t stream)
{
    if (rays->n == 0) return NIF_OK;
    k_bin_offsets<<<(ws->n_bins + 1023u) / 1024u, 1024, 0, stream>>>(ws->bin_count, ws->n_bins, ws->scratch,
                                                                      walk && walk->round > 0 ? walk->n_list : nullptr);
    k_scatter_hits<<<(unsigned)((rays->n + 255) / 256), 256, 0, stream>>>(
        (long long)rays->n, bvh->nv, ws->bin_shift, ws->nvb, out->voxel_id, ws->bin_count, ws->rank, ws->hit_list,
        walk && walk->round > 0 ? walk->ray_list : nullptr, walk ? walk->n_list : nullptr);
    nif_count_launch(2);
    NIF_CUDA_TRY(cudaGetLastError());
    return NIF_OK;
}
