// nif_build.cu -- step (a0): per-pose build.  PAPER.md:41 "We voxelize the geometry in the rest
// space and apply parameterized deformation to obtain deformed voxels. For each deformation
// pose, we build a simple BVH over the deformed voxels".
//
// B200 design: the deformation keeps the rest lattice's topology, so
// the hierarchy is the sparse octree of the REST lattice (8-wide nodes, Morton order, children
// of a node contiguous one level down) and only the boxes depend on the pose.  Every step is a
// flat data-parallel kernel: deform (nv+1)^3 corners, per-brick occupancy masks, one exclusive
// scan per level, one node-write pass per level, bottom-up.
#include "nif_common.cuh"

#include <new>

namespace {

__host__ __device__ inline uint32_t spread3(uint32_t x)      // 10 bits -> every third bit
{
    x &= 0x3ffu;
    x = (x | (x << 16)) & 0x030000ffu;
    x = (x | (x << 8)) & 0x0300f00fu;
    x = (x | (x << 4)) & 0x030c30c3u;
    x = (x | (x << 2)) & 0x09249249u;
    return x;
}
__host__ __device__ inline uint32_t compact3(uint32_t x)
{
    x &= 0x09249249u;
    x = (x | (x >> 2)) & 0x030c30c3u;
    x = (x | (x >> 4)) & 0x0300f00fu;
    x = (x | (x >> 8)) & 0x030000ffu;
    x = (x | (x >> 16)) & 0x3ffu;
    return x;
}

// ---- O1/O2: rest lattice -> deformed lattice (R7, R28) ---------------------------------
// The lattice entry is the CORRECTLY ROUNDED fp32 value of the closed form (twist about +y by
// theta_max (y+1)/2, then circular-arc bend about z), a real function of the fp64 rest coordinate
// (2i-nv)/nv and the fp32 pose parameters: hit ids must be bit-exact against an independent
// implementation (B:5), and a last-bit difference of a corner can move a grazing ray to another voxel.
// Fast path: fp64 with CUDA's sincos (absolute error far below LATTICE_E for |coordinate| < 8), rounded
// once.  Where that value lies within LATTICE_E of the midpoint of two adjacent fp32 numbers -- where the
// fp64 error could change the rounding; exact zeros included -- the point is re-evaluated in
// double-double arithmetic (~105 bits: error-free sums and fma products, Taylor series for sin/cos after
// a three-word pi/2 reduction) and rounded from the (hi, lo) pair without double rounding.
struct dd { double hi, lo; };

__device__ __forceinline__ dd dd_quick(double a, double b)       // |a| >= |b| or a == 0
{
    const double s = __dadd_rn(a, b);
    return dd{s, __dsub_rn(b, __dsub_rn(s, a))};
}
__device__ __forceinline__ dd dd_two_sum(double a, double b)
{
    const double s = __dadd_rn(a, b), bb = __dsub_rn(s, a);
    return dd{s, __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb))};
}
__device__ __forceinline__ dd dd_two_prod(double a, double b)
{
    const double p = __dmul_rn(a, b);
    return dd{p, __fma_rn(a, b, -p)};
}
__device__ __forceinline__ dd dd_from(double a) { return dd{a, 0.0}; }
__device__ __forceinline__ dd dd_neg(dd a) { return dd{-a.hi, -a.lo}; }
__device__ __forceinline__ dd dd_add(dd a, dd b)
{
    dd s = dd_two_sum(a.hi, b.hi);
    const dd t = dd_two_sum(a.lo, b.lo);
    s = dd_quick(s.hi, __dadd_rn(s.lo, t.hi));
    return dd_quick(s.hi, __dadd_rn(s.lo, t.lo));
}
__device__ __forceinline__ dd dd_sub(dd a, dd b) { return dd_add(a, dd_neg(b)); }
__device__ __forceinline__ dd dd_mul(dd a, dd b)
{
    if (a.hi == 0.0 || b.hi == 0.0) return dd{__dmul_rn(a.hi, b.hi), 0.0};       // keeps exact (signed) zeros
    const dd p = dd_two_prod(a.hi, b.hi);
    return dd_quick(p.hi, __dadd_rn(p.lo, __dadd_rn(__dmul_rn(a.hi, b.lo), __dmul_rn(a.lo, b.hi))));
}
__device__ __forceinline__ dd dd_div(dd a, dd b)
{
    if (a.hi == 0.0) return dd{__ddiv_rn(a.hi, b.hi), 0.0};
    const double q1 = __ddiv_rn(a.hi, b.hi);
    dd r = dd_sub(a, dd_mul(dd_from(q1), b));
    const double q2 = __ddiv_rn(r.hi, b.hi);
    r = dd_sub(r, dd_mul(dd_from(q2), b));
    const double q3 = __ddiv_rn(r.hi, b.hi);
    return dd_add(dd_quick(q1, q2), dd_from(q3));
}
// sin and cos of a double-double argument (|a| up to a few hundred)
__device__ void dd_sincos(dd a, dd& s_out, dd& c_out)
{
    const double kq = rint(__dmul_rn(a.hi, 0.6366197723675814));               // nearest multiple of pi/2
    dd r = a;
    if (kq != 0.0) {
        r = dd_sub(r, dd_two_prod(kq, 1.5707963267948966));                     // pi/2 in three words
        r = dd_sub(r, dd_two_prod(kq, 6.123233995736766e-17));
        r = dd_sub(r, dd_two_prod(kq, -1.4973849048591698e-33));
    }
    const dd r2 = dd_mul(r, r);
    dd s = r, c = dd_from(1.0), ts = r, tc = dd_from(1.0);
    for (int n = 1; n <= 16; ++n) {                                             // |r| <= pi/4: r^33/33! < 2^-130
        tc = dd_div(dd_mul(tc, r2), dd_from((double)((2 * n - 1) * (2 * n))));
        ts = dd_div(dd_mul(ts, r2), dd_from((double)((2 * n) * (2 * n + 1))));
        if (n & 1) { c = dd_sub(c, tc); s = dd_sub(s, ts); }
        else { c = dd_add(c, tc); s = dd_add(s, ts); }
    }
    const int quad = (int)((long long)kq & 3LL);
    if (quad == 0) { s_out = s; c_out = c; }
    else if (quad == 1) { s_out = c; c_out = dd_neg(s); }
    else if (quad == 2) { s_out = dd_neg(s); c_out = dd_neg(c); }
    else { s_out = dd_neg(c); c_out = s; }
}
// RN_fp32(hi + lo) without double rounding: hi alone decides unless it sits exactly on an fp32 midpoint
__device__ __forceinline__ float dd_round_f32(dd v)
{
    const float f = __double2float_rn(v.hi);
    if ((double)f == v.hi || !isfinite(f)) return f;
    const float below = (double)f < v.hi ? f : nextafterf(f, -INFINITY);
    const float above = (double)f < v.hi ? nextafterf(f, INFINITY) : f;
    const double mid = 0.5 * ((double)below + (double)above);
    if (v.hi < mid) return below;
    if (v.hi > mid) return above;
    return v.lo > 0.0 ? above : (v.lo < 0.0 ? below : f);
}
__device__ void deform_point_dd(double x, double y, double z, float theta_max, float k, float& X, float& Y, float& Z)
{
    const dd a = dd_div(dd_mul(dd_from((double)theta_max), dd_two_sum(y, 1.0)), dd_from(2.0));
    dd sa, ca;
    dd_sincos(a, sa, ca);
    const dd dx = dd_from(x), dz = dd_from(z);
    const dd tx = dd_add(dd_mul(dx, ca), dd_mul(dz, sa));
    const dd ty = dd_from(y);
    const dd tz = dd_add(dd_mul(dd_neg(dx), sa), dd_mul(dz, ca));
    if (fabs((double)k) < 1e-6) { X = dd_round_f32(tx); Y = dd_round_f32(ty); Z = dd_round_f32(tz); return; }
    const dd kd = dd_from((double)k);
    const dd al = dd_mul(kd, tx);
    dd sal, cal, sh, ch;
    dd_sincos(al, sal, cal);
    dd_sincos(dd_div(al, dd_from(2.0)), sh, ch);
    X = dd_round_f32(dd_div(dd_mul(dd_sub(dd_from(1.0), dd_mul(kd, ty)), sal), kd));
    Y = dd_round_f32(dd_add(dd_mul(ty, cal), dd_div(dd_mul(dd_from(2.0), dd_mul(sh, sh)), kd)));
    Z = dd_round_f32(tz);
}

constexpr double LATTICE_E = 9.094947017729282e-13;      // 2^-40

// could an error of LATTICE_E change the fp32 rounding of v ?
__device__ __forceinline__ bool rounding_in_doubt(double v)
{
    const float f = __double2float_rn(v);
    if (!isfinite(f)) return true;
    const double lo = 0.5 * ((double)f + (double)nextafterf(f, -INFINITY));
    const double hi = 0.5 * ((double)f + (double)nextafterf(f, INFINITY));
    return fabs(v - lo) <= LATTICE_E || fabs(v - hi) <= LATTICE_E;
}

__global__ void k_deform_lattice(int nv, float theta_max_f, float k_f, float4* __restrict__ lat)
{
    const double theta_max = (double)theta_max_f, k = (double)k_f;
    const size_t np1 = (size_t)nv + 1;
    const size_t total = np1 * np1 * np1;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (size_t)gridDim.x * blockDim.x) {
        int i = (int)(idx % np1), j = (int)((idx / np1) % np1), kk = (int)(idx / (np1 * np1));
        double x = __ddiv_rn(__dsub_rn(__dmul_rn(2.0, (double)i), (double)nv), (double)nv);
        double y = __ddiv_rn(__dsub_rn(__dmul_rn(2.0, (double)j), (double)nv), (double)nv);
        double z = __ddiv_rn(__dsub_rn(__dmul_rn(2.0, (double)kk), (double)nv), (double)nv);
        double a = __ddiv_rn(__dmul_rn(theta_max, __dadd_rn(y, 1.0)), 2.0);
        double sa, ca;
        sincos(a, &sa, &ca);
        double tx = __dadd_rn(__dmul_rn(x, ca), __dmul_rn(z, sa));
        double ty = y;
        double tz = __dadd_rn(__dmul_rn(-x, sa), __dmul_rn(z, ca));
        double X = tx, Y = ty, Z = tz;
        if (fabs(k) >= 1e-6) {
            double al = __dmul_rn(k, tx);
            double sal, cal;
            sincos(al, &sal, &cal);
            double sh = sin(__ddiv_rn(al, 2.0));
            X = __ddiv_rn(__dmul_rn(__dsub_rn(1.0, __dmul_rn(k, ty)), sal), k);
            Y = __dadd_rn(__dmul_rn(ty, cal), __ddiv_rn(__dmul_rn(__dmul_rn(2.0, sh), sh), k));
        }
        float fx = (float)X, fy = (float)Y, fz = (float)Z;
        if (rounding_in_doubt(X) || rounding_in_doubt(Y) || rounding_in_doubt(Z))
            deform_point_dd(x, y, z, theta_max_f, k_f, fx, fy, fz);
        // a zero coordinate is stored as +0 (R28): -0 + 0 = +0 under round-to-nearest
        lat[idx] = make_float4(__fadd_rn(fx, 0.0f), __fadd_rn(fy, 0.0f), __fadd_rn(fz, 0.0f), 0.0f);
    }
}

// user-supplied deformed lattice ("user-specified deformation"): xyz floats -> the float4 lattice
__global__ void k_import_lattice(size_t total, const float* __restrict__ xyz, float4* __restrict__ lat)
{
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x)
        lat[idx] = make_float4(xyz[3 * idx], xyz[3 * idx + 1], xyz[3 * idx + 2], 0.0f);
}

// ---- occupancy masks ------------------------------------------------------------------------
// level 1: one Morton-indexed brick of 2x2x2 voxels; bit c = octant (c&1, (c>>1)&1, c>>2).
// counters[0] += occupied voxels; counters[1] = max (iy+1) over occupied voxels.
__global__ void k_brick_mask(int nv, const uint8_t* __restrict__ occ, uint32_t n_bricks,
                             uint8_t* __restrict__ mask, uint32_t* __restrict__ counters)
{
    uint32_t m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n_bricks) return;
    uint32_t bx = compact3(m), by = compact3(m >> 1), bz = compact3(m >> 2);
    uint32_t bits = 0; int top = 0;
    for (int c = 0; c < 8; ++c) {
        int ix = 2 * bx + (c & 1), iy = 2 * by + ((c >> 1) & 1), iz = 2 * bz + (c >> 2);
        if (ix < nv && iy < nv && iz < nv && occ[(size_t)ix + (size_t)nv * ((size_t)iy + (size_t)nv * iz)]) {
            bits |= 1u << c;
            top = max(top, iy + 1);
        }
    }
    mask[m] = (uint8_t)bits;
    if (bits) {
        atomicAdd(&counters[0], (uint32_t)__popc(bits));
        atomicMax(&counters[1], (uint32_t)top);
    }
}

__global__ void k_upper_mask(const uint8_t* __restrict__ lower, uint32_t n_cells,
                             uint8_t* __restrict__ mask)
{
    uint32_t m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n_cells) return;
    const uint2 v = *reinterpret_cast<const uint2*>(lower + 8 * (size_t)m);   // 8 child masks
    uint32_t bits = 0;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        if ((v.x >> (8 * c)) & 0xffu) bits |= 1u << c;
        if ((v.y >> (8 * c)) & 0xffu) bits |= 1u << (4 + c);
    }
    mask[m] = (uint8_t)bits;
}

// ---- exclusive scan of (mask != 0): three passes, 2048 elements per block -------------------
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_PER_THREAD = 8;
constexpr int SCAN_BLOCK = SCAN_THREADS * SCAN_PER_THREAD;

__device__ inline uint32_t block_exclusive_scan(uint32_t v, uint32_t* total)
{
    __shared__ uint32_t warp_sums[SCAN_THREADS / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    if (lane == 31) warp_sums[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        uint32_t s = lane < SCAN_THREADS / 32 ? warp_sums[lane] : 0;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, s, d);
            if (lane >= d) s += t;
        }
        if (lane < SCAN_THREADS / 32) warp_sums[lane] = s;        // inclusive over warps
    }
    __syncthreads();
    uint32_t warp_off = wid ? warp_sums[wid - 1] : 0;
    *total = warp_sums[SCAN_THREADS / 32 - 1];
    __syncthreads();
    return warp_off + inc - v;
}

__global__ void k_scan_count(const uint8_t* __restrict__ mask, uint32_t n, uint32_t* __restrict__ sums)
{
    uint32_t base = blockIdx.x * SCAN_BLOCK + threadIdx.x * SCAN_PER_THREAD;
    uint32_t c = 0;
    for (int i = 0; i < SCAN_PER_THREAD; ++i)
        if (base + i < n && mask[base + i]) ++c;
    uint32_t total;
    block_exclusive_scan(c, &total);
    if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

__global__ void k_scan_sums(uint32_t* __restrict__ sums, uint32_t nb, uint32_t* __restrict__ total_out)
{
    __shared__ uint32_t carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (uint32_t start = 0; start < nb; start += SCAN_THREADS) {
        uint32_t i = start + threadIdx.x;
        uint32_t v = i < nb ? sums[i] : 0;
        uint32_t total;
        uint32_t ex = block_exclusive_scan(v, &total);
        uint32_t c = carry;
        if (i < nb) sums[i] = c + ex;
        __syncthreads();
        if (threadIdx.x == 0) carry = c + total;
        __syncthreads();
    }
    if (threadIdx.x == 0) *total_out = carry;
}

__global__ void k_scan_write(const uint8_t* __restrict__ mask, uint32_t n,
                             const uint32_t* __restrict__ sums, uint32_t* __restrict__ offs)
{
    uint32_t base = blockIdx.x * SCAN_BLOCK + threadIdx.x * SCAN_PER_THREAD;
    uint32_t f[SCAN_PER_THREAD]; uint32_t c = 0;
    for (int i = 0; i < SCAN_PER_THREAD; ++i) {
        f[i] = (base + i < n && mask[base + i]) ? 1u : 0u;
        c += f[i];
    }
    uint32_t total;
    uint32_t ex = block_exclusive_scan(c, &total) + sums[blockIdx.x];
    for (int i = 0; i < SCAN_PER_THREAD; ++i) {
        if (base + i < n) offs[base + i] = ex;
        ex += f[i];
    }
}

// ---- node writes, bottom-up -----------------------------------------------------------------
__device__ inline void store_node(NifNode* dst, const NifNode& nd)
{
    const float4* s = reinterpret_cast<const float4*>(&nd);
    float4* d = reinterpret_cast<float4*>(dst);
#pragma unroll
    for (int i = 0; i < 16; ++i) d[i] = s[i];
}

// child boxes as stored in a node: one ulp outwards (nif_traverse.cu slab_node); the exact boxes stay in
// `boxes` for the level above and for the root
// (at least 1e-20 in absolute terms: next to 0 an ulp is a denormal, and (hi - o) * FLT_MAX must stay huge
// for a ray parallel to the slab with o exactly on the plane)
__device__ __forceinline__ float ulp_down(float v) { return isfinite(v) ? fminf(nextafterf(v, -INFINITY), v - 1e-20f) : v; }
__device__ __forceinline__ float ulp_up(float v) { return isfinite(v) ? fmaxf(nextafterf(v, INFINITY), v + 1e-20f) : v; }

__global__ void k_write_bricks(int nv, uint32_t n_bricks, const uint8_t* __restrict__ mask,
                               const uint32_t* __restrict__ offs, uint32_t node_base,
                               const float4* __restrict__ lat, NifNode* __restrict__ nodes,
                               float4* __restrict__ boxes)
{
    uint32_t m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n_bricks) return;
    uint32_t bits = mask[m];
    if (!bits) return;
    uint32_t bx = compact3(m), by = compact3(m >> 1), bz = compact3(m >> 2);
    const size_t np1 = (size_t)nv + 1;
    NifNode nd;
    float blo[3] = {INFINITY, INFINITY, INFINITY}, bhi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (int c = 0; c < 8; ++c) {
        float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
        uint32_t id = 0xffffffffu;
        if (bits & (1u << c)) {
            int ix = 2 * bx + (c & 1), iy = 2 * by + ((c >> 1) & 1), iz = 2 * bz + (c >> 2);
            id = (uint32_t)ix + (uint32_t)nv * ((uint32_t)iy + (uint32_t)nv * (uint32_t)iz);
            for (int q = 0; q < 8; ++q) {     // exact AABB of the 8 deformed corners (min/max: no rounding)
                float4 p = lat[(size_t)(ix + (q & 1)) + np1 * ((size_t)(iy + ((q >> 1) & 1)) + np1 * (size_t)(iz + (q >> 2)))];
                lo[0] = fminf(lo[0], p.x); hi[0] = fmaxf(hi[0], p.x);
                lo[1] = fminf(lo[1], p.y); hi[1] = fmaxf(hi[1], p.y);
                lo[2] = fminf(lo[2], p.z); hi[2] = fmaxf(hi[2], p.z);
            }
            for (int a = 0; a < 3; ++a) { blo[a] = fminf(blo[a], lo[a]); bhi[a] = fmaxf(bhi[a], hi[a]); }
        }
        for (int a = 0; a < 3; ++a) { nd.lo[a][c] = ulp_down(lo[a]); nd.hi[a][c] = ulp_up(hi[a]); }
        nd.child[c] = id;
    }
    nd.mask = bits; nd.is_brick = 1;
    for (int i = 0; i < 6; ++i) nd.pad[i] = 0;
    nd.pad[0] = 2u * bx + (uint32_t)nv * (2u * by + (uint32_t)nv * 2u * bz);   // voxel id of octant 0
    uint32_t idx = node_base + offs[m];
    store_node(nodes + idx, nd);
    boxes[2 * (size_t)idx] = make_float4(blo[0], blo[1], blo[2], 0.f);
    boxes[2 * (size_t)idx + 1] = make_float4(bhi[0], bhi[1], bhi[2], 0.f);
}

__global__ void k_write_level(uint32_t n_cells, const uint8_t* __restrict__ mask,
                              const uint32_t* __restrict__ offs, uint32_t node_base,
                              const uint8_t* __restrict__ child_mask,
                              const uint32_t* __restrict__ child_offs, uint32_t child_base,
                              NifNode* __restrict__ nodes, float4* __restrict__ boxes)
{
    uint32_t m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n_cells) return;
    uint32_t bits = mask[m];
    if (!bits) return;
    NifNode nd;
    float blo[3] = {INFINITY, INFINITY, INFINITY}, bhi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (int c = 0; c < 8; ++c) {
        float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
        uint32_t id = 0xffffffffu;
        if (bits & (1u << c)) {
            id = child_base + child_offs[8 * (size_t)m + c];
            float4 l = boxes[2 * (size_t)id], h = boxes[2 * (size_t)id + 1];
            lo[0] = l.x; lo[1] = l.y; lo[2] = l.z; hi[0] = h.x; hi[1] = h.y; hi[2] = h.z;
            for (int a = 0; a < 3; ++a) { blo[a] = fminf(blo[a], lo[a]); bhi[a] = fmaxf(bhi[a], hi[a]); }
        }
        for (int a = 0; a < 3; ++a) { nd.lo[a][c] = ulp_down(lo[a]); nd.hi[a][c] = ulp_up(hi[a]); }
        nd.child[c] = id;
    }
    (void)child_mask;
    nd.mask = bits; nd.is_brick = 0;
    for (int i = 0; i < 6; ++i) nd.pad[i] = 0;
    // existing children are consecutive nodes (exclusive scan over Morton-ordered cells): first one
    nd.pad[0] = child_base + child_offs[8 * (size_t)m + (size_t)(__ffs((int)bits) - 1)];
    uint32_t idx = node_base + offs[m];
    store_node(nodes + idx, nd);
    boxes[2 * (size_t)idx] = make_float4(blo[0], blo[1], blo[2], 0.f);
    boxes[2 * (size_t)idx + 1] = make_float4(bhi[0], bhi[1], bhi[2], 0.f);
}

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct BuildLayout {
    int P, levels;                       // padded pow2 resolution, hierarchy levels (1..levels)
    size_t cells[12];                    // cells[l], l = 1..levels
    size_t off_lattice, off_counters, off_sums, off_mask[12], off_offs[12], off_nodes;
    size_t fixed_bytes;
};

BuildLayout make_layout(int nv)
{
    BuildLayout L{};
    int P = 2;
    while (P < nv) P <<= 1;
    L.P = P;
    int levels = 0;
    for (int p = P; p > 1; p >>= 1) ++levels;
    L.levels = levels;
    size_t off = 0;
    const size_t np1 = (size_t)nv + 1;
    L.off_lattice = off; off = align_up(off + np1 * np1 * np1 * sizeof(float4), 256);
    L.off_counters = off; off = align_up(off + 64 * sizeof(uint32_t), 256);
    size_t c1 = (size_t)(P / 2) * (P / 2) * (P / 2);
    L.off_sums = off; off = align_up(off + (c1 / SCAN_BLOCK + 2) * sizeof(uint32_t), 256);
    for (int l = 1; l <= levels; ++l) {
        size_t c = (size_t)(P >> l) * (P >> l) * (P >> l);
        L.cells[l] = c;
        L.off_mask[l] = off; off = align_up(off + align_up(c, 8), 256);
        L.off_offs[l] = off; off = align_up(off + c * sizeof(uint32_t), 256);
    }
    L.off_nodes = off;
    L.fixed_bytes = off;
    return L;
}

size_t max_nodes_for(const BuildLayout& L, int64_t max_occ)
{
    size_t total = 0;
    for (int l = 1; l <= L.levels; ++l)
        total += (size_t)((int64_t)L.cells[l] < max_occ ? (int64_t)L.cells[l] : max_occ);
    return total ? total : 1;
}

constexpr size_t NODE_BYTES = sizeof(NifNode) + 2 * sizeof(float4);

int device_is_sm100()
{
    int dev = 0, major = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return 0; }
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
        (void)cudaGetLastError(); return 0;
    }
    return major == 10;
}

// fold-over check (R7): the twist keeps y, so the largest k*y over occupied corners is
// k * rest-y of the highest occupied corner.
bool pose_folds_over(const nif_deform_params* pose, int nv, uint32_t top_iy)
{
    if (fabsf(pose->bend_k) < 1e-6f) return false;
    double ytop = (2.0 * (double)top_iy - nv) / nv;
    double ybot = -1.0;                           // k < 0 folds at the bottom; be conservative
    double worst = pose->bend_k > 0 ? (double)pose->bend_k * ytop : (double)pose->bend_k * ybot;
    return worst >= 1.0 - 1e-3;
}

// pose != NULL: closed-form deformation; else copy the user's deformed lattice
void launch_deform(int nv, const nif_deform_params* pose, const float* user_lattice, float4* lattice, cudaStream_t stream)
{
    const size_t np1 = (size_t)nv + 1, total = np1 * np1 * np1;
    int blocks = (int)((total + 255) / 256);
    if (blocks > 148 * 32) blocks = 148 * 32;
    if (pose) k_deform_lattice<<<blocks, 256, 0, stream>>>(nv, pose->twist_theta_max, pose->bend_k, lattice);
    else k_import_lattice<<<blocks, 256, 0, stream>>>(total, user_lattice, lattice);
    nif_count_launch(1);
}

// boxes of every node from the deformed lattice, bottom-up, with the topology (masks, scan offsets,
// node ranges) already in the workspace; reads the root box back (SYNCHRONISES).
int write_levels(nif_bvh* b, const BuildLayout& L, cudaStream_t stream)
{
    char* ws = b->ws;
    NifNode* nodes = (NifNode*)(ws + L.off_nodes);
    float4* boxes = (float4*)(ws + L.off_nodes + align_up(b->node_capacity * sizeof(NifNode), 256));
    const float4* lattice = (const float4*)(ws + L.off_lattice);
    for (int l = 1; l <= L.levels; ++l) {
        const uint32_t c = (uint32_t)L.cells[l];
        const uint8_t* mask = (const uint8_t*)(ws + L.off_mask[l]);
        const uint32_t* offs = (const uint32_t*)(ws + L.off_offs[l]);
        if (l == 1)
            k_write_bricks<<<(c + 127) / 128, 128, 0, stream>>>(b->nv, c, mask, offs, b->level_base[1], lattice, nodes, boxes);
        else
            k_write_level<<<(c + 127) / 128, 128, 0, stream>>>(
                c, mask, offs, b->level_base[l], (const uint8_t*)(ws + L.off_mask[l - 1]),
                (const uint32_t*)(ws + L.off_offs[l - 1]), b->level_base[l - 1], nodes, boxes);
        nif_count_launch(1);
    }
    b->root = (int32_t)b->level_base[L.levels];
    float4 rb[2];
    cudaError_t e = cudaMemcpyAsync(rb, boxes + 2 * (size_t)b->root, sizeof(rb), cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) { (void)cudaGetLastError(); return NIF_ERR_CUDA; }
    b->lo[0] = rb[0].x; b->lo[1] = rb[0].y; b->lo[2] = rb[0].z;
    b->hi[0] = rb[1].x; b->hi[1] = rb[1].y; b->hi[2] = rb[1].z;
    return NIF_OK;
}

}  // namespace

extern "C" int nif_device_supported(void) { return device_is_sm100(); }

extern "C" int nif_bvh_workspace_bytes(int32_t nv, int64_t max_occupied, size_t* bytes)
{
    if (!bytes || nv < 2 || nv > 512 || max_occupied < 0) return NIF_ERR_INVALID_ARG;
    int64_t all = (int64_t)nv * nv * nv;
    if (max_occupied > all) max_occupied = all;
    BuildLayout L = make_layout(nv);
    *bytes = L.fixed_bytes + align_up(max_nodes_for(L, max_occupied) * NODE_BYTES, 256) + 256;
    return NIF_OK;
}

static int build_common(const nif_voxel_set* voxels, const nif_deform_params* pose, const float* user_lattice,
                        void* workspace, size_t workspace_bytes, void* stream_, nif_bvh** out)
{
    if (!voxels || (!pose && !user_lattice) || !workspace || !out || !voxels->occupancy) return NIF_ERR_INVALID_ARG;
    const int nv = voxels->nv;
    if (nv < 2 || nv > 512) return NIF_ERR_INVALID_ARG;
    if (pose && (!isfinite(pose->twist_theta_max) || !isfinite(pose->bend_k))) return NIF_ERR_INVALID_ARG;
    if (((uintptr_t)workspace & 255u) != 0) return NIF_ERR_WORKSPACE;
    if (!device_is_sm100()) return NIF_ERR_UNSUPPORTED;
    cudaStream_t stream = (cudaStream_t)stream_;
    const BuildLayout L = make_layout(nv);
    if (workspace_bytes < L.fixed_bytes + NODE_BYTES) return NIF_ERR_WORKSPACE;
    char* ws = (char*)workspace;
    float4* lattice = (float4*)(ws + L.off_lattice);
    uint32_t* counters = (uint32_t*)(ws + L.off_counters);
    uint32_t* sums = (uint32_t*)(ws + L.off_sums);
    const size_t node_capacity = (workspace_bytes - L.off_nodes) / NODE_BYTES;

    NIF_CUDA_TRY(cudaMemsetAsync(counters, 0, 64 * sizeof(uint32_t), stream));
    launch_deform(nv, pose, user_lattice, lattice, stream);
    for (int l = 1; l <= L.levels; ++l) {
        const uint32_t c = (uint32_t)L.cells[l];
        uint8_t* mask = (uint8_t*)(ws + L.off_mask[l]);
        uint32_t* offs = (uint32_t*)(ws + L.off_offs[l]);
        if (l == 1)
            k_brick_mask<<<(c + 255) / 256, 256, 0, stream>>>(nv, voxels->occupancy, c, mask, counters);
        else
            k_upper_mask<<<(c + 255) / 256, 256, 0, stream>>>((const uint8_t*)(ws + L.off_mask[l - 1]), c, mask);
        const uint32_t nb = (c + SCAN_BLOCK - 1) / SCAN_BLOCK;
        k_scan_count<<<nb, SCAN_THREADS, 0, stream>>>(mask, c, sums);
        k_scan_sums<<<1, SCAN_THREADS, 0, stream>>>(sums, nb, counters + 2 + l);
        k_scan_write<<<nb, SCAN_THREADS, 0, stream>>>(mask, c, sums, offs);
        nif_count_launch(4);
    }
    uint32_t h_counters[64];
    NIF_CUDA_TRY(cudaMemcpyAsync(h_counters, counters, sizeof(h_counters), cudaMemcpyDeviceToHost, stream));
    NIF_CUDA_TRY(cudaStreamSynchronize(stream));
    NIF_CUDA_TRY(cudaGetLastError());

    const uint32_t n_occ = h_counters[0];
    if (n_occ && pose && pose_folds_over(pose, nv, h_counters[1])) return NIF_ERR_DEFORM_SINGULAR;
    uint32_t base[12] = {0};
    size_t n_nodes = 0;
    for (int l = 1; l <= L.levels; ++l) { base[l] = (uint32_t)n_nodes; n_nodes += h_counters[2 + l]; }
    if (n_nodes > node_capacity) return NIF_ERR_WORKSPACE;
    NifNode* nodes = (NifNode*)(ws + L.off_nodes);
    float4* boxes = (float4*)(ws + L.off_nodes + align_up(node_capacity * sizeof(NifNode), 256));
    // boxes region must fit too: node_capacity was computed with NODE_BYTES per node, minus alignment slack
    if ((char*)(boxes + 2 * n_nodes) > ws + workspace_bytes) return NIF_ERR_WORKSPACE;

    nif_bvh* b = new (std::nothrow) nif_bvh();
    if (!b) return NIF_ERR_CUDA;
    b->nv = nv; b->n_occupied = (int32_t)n_occ; b->n_nodes = (int32_t)n_nodes; b->depth = L.levels;
    b->root = -1;
    b->theta_max = pose ? pose->twist_theta_max : 0.0f; b->bend_k = pose ? pose->bend_k : 0.0f;
    b->local_inverse = pose ? 0 : 1;
    b->lattice = lattice; b->nodes = nodes;
    for (int a = 0; a < 3; ++a) { b->lo[a] = 0.f; b->hi[a] = 0.f; }
    b->ws = ws; b->node_capacity = node_capacity; b->top_iy = h_counters[1];
    for (int l = 0; l < 12; ++l) b->level_base[l] = base[l];
    if (n_occ) {
        int rc = write_levels(b, L, stream);
        if (rc != NIF_OK) { delete b; return rc; }
    }
    *out = b;
    return NIF_OK;
}

extern "C" int nif_build_deformed_bvh(const nif_voxel_set* voxels, const nif_deform_params* pose,
                                      void* workspace, size_t workspace_bytes, void* stream, nif_bvh** out)
{
    if (!pose) return NIF_ERR_INVALID_ARG;
    return build_common(voxels, pose, nullptr, workspace, workspace_bytes, stream, out);
}

extern "C" int nif_build_bvh_from_lattice(const nif_voxel_set* voxels, const float* lattice_xyz,
                                          void* workspace, size_t workspace_bytes, void* stream, nif_bvh** out)
{
    if (!lattice_xyz) return NIF_ERR_INVALID_ARG;
    return build_common(voxels, nullptr, lattice_xyz, workspace, workspace_bytes, stream, out);
}

// Same voxel set, new pose: the hierarchy's topology is the rest lattice's octree (pose-independent),
// so only the corner lattice and the boxes are recomputed.
extern "C" int nif_bvh_refit(nif_bvh* b, const nif_deform_params* pose, void* stream_)
{
    if (!b || !pose) return NIF_ERR_INVALID_ARG;
    if (!isfinite(pose->twist_theta_max) || !isfinite(pose->bend_k)) return NIF_ERR_INVALID_ARG;
    if (!device_is_sm100()) return NIF_ERR_UNSUPPORTED;
    if (b->n_occupied && pose_folds_over(pose, b->nv, b->top_iy)) return NIF_ERR_DEFORM_SINGULAR;
    cudaStream_t stream = (cudaStream_t)stream_;
    const BuildLayout L = make_layout(b->nv);
    launch_deform(b->nv, pose, nullptr, (float4*)(b->ws + L.off_lattice), stream);
    b->theta_max = pose->twist_theta_max; b->bend_k = pose->bend_k; b->local_inverse = 0;
    if (b->n_occupied) return write_levels(b, L, stream);
    NIF_CUDA_TRY(cudaStreamSynchronize(stream));
    return NIF_OK;
}

extern "C" int nif_bvh_refit_lattice(nif_bvh* b, const float* lattice_xyz, void* stream_)
{
    if (!b || !lattice_xyz) return NIF_ERR_INVALID_ARG;
    if (!device_is_sm100()) return NIF_ERR_UNSUPPORTED;
    cudaStream_t stream = (cudaStream_t)stream_;
    const BuildLayout L = make_layout(b->nv);
    launch_deform(b->nv, nullptr, lattice_xyz, (float4*)(b->ws + L.off_lattice), stream);
    b->theta_max = 0.0f; b->bend_k = 0.0f; b->local_inverse = 1;
    if (b->n_occupied) return write_levels(b, L, stream);
    NIF_CUDA_TRY(cudaStreamSynchronize(stream));
    return NIF_OK;
}

extern "C" int nif_bvh_get_info(const nif_bvh* b, nif_bvh_info* info)
{
    if (!b || !info) return NIF_ERR_INVALID_ARG;
    info->nv = b->nv; info->n_occupied = b->n_occupied; info->n_nodes = b->n_nodes;
    info->depth = b->depth;
    for (int a = 0; a < 3; ++a) { info->lo[a] = b->lo[a]; info->hi[a] = b->hi[a]; }
    info->theta_max = b->theta_max; info->bend_k = b->bend_k;
    return NIF_OK;
}

extern "C" int nif_bvh_get_lattice(const nif_bvh* b, const float** lattice_xyzw)
{
    if (!b || !lattice_xyzw) return NIF_ERR_INVALID_ARG;
    *lattice_xyzw = reinterpret_cast<const float*>(b->lattice);
    return NIF_OK;
}

extern "C" void nif_bvh_destroy(nif_bvh* b) { delete b; }
