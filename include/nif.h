/* nif.h -- C ABI of libnif.so: batched inference of the voxel-deformation-aware neural
 * intersection query (arxiv 2604.24666) on one NVIDIA B200 (sm_100a).
 *
 * Citations: P:NN = PAPER.md line NN; B:NN = BASELINE.json line NN; R# = DESIGN.md section 3
 * (readings adopted where the paper is silent).
 *
 * The query, per ray (Fig. 2; B:5):
 *   (1) find the nearest deformed voxel with its entry/exit parameters t_in, t_out by
 *       traversing a BVH built over the occupied voxels after the pose's deformation,
 *   (2) map entry and exit points back to rest space with the inverse deformation,
 *   (3) encode both with psi(x) = phi(gamma(x)) (Eq. 1),
 *   (4) run the shared MLP, (5) decode the heads.
 *
 * General conventions
 *   - Every pointer inside a descriptor struct is a DEVICE pointer owned by the caller unless
 *     the field comment says HOST.  The library never frees caller memory.  Large buffers
 *     (BVH, per-query scratch) live in caller-provided workspaces; the library itself only
 *     allocates the small repacked weight images of a nif_net (< 2 MiB) and the staging
 *     buffers of a nif_stage.
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).  nif_query only
 *     enqueues work and returns; calls documented as "synchronises" wait for the stream.
 *     The enqueue-only calls (nif_query, nif_query_multi, nif_query_poses) allocate nothing, copy nothing
 *     from host memory and can be captured in a CUDA graph and replayed (rays and outputs are read /
 *     written at replay; the BVHs' device data and pose parameters are the ones seen at capture time).
 *   - Return value: NIF_OK (0) or a negative nif_status.  On error no output is written.
 *     No exceptions, no abort(), nothing printed.
 *   - There is no CPU fallback: on a device that is not compute capability 10.x every entry
 *     point that would launch a kernel returns NIF_ERR_UNSUPPORTED.
 */
#ifndef NIF_H_
#define NIF_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    NIF_OK = 0,
    NIF_ERR_INVALID_ARG = -1,      /* null pointer, negative count, size out of range          */
    NIF_ERR_UNSUPPORTED = -2,      /* shape/dtype the kernels do not cover, or not an sm_100 GPU */
    NIF_ERR_DEFORM_SINGULAR = -3,  /* bend folds over: some occupied corner has k*y >= 1 - 1e-3 (R7) */
    NIF_ERR_WORKSPACE = -4,        /* workspace too small or misaligned                        */
    NIF_ERR_CUDA = -5,             /* a CUDA runtime call failed                               */
    NIF_ERR_INTERNAL = -6,         /* an internal limit was exceeded (reported by nif_query_last_hit_count) */
    NIF_ERR_STATIC_LIMIT = -7      /* nif_query_static: batch larger than NIF_STATIC_MAX_RAYS   */
} nif_status;

enum { NIF_F32 = 0, NIF_F16 = 1 };            /* nif_net_desc.dtype */

/* nif_net_desc.enc_mode: how positional encoding gamma and hash grid phi are combined (R1).
 *   NIF_ENC_COMPOSE  psi(x) = phi(gamma(x)), Eq. 1: every one of the S = 1 + 2B samples of
 *                    gamma goes through the grid; D_in = 2 * S * L * F.  The paper's encoding; default.
 *   NIF_ENC_CONCAT   psi(x) = [ x, sin(2^0 x), cos(2^0 x), ..., sin(2^(B-1) x), cos(2^(B-1) x), phi(x) ]
 *                    (B:5 "positional frequency terms plus a multiresolution hash grid"): per band sin of
 *                    the three axes then cos of the three axes, raw values, then the L*F grid features of
 *                    the point; D_in = 2 * (3 + 6B + L * F), entry endpoint then exit endpoint.
 *                    Not with feat = 3. */
enum { NIF_ENC_COMPOSE = 0, NIF_ENC_CONCAT = 1 };

/* nif_query flags */
enum {
    NIF_OCCLUSION_ONLY = 1u,   /* decode only the occlusion head (B:10); other head outputs untouched */
    NIF_ENGINE_FFMA    = 2u,   /* force the scalar-FMA encode+MLP kernel even for NIF_F16 nets        */
    NIF_TRAVERSE_ONLY  = 4u,   /* step (1) only: voxel_id, t_in, t_out                                */
    /* The traversal has two kernels: one thread per ray with static assignment (best for coherent
     * batches such as camera rays) and persistent warps with dynamic ray fetch (best for incoherent
     * batches).  By default a device-side vote over sampled ray groups picks one; these force it.
     * Results are identical either way.  A batch that is a row-major image (n = width x height, width a multiple of
     * 8, height of 4, consecutive rays one pixel apart) is recognised on the device as well, and the static kernel then
     * gives each warp a tile of 8 x 4 pixels instead of 32 pixels of a row: faster, same results; nothing to set. */
    NIF_TRAVERSE_COHERENT   = 8u,
    NIF_TRAVERSE_INCOHERENT = 16u,
    /* Diagnostic: the tensor-core kernel fills its A operand with a constant instead of gathering from
     * the table, so a timed query measures the tcgen05 MLP pipeline alone (head outputs are then
     * meaningless).  bench.py --probe-mlp reports the tensor-pipe rate it reaches. */
    NIF_PROBE_SKIP_GATHER   = 32u,
    /* Distance head variant of P:87 ("We replace the sigmoid output with ReLU and regress
     * log-transformed distances"; R24): y = ReLU(z1) is log(1 + D) of the ACCUMULATED distance, so
     * dist_total = expm1(max(z1, 0)) and distance = dist_total - t_in.  Default is the
     * scale-invariant head sigmoid(z1) * (t_out - t_in) (B:7; R14). */
    NIF_DIST_LOG            = 64u
};

#define NIF_N_OUT 12   /* logits per ray: occlusion 1, distance 1, normal 3, albedo 3, material 4 (B:7) */

typedef struct nif_bvh nif_bvh;       /* opaque host object; its device data lives in the caller's workspace */
typedef struct nif_net nif_net;       /* opaque host object: table pointer + repacked weights               */
typedef struct nif_stage nif_stage;   /* opaque: device staging buffers + streams for nif_query_host        */

/* Rest-space voxelisation: nv^3 lattice over [-1,1]^3, voxel (ix,iy,iz) has
 * id = ix + nv*(iy + nv*iz) and is occupied iff occupancy[id] != 0. */
typedef struct {
    int32_t nv;                   /* 2 <= nv <= 512 */
    const uint8_t* occupancy;     /* DEVICE, nv^3 bytes */
} nif_voxel_set;

/* Parameterised deformation (formulas B:7-11, R7): twist about +y by
 * twist_theta_max*(y+1)/2, then bend about z with curvature bend_k (|k| < 1e-6 = no bend).
 * (0, 0) is the identity pose. */
typedef struct {
    float twist_theta_max;
    float bend_k;
} nif_deform_params;

/* Encoding + MLP shape (B:7-11).  D_in = 2 * (1 + 2*pe_bands) * levels * feat
 * (NIF_ENC_COMPOSE). */
typedef struct {
    int32_t pe_bands;             /* B: sinusoidal bands (the paper's "F"), 0..8          */
    int32_t levels;               /* L: hash-grid levels, 1..16                                 */
    int32_t log2_T;               /* table entries per level = 2^log2_T, 4..24                  */
    int32_t feat;                 /* F: features per entry, 1..4.  F = 3 (the paper's own setup) is
                                   * stored padded to 4 inside the library: the table is then COPIED   */
    const int32_t* level_res;     /* HOST, `levels` entries: grid resolution N_l of each level  */
    int32_t hidden_layers;        /* H: 1..8                                                    */
    int32_t width;                /* W: 16..128, multiple of 16                                 */
    int32_t dtype;                /* NIF_F32: table/weights float; NIF_F16: table/weights __half */
    int32_t enc_mode;             /* NIF_ENC_COMPOSE (0) or NIF_ENC_CONCAT                      */
} nif_net_desc;

typedef struct {
    int64_t n;                    /* rays in the batch, >= 0 */
    const float* origin;          /* n*3 */
    const float* dir;             /* n*3, unit length */
} nif_ray_batch;

/* Outputs, all DEVICE, struct-of-arrays.  voxel_id/t_in/t_out are always written.
 * Miss ray: voxel_id = -1, t_in = t_out = +inf, every head output 0 (R18).
 * Head pointers may be NULL only with NIF_TRAVERSE_ONLY; with NIF_OCCLUSION_ONLY only
 * `occlusion` is required.  raw_logits is optional (NULL to skip). */
typedef struct {
    int32_t* voxel_id;            /* n   rest-space linear id of the nearest deformed voxel        */
    float* t_in;                  /* n   entry parameter along the ray (deformed space, unit dir)  */
    float* t_out;                 /* n   exit parameter                                            */
    float* occlusion;             /* n   sigmoid(z0)                                               */
    float* distance;              /* n   sigmoid(z1) * (t_out - t_in)                     */
    float* dist_total;            /* n   D = t_in + distance            (k = 0)              */
    float* normal;                /* 3n  z2..4 normalised                                          */
    float* albedo;                /* 3n  sigmoid(z5..7)                                            */
    float* material_logits;       /* 4n  z8..11                                                    */
    float* raw_logits;            /* 12n optional                                                  */
    /* Hit positions ("we reconstruct hit positions along the same segmented ray in rest space"),
     * both optional (NULL to skip), zeros for a miss, not written with NIF_OCCLUSION_ONLY:          */
    float* hit_position;          /* 3n  deformed space: o + dist_total * d                        */
    float* hit_position_rest;     /* 3n  rest space, [-1,1]^3 coordinates: on the straight segment */
                                  /*     between the rest images of entry and exit at the   */
                                  /*     fraction clamp(distance / (t_out - t_in), 0, 1)           */
} nif_query_out;

typedef struct {
    int32_t nv;
    int32_t n_occupied;           /* occupied voxels                                   */
    int32_t n_nodes;              /* BVH nodes                                         */
    int32_t depth;                /* levels of the hierarchy (root = depth-1)          */
    float lo[3], hi[3];           /* bounding box of the posed object (root box)       */
    float theta_max, bend_k;
} nif_bvh_info;

/* -------- step (a0): per-pose build ("For each deformation pose, we build a simple BVH
 * over the deformed voxels") ------------------------------------------------------------- */

/* Bytes of workspace nif_build_deformed_bvh needs for an nv^3 grid with at most
 * `max_occupied` occupied voxels (pass nv^3 if unknown).  Host-only, no CUDA call. */
int nif_bvh_workspace_bytes(int32_t nv, int64_t max_occupied, size_t* bytes);

/* Deforms the (nv+1)^3 corner lattice (fp64 evaluation, one rounding to fp32), computes the
 * exact AABB of every occupied deformed voxel and builds the 8-wide hierarchy over them.
 * `workspace`: DEVICE, 256-byte aligned, at least nif_bvh_workspace_bytes; it holds the BVH
 * for the lifetime of *out and must not be touched by the caller.  SYNCHRONISES `stream`
 * (it reads back counts and the fold-over check).  Errors: NIF_ERR_DEFORM_SINGULAR,
 * NIF_ERR_WORKSPACE (also when the grid holds more than the max_occupied the workspace was
 * sized for), NIF_ERR_INVALID_ARG, NIF_ERR_CUDA. */
int nif_build_deformed_bvh(const nif_voxel_set* voxels, const nif_deform_params* pose,
                           void* workspace, size_t workspace_bytes, void* stream, nif_bvh** out);

/* The same for a USER-SPECIFIED deformation given as the deformed corner lattice itself:
 * `lattice_xyz`: DEVICE, (nv+1)^3 x 3 floats, lattice point (i,j,k) at index i + (nv+1)*(j + (nv+1)*k),
 * copied into the workspace.  No closed-form inverse exists for such a pose, so nif_query maps entry and
 * exit points back with the voxel-local inverse of the trilinear interpolant of the hit voxel's 8 deformed
 * corners (R27: Newton, 5 iterations, fp32).  The lattice must not fold over (positive Jacobian);
 * this is not checked.  nif_bvh_refit_lattice replaces the lattice of an existing BVH (any BVH: a
 * closed-form one becomes a lattice one).  Both SYNCHRONISE. */
int nif_build_bvh_from_lattice(const nif_voxel_set* voxels, const float* lattice_xyz,
                               void* workspace, size_t workspace_bytes, void* stream, nif_bvh** out);
int nif_bvh_refit_lattice(nif_bvh* bvh, const float* lattice_xyz, void* stream);

/* New pose for the same voxel set: recomputes the deformed corner lattice and every box of the
 * hierarchy in place; the topology (which is the sparse octree of the REST lattice) is reused, so no
 * occupancy pass, scan or allocation happens.  The result is bit-identical to a fresh
 * nif_build_deformed_bvh with that pose.  SYNCHRONISES `stream` (reads the root box back).  On
 * NIF_ERR_DEFORM_SINGULAR the BVH keeps its previous pose.  Queries enqueued earlier on another
 * stream must have finished. */
int nif_bvh_refit(nif_bvh* bvh, const nif_deform_params* pose, void* stream);

int nif_bvh_get_info(const nif_bvh* bvh, nif_bvh_info* info);      /* host-only */

/* DEVICE pointer to the deformed corner lattice: (nv+1)^3 float4 (x,y,z,0), lattice point
 * (i,j,k) at index i + (nv+1)*(j + (nv+1)*k).  Valid while the BVH lives.  For parity tests. */
int nif_bvh_get_lattice(const nif_bvh* bvh, const float** lattice_xyzw);

void nif_bvh_destroy(nif_bvh* bvh);                                /* frees the host object only */

/* -------- network ------------------------------------------------------------------------ */

/* `table`: DEVICE, layout table[l][index][f], every level 2^log2_T entries, float (NIF_F32) or
 * __half (NIF_F16); borrowed for the lifetime of the net (not copied, except feat = 3: the
 * library keeps its own copy padded to 4 features per entry, levels * 2^log2_T * 4 elements).
 * `weights`: HOST array of hidden_layers+1 DEVICE pointers; weights[i] is row-major
 * (fan_out, fan_in): (W, D_in), (W, W)..., (12, W); same element type as the table.  Copied and
 * repacked on `stream` (tensor-core operand images, zero-padded output layer).  SYNCHRONISES. */
int nif_net_create(const nif_net_desc* desc, const void* table, const void* const* weights,
                   void* stream, nif_net** out);
void nif_net_destroy(nif_net* net);

/* 1 if nif_query runs this net on the tcgen05 fused encode+MLP kernel, 0 if on the scalar-FMA
 * kernel (NIF_F32 nets, shapes the tensor-core kernel does not cover), negative on error.
 * Host-only. */
int nif_net_uses_tensor_cores(const nif_net* net);

/* -------- steps (a1)-(a5): the query ------------------------------------------------------ */

/* Scratch bytes nif_query needs for a batch of n rays.  Host-only. */
int nif_query_workspace_bytes(int64_t n, size_t* bytes);

/* Enqueues the whole hot path on `stream` and returns without synchronising.
 * `workspace`: DEVICE, 256-byte aligned, >= nif_query_workspace_bytes(rays->n); contents are
 * scratch (hit-ray compaction list and counters) and may be reused by the next call on the
 * same stream.  Several poses (B:9) = one nif_bvh per pose sharing one net, and either one nif_query
 * per pose or one nif_query_poses for all of them. */
int nif_query(const nif_bvh* bvh, const nif_net* net, const nif_ray_batch* rays,
              const nif_query_out* out, void* workspace, size_t workspace_bytes,
              unsigned flags, void* stream);

/* Several poses of one object in one query (B:9 "8 poses ... One BVH per pose ... Network ... shared across
 * all poses"): ray r is traced against bvhs[pose_id[r]].  `bvhs`: HOST array of n_poses (1..64) BVHs of the
 * same grid size and the same kind (all closed-form or all lattice poses); `pose_id`: DEVICE, rays->n entries
 * in [0, n_poses).  Everything else as nif_query (same outputs, same flags except NIF_PROBE_SKIP_GATHER).
 * Hit rays are grouped by the REST-space voxel they hit across poses, which is what the shared hash grid is
 * indexed by, so one batched call is faster than n_poses separate ones.  Workspace:
 * nif_query_poses_workspace_bytes(rays->n).  Enqueue only. */
int nif_query_poses_workspace_bytes(int64_t n, size_t* bytes);
int nif_query_poses(const nif_bvh* const* bvhs, int32_t n_poses, const nif_net* net,
                    const nif_ray_batch* rays, const int32_t* pose_id, const nif_query_out* out,
                    void* workspace, size_t workspace_bytes, unsigned flags, void* stream);

/* -------- evaluation-time multi-voxel walk (R22, R23) ------------------- */

/* Outcome of a walk, per ray. */
enum {
    NIF_WALK_MISS      = 0,    /* the ray left the object without a predicted hit: outputs as for a miss (R18) */
    NIF_WALK_HIT       = 1,    /* accepted in voxel k = steps-1: `out` holds that voxel's outputs              */
    NIF_WALK_MAX_STEPS = 2     /* max_steps voxels evaluated, none accepted: `out` holds the last one's        */
};

typedef struct {
    int32_t* status;              /* n   NIF_WALK_*                                                         */
    int32_t* steps;               /* n   voxels on which the network was evaluated                          */
    float* dist_accum;            /* n   sum_{j<k}(delta_j + l_j) + delta_k + t_k of P:61, accumulated term  */
                                  /*     by term along the ray (delta signed, R23); the partial sum for     */
                                  /*     NIF_WALK_MAX_STEPS; 0 for NIF_WALK_MISS                            */
} nif_walk_out;

/* Scratch bytes nif_query_multi needs for a batch of n rays.  Host-only. */
int nif_query_multi_workspace_bytes(int64_t n, size_t* bytes);

/* The intersection query continued across voxels.  Each ray visits the occupied deformed voxels it
 * crosses in order of (t_in, id) -- the first by the BVH, each next one the successor of the
 * one before, which is the neighbour across the exit face on a conforming lattice and skips empty
 * gaps (R22) -- and the network is evaluated on each voxel's rest-space segment exactly as in
 * nif_query.  The walk stops at the first voxel whose predicted occlusion is >= 0.5; `out` then holds
 * that voxel's id, t_in, t_out and head outputs (dist_total = t_in + distance is the ray parameter of
 * the predicted hit) and walk->dist_accum the literal segmented sum of P:61.  1 <= max_steps <= 4096.
 * Flags as nif_query (not NIF_TRAVERSE_ONLY).  Enqueues max_steps rounds of
 * {successor traversal, encode+MLP, accept/continue} on `stream`; rounds with no ray left are empty
 * launches.  Does not synchronise.  All pointers DEVICE. */
int nif_query_multi(const nif_bvh* bvh, const nif_net* net, const nif_ray_batch* rays,
                    const nif_query_out* out, const nif_walk_out* walk, int32_t max_steps,
                    void* workspace, size_t workspace_bytes, unsigned flags, void* stream);

/* -------- end-to-end with HOST buffers ---------------------------------------------------- */

/* Staging for nif_query_host: three slots of device buffers for `chunk_rays` rays each (inputs,
 * outputs, query workspace), one stream per slot.  chunk_rays >= 1. */
int nif_stage_create(int64_t chunk_rays, nif_stage** out);
void nif_stage_destroy(nif_stage* stage);

/* Same query with HOST pointers in `rays` and `out` (pinned memory recommended; pageable
 * works but copies synchronously).  Splits the batch into chunks, overlapping the host->device
 * copy of chunk i+1, the kernels of chunk i and the device->host copy of chunk i-1 (the first
 * chunks are shorter than chunk_rays so that the device->host stream starts early).
 * SYNCHRONISES: on return every output is in host memory. */
int nif_query_host(const nif_bvh* bvh, const nif_net* net, nif_stage* stage,
                   const nif_ray_batch* rays_host, const nif_query_out* out_host, unsigned flags);

/* The same with a COMPACT return: voxel_id, t_in, t_out for every ray (HOST, n entries each, as above), but head
 * outputs only for the rays that hit a voxel -- a miss ray's heads are zeros by definition (R18), and on a
 * primary-ray frame most of the bytes the dense entry point copies back are those zeros.  *n_hit receives the
 * number of hit rays; row i (0 <= i < *n_hit) of every head array in `out_host` (HOST, capacity n rows) holds the
 * outputs of ray hit_ray_host[i] (HOST, capacity n).  Rows are grouped by staging chunk and, inside a chunk,
 * by the voxel the ray hit; no other order is promised.  raw_logits and the hit-position outputs are not
 * available in this form (must be NULL); NIF_OCCLUSION_ONLY writes only `occlusion`.  SYNCHRONISES. */
int nif_query_host_compact(const nif_bvh* bvh, const nif_net* net, nif_stage* stage,
                           const nif_ray_batch* rays_host, const nif_query_out* out_host,
                           int32_t* hit_ray_host, int64_t* n_hit, unsigned flags);

/* -------- the query without any allocation ------------------------------------------------- */

/* nif_query for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): the same steps (a1)-(a5), the same kernels, the same outputs and
 * flags as nif_query -- but the scratch (hit counter, hit-ray bins, hit list) lives in a device array that is
 * part of the library image instead of a caller workspace.
 *   - Limit: rays->n <= NIF_STATIC_MAX_RAYS (2,097,152 = one 1920x1080 frame and a bit); a larger batch
 *     returns NIF_ERR_STATIC_LIMIT and enqueues nothing.  Use nif_query with your own workspace beyond it.
 *   - Cost: every GPU on which the library is loaded holds NIF_STATIC_SCRATCH_BYTES (24 MiB) of device memory
 *     until the process exits, whether or not this entry point is ever called.
 *   - The call makes no cudaMalloc / cudaFree and calls no allocating library routine: it enqueues one
 *     cudaMemsetAsync and the kernels on `stream` and returns without synchronising.  The first call made with
 *     a given device current looks the array's device address up (cudaGetSymbolAddress, once per device, with
 *     that device current): make that first call outside a graph capture.
 *   - Sharing: ALL calls on a device use the one array, which keeps the previous call's contents; the parts
 *     that must start at zero (header, bin counters) are cleared on `stream` at the start of each call.  Calls
 *     are safe back to back on one stream; calls whose GPU work can overlap (different streams without an
 *     ordering between them, or concurrent host threads on different streams) RACE on the array and give
 *     wrong results.  nif_query_last_hit_count is not available for it (no workspace pointer to hand in).
 * All pointers as in nif_query: `rays`, `out` DEVICE arrays owned by the caller.  Errors: those of nif_query,
 * plus NIF_ERR_STATIC_LIMIT. */
#define NIF_STATIC_MAX_RAYS      2097152
#define NIF_STATIC_SCRATCH_BYTES 25166336      /* 64 B header + 8 MiB bins + 8 B per ray, rounded as nif_query_workspace_bytes */
int nif_query_static(const nif_bvh* bvh, const nif_net* net, const nif_ray_batch* rays,
                     const nif_query_out* out, unsigned flags, void* stream);

/* -------- diagnostics --------------------------------------------------------------------- */

/* Counters of the last nif_query on this workspace: hit rays found by the traversal.  Reads the 64-byte
 * scratch header back; SYNCHRONISES `stream`.  Returns NIF_ERR_INTERNAL if a per-ray traversal stack
 * overflowed during that query (the hierarchy is at most 9 levels deep for nv <= 512 and the stack holds
 * 7 entries per level, so this cannot happen; it is a status instead of a silent truncation). */
int nif_query_last_hit_count(const void* workspace, void* stream, int64_t* n_hit);

/* Per-kernel timing of nif_query (bench.py's roofline figure is taken from it).  After
 * nif_profile_enable(1) every nif_query records CUDA events on its stream before the traversal
 * kernel, between it and the encode+MLP kernel, and after; up to 512 queries are remembered.
 * nif_profile_read SYNCHRONISES on those events, returns the summed kernel milliseconds of the
 * remembered queries and forgets them.  nif_profile_enable(0) switches the events off again. */
int nif_profile_enable(int on);
int nif_profile_read(double* traverse_ms, double* network_ms, int64_t* n_queries);

/* Gather probes: the denominators of the gather roofline.  All SMs issue independent
 * 4-byte loads into the DEVICE buffer `buf` (`bytes` rounded down to a power-of-two number of 32-byte sectors),
 * `iters` batches of 8 loads per thread, 512-thread blocks.
 *   mode 0, "divergent": every lane reads its own pseudo-random sector (its own 128-byte line), as the hashed
 *           levels of the encoding do; a warp load is 32 L1 wavefronts, so this is the L1/LSU divergent-access
 *           ceiling.  Returned rate: lane loads = wavefronts = sectors per second.
 *   mode 1, "coalesced sectors": a warp reads one pseudo-random 128-byte line (4 sectors, 8 lanes each); one
 *           wavefront moves 4 sectors, so the rate is what L2 (a buffer that fits it) or HBM (a larger one)
 *           delivers to the SMs.  Returned rate: 32-byte sectors per second.
 * `smem_bytes` of (untouched) dynamic shared memory per block shrink the L1 data cache to what a kernel with
 * that footprint is left with (4 blocks per SM, 2 above 56 KiB, 1 above 113 KiB).  Best of 3 timed launches
 * (its milliseconds in *ms, optional).  SYNCHRONISES. */
int nif_probe_gather(const void* buf, size_t bytes, int iters, size_t smem_bytes, int mode, void* stream,
                     double* sectors_per_s, double* ms);

/* Kernels launched by the library since load (every nif_* call adds its launches). */
int64_t nif_kernel_launch_count(void);

const char* nif_error_string(int status);

#ifdef __cplusplus
}
#endif
#endif /* NIF_H_ */
