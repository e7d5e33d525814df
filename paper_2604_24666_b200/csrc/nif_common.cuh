// nif_common.cuh -- internal types shared by the CUDA translation units of libnif.so.
// Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include <math.h>

#include "nif.h"

#define NIF_MAX_LEVELS 16
#define NIF_MAX_LAYERS 9      // hidden_layers (<= 8) + output layer
#define NIF_MAX_BANDS 8

// One node of the 8-wide hierarchy over deformed voxels.
// Children are the non-empty octants of an octree cell of the REST lattice; the boxes are the
// exact fp32 min/max of the DEFORMED voxels below them, so boxes nest exactly and culling is
// bit-exactly conservative (R10).  256 bytes = two 128 B lines.
struct __align__(16) NifNode {
    float lo[3][8];        // [axis][child]
    float hi[3][8];
    uint32_t child[8];     // is_brick ? rest-space voxel id : node index
    uint32_t mask;         // bit c set <=> child c exists
    uint32_t is_brick;     // children are voxels (lowest level)
    uint32_t pad[6];       // pad[0]: brick -> voxel id of octant 0; inner -> index of the first existing child
                           // (children of a node are consecutive nodes), so child ids need no lookup
};
static_assert(sizeof(NifNode) == 256, "NifNode must be 256 bytes");

struct nif_bvh {
    int32_t nv;
    int32_t n_occupied;
    int32_t n_nodes;
    int32_t depth;
    int32_t root;          // node index, -1 if the grid is empty
    float lo[3], hi[3];
    float theta_max, bend_k;
    int32_t local_inverse; // built from a user lattice: map back with the voxel-local inverse (R27)
    const float4* lattice; // device, (nv+1)^3
    const NifNode* nodes;  // device
    // kept for nif_bvh_refit: the topology (masks, offsets, node ranges) is pose-independent
    char* ws;              // caller workspace the BVH lives in
    size_t node_capacity;
    uint32_t level_base[12];
    uint32_t top_iy;       // max (iy+1) over occupied voxels: fold-over check (R7)
};

// Encoding geometry handed to kernels by value.
struct NifEnc {
    int32_t bands, levels, log2_T, feat;
    int32_t res[NIF_MAX_LEVELS];
    uint32_t dense_mask;   // bit l set <=> level l is dense ((N+1)^3 <= T)
    int32_t mode;          // NIF_ENC_COMPOSE | NIF_ENC_CONCAT
};

struct nif_net {
    nif_net_desc desc;
    NifEnc enc;
    int32_t d_in;
    const void* table;                 // borrowed device pointer (or table_owned)
    void* table_owned;                 // feat == 3: the library's copy padded to 4 features per entry
    void* w_plain[NIF_MAX_LAYERS];     // device copies, row-major (fan_out, fan_in), net dtype
    void* w_tc;                        // device: tensor-core operand images (NIF_F16 only)
    size_t w_tc_bytes;
    size_t w_tc_layer_off[NIF_MAX_LAYERS];
    int tc_supported;
};

// per-query scratch layout (device):
//   [NifQueryScratch header][uint32 bin_count[NIF_MAX_BINS]][uint32 rank[n]][int32 hit_list[n]]
// Hit rays are binned by the voxel they hit (bricks of voxels when nv^3 > NIF_MAX_BINS) so that the
// 128-ray tiles of the encode kernel are spatially coherent in rest space.
#define NIF_MAX_BINS (1u << 21)
struct NifQueryScratch {
    unsigned long long n_hit;          // cursor of the bin allocation = hit rays once k_bin_offsets has run
    unsigned int tile_counter;         // dynamic ray fetch counter of the traversal kernel
    unsigned int pad[13];              // [0] coherent decision, [1] votes, [2] finished blocks, [3] stack overflow status,
                                       // [4] tile counter of the encode kernel, [5] image width (0: batch is not an image), [6] its detection
};
static_assert(sizeof(NifQueryScratch) == 64, "scratch header is 64 bytes");

struct NifQueryWs {                    // pointers into the caller's workspace
    NifQueryScratch* scratch;
    uint32_t* bin_count;
    uint32_t* rank;
    int32_t* hit_list;
    uint32_t n_bins;
    int bin_shift, nvb;                // bin = (ix >> s) + nvb * ((iy >> s) + nvb * (iz >> s))
};

// nif_query_poses: what the kernels need of one pose's BVH (device array, one entry per pose)
#define NIF_MAX_POSES 64
struct NifPoseDesc {
    const NifNode* nodes;
    const float4* lat;
    float lo[3], hi[3];                // root box
    int32_t root;
    float theta_max, bend_k;
    int32_t local_inverse;
    int32_t pad[2];
};
static_assert(sizeof(NifPoseDesc) == 64, "pose descriptor is 64 bytes");

struct NifPoseBatch {                  // NULL pointers outside nif_query_poses
    const NifPoseDesc* poses;          // device
    const int32_t* pose_id;            // device, per ray
    int n_poses;
};

// one round of the multi-voxel walk (nif_walk.cu): round 0 is the plain nearest-voxel query over all
// rays; rounds >= 1 run over `ray_list` (rays still walking) and look for each ray's next voxel
struct NifWalkRound {
    int round;
    const int32_t* ray_list;           // device, *n_list entries
    const unsigned int* n_list;        // device
    float* dist_accum;                 // nif_walk_out.dist_accum
};

extern "C" void nif_count_launch(int n);

#define NIF_CUDA_TRY(expr)                                   \
    do {                                                     \
        cudaError_t _e = (expr);                             \
        if (_e != cudaSuccess) { (void)cudaGetLastError(); return NIF_ERR_CUDA; } \
    } while (0)

// launchers implemented in the individual .cu files
int nif_launch_traverse(const nif_bvh* bvh, const nif_ray_batch* rays, const nif_query_out* out,
                        const NifQueryWs* ws, unsigned flags, const NifWalkRound* walk, cudaStream_t stream,
                        const NifPoseBatch* batch = nullptr);
int nif_launch_bin_hits(const nif_bvh* bvh, const nif_ray_batch* rays, const nif_query_out* out,
                        const NifQueryWs* ws, const NifWalkRound* walk, cudaStream_t stream);
int nif_launch_clear_bins(const NifQueryWs* ws, const unsigned int* n_list, cudaStream_t stream);
void nif_query_ws_layout(const nif_bvh* bvh, int64_t n, void* workspace, NifQueryWs* ws);
int nif_launch_ffma(const nif_bvh* bvh, const nif_net* net, const nif_ray_batch* rays,
                    const nif_query_out* out, const NifQueryScratch* scratch,
                    const int32_t* hit_list, unsigned flags, cudaStream_t stream,
                    const NifPoseBatch* batch = nullptr);
int nif_launch_fused_tc(const nif_bvh* bvh, const nif_net* net, const nif_ray_batch* rays,
                        const nif_query_out* out, NifQueryScratch* scratch,
                        const int32_t* hit_list, unsigned flags, cudaStream_t stream,
                        const NifPoseBatch* batch = nullptr);
int nif_tc_pack_weights(nif_net* net, cudaStream_t stream);
int nif_tc_supported(const nif_net_desc* d);

extern "C" int nif_device_supported(void);
// multiprocessor count of the CURRENT device (cached per device ordinal); <= 0 on error
int nif_sm_count();

// per-kernel event timing hooks (nif_probe.cu); slot < 0 = profiling off
int nif_prof_begin(cudaStream_t stream);
void nif_prof_mark(int slot, int which, cudaStream_t stream);
