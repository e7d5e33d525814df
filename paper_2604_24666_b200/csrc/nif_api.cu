// nif_api.cu -- C ABI glue of libnif.so (include/nif.h): argument validation, network object,
// nif_query (enqueue only), the host-buffer end-to-end entry and diagnostics.
#include "nif_common.cuh"

#include <atomic>
#include <new>
#include <string.h>

extern "C" int nif_device_supported(void);

namespace {
std::atomic<long long> g_launches{0};
inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
inline size_t elem_bytes(int dtype) { return dtype == NIF_F16 ? 2 : 4; }
}  // namespace

int nif_sm_count()
{
    static std::atomic<int> cache[64];                        // 0 = not asked yet
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return -1; }
    if (dev >= 0 && dev < 64) {
        const int c = cache[dev].load(std::memory_order_relaxed);
        if (c > 0) return c;
    }
    int n = 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { (void)cudaGetLastError(); return -1; }
    if (dev >= 0 && dev < 64) cache[dev].store(n, std::memory_order_relaxed);
    return n;
}

extern "C" void nif_count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
extern "C" int64_t nif_kernel_launch_count(void) { return (int64_t)g_launches.load(); }

extern "C" const char* nif_error_string(int status)
{
    switch (status) {
        case NIF_OK: return "ok";
        case NIF_ERR_INVALID_ARG: return "invalid argument";
        case NIF_ERR_UNSUPPORTED: return "unsupported shape, dtype or device (needs sm_100)";
        case NIF_ERR_DEFORM_SINGULAR: return "deformation folds over (bend k*y >= 1)";
        case NIF_ERR_WORKSPACE: return "workspace too small or misaligned";
        case NIF_ERR_CUDA: return "CUDA runtime error";
        case NIF_ERR_INTERNAL: return "internal limit exceeded (traversal stack overflow): results invalid";
        case NIF_ERR_STATIC_LIMIT: return "batch exceeds NIF_STATIC_MAX_RAYS, the size nif_query_static's fixed scratch serves";
        default: return "unknown status";
    }
}

// ---------------------------------------------------------------------------------------------
// network
// ---------------------------------------------------------------------------------------------
namespace {
// feat == 3 (the paper's own configuration, "feature dim 3"): entries are stored padded to 4
// features (8- or 16-byte aligned vector loads) and the first layer gets a zero column per pad
// feature, so the network function is unchanged.
template <typename T>
__global__ void k_pad_table_3to4(const T* __restrict__ src, T* __restrict__ dst, size_t n_entries)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_entries) return;
    dst[4 * i] = src[3 * i]; dst[4 * i + 1] = src[3 * i + 1]; dst[4 * i + 2] = src[3 * i + 2];
    dst[4 * i + 3] = (T)0.0f;
}
template <typename T>
__global__ void k_pad_w1_3to4(const T* __restrict__ src, T* __restrict__ dst, int rows, int groups)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;        // over rows * groups * 4
    if (i >= rows * groups * 4) return;
    const int f = i & 3, g = (i >> 2) % groups, r = i / (groups * 4);
    dst[i] = f < 3 ? src[(size_t)r * groups * 3 + (size_t)g * 3 + f] : (T)0.0f;
}
}  // namespace

static int validate_desc(const nif_net_desc* d)
{
    if (!d || !d->level_res) return NIF_ERR_INVALID_ARG;
    if (d->pe_bands < 0 || d->pe_bands > NIF_MAX_BANDS) return NIF_ERR_INVALID_ARG;
    if (d->levels < 1 || d->levels > NIF_MAX_LEVELS) return NIF_ERR_INVALID_ARG;
    if (d->log2_T < 4 || d->log2_T > 24) return NIF_ERR_INVALID_ARG;
    if (d->hidden_layers < 1 || d->hidden_layers > NIF_MAX_LAYERS - 1) return NIF_ERR_INVALID_ARG;
    if (d->dtype != NIF_F32 && d->dtype != NIF_F16) return NIF_ERR_INVALID_ARG;
    for (int l = 0; l < d->levels; ++l)
        if (d->level_res[l] < 1 || d->level_res[l] > (1 << 20)) return NIF_ERR_INVALID_ARG;
    if (d->feat < 1 || d->feat > 4) return NIF_ERR_UNSUPPORTED;
    if (d->enc_mode != NIF_ENC_COMPOSE && d->enc_mode != NIF_ENC_CONCAT) return NIF_ERR_INVALID_ARG;
    if (d->enc_mode == NIF_ENC_CONCAT && d->feat == 3) return NIF_ERR_UNSUPPORTED;
    if (d->width < 16 || d->width > 128 || (d->width % 16) != 0) return NIF_ERR_UNSUPPORTED;
    return NIF_OK;
}

extern "C" int nif_net_create(const nif_net_desc* desc, const void* table, const void* const* weights,
                              void* stream_, nif_net** out)
{
    int rc = validate_desc(desc);
    if (rc != NIF_OK) return rc;
    if (!table || !weights || !out) return NIF_ERR_INVALID_ARG;
    for (int i = 0; i <= desc->hidden_layers; ++i)
        if (!weights[i]) return NIF_ERR_INVALID_ARG;
    if (!nif_device_supported()) return NIF_ERR_UNSUPPORTED;
    cudaStream_t stream = (cudaStream_t)stream_;

    nif_net* net = new (std::nothrow) nif_net();
    if (!net) return NIF_ERR_CUDA;
    memset(net, 0, sizeof(*net));
    net->desc = *desc;
    net->desc.level_res = nullptr;                 // host pointer is not kept
    net->enc.bands = desc->pe_bands; net->enc.levels = desc->levels;
    net->enc.log2_T = desc->log2_T; net->enc.feat = desc->feat;
    net->enc.dense_mask = 0;
    net->enc.mode = desc->enc_mode;
    const unsigned long long T = 1ull << desc->log2_T;
    for (int l = 0; l < desc->levels; ++l) {
        net->enc.res[l] = desc->level_res[l];
        const unsigned long long np1 = (unsigned long long)desc->level_res[l] + 1ull;   // 64-bit compare (R6)
        if (np1 * np1 * np1 <= T) net->enc.dense_mask |= 1u << l;
    }
    const bool pad3 = desc->feat == 3;
    const int feat = pad3 ? 4 : desc->feat;
    net->desc.feat = feat; net->enc.feat = feat;
    const int groups = 2 * (1 + 2 * desc->pe_bands) * desc->levels;      // (endpoint, sample, level) triples
    net->d_in = desc->enc_mode == NIF_ENC_CONCAT ? 2 * (3 + 6 * desc->pe_bands + desc->levels * feat) : groups * feat;
    net->table = table;
    const size_t eb = elem_bytes(desc->dtype);
    if (pad3) {
        const size_t n_entries = (size_t)desc->levels << desc->log2_T;
        if (cudaMalloc(&net->table_owned, n_entries * 4 * eb) != cudaSuccess) {
            (void)cudaGetLastError(); nif_net_destroy(net); return NIF_ERR_CUDA;
        }
        const unsigned blocks = (unsigned)((n_entries + 255) / 256);
        if (desc->dtype == NIF_F16)
            k_pad_table_3to4<__half><<<blocks, 256, 0, stream>>>((const __half*)table, (__half*)net->table_owned, n_entries);
        else
            k_pad_table_3to4<float><<<blocks, 256, 0, stream>>>((const float*)table, (float*)net->table_owned, n_entries);
        nif_count_launch(1);
        net->table = net->table_owned;
    }
    for (int i = 0; i <= desc->hidden_layers; ++i) {
        const size_t fan_out = i == desc->hidden_layers ? NIF_N_OUT : (size_t)desc->width;
        const size_t fan_in = i == 0 ? (size_t)net->d_in : (size_t)desc->width;
        const size_t bytes = fan_out * fan_in * eb;
        cudaError_t e = cudaMalloc(&net->w_plain[i], bytes);
        if (e == cudaSuccess) {
            if (i == 0 && pad3) {
                const int total = (int)fan_out * groups * 4;
                if (desc->dtype == NIF_F16)
                    k_pad_w1_3to4<__half><<<(total + 255) / 256, 256, 0, stream>>>((const __half*)weights[0], (__half*)net->w_plain[0], (int)fan_out, groups);
                else
                    k_pad_w1_3to4<float><<<(total + 255) / 256, 256, 0, stream>>>((const float*)weights[0], (float*)net->w_plain[0], (int)fan_out, groups);
                nif_count_launch(1);
                e = cudaGetLastError();
            } else {
                e = cudaMemcpyAsync(net->w_plain[i], weights[i], bytes, cudaMemcpyDeviceToDevice, stream);
            }
        }
        if (e != cudaSuccess) { (void)cudaGetLastError(); nif_net_destroy(net); return NIF_ERR_CUDA; }
    }
    net->tc_supported = nif_tc_supported(&net->desc);
    if (net->tc_supported) {
        rc = nif_tc_pack_weights(net, stream);
        if (rc != NIF_OK) { nif_net_destroy(net); return rc; }
    }
    if (cudaStreamSynchronize(stream) != cudaSuccess) { (void)cudaGetLastError(); nif_net_destroy(net); return NIF_ERR_CUDA; }
    *out = net;
    return NIF_OK;
}

extern "C" void nif_net_destroy(nif_net* net)
{
    if (!net) return;
    for (int i = 0; i < NIF_MAX_LAYERS; ++i)
        if (net->w_plain[i]) cudaFree(net->w_plain[i]);
    if (net->w_tc) cudaFree(net->w_tc);
    if (net->table_owned) cudaFree(net->table_owned);
    delete net;
}

extern "C" int nif_net_uses_tensor_cores(const nif_net* net)
{
    if (!net) return NIF_ERR_INVALID_ARG;
    return net->desc.dtype == NIF_F16 && net->tc_supported ? 1 : 0;
}

// ---------------------------------------------------------------------------------------------
// query
// ---------------------------------------------------------------------------------------------
extern "C" int nif_query_workspace_bytes(int64_t n, size_t* bytes)
{
    if (!bytes || n < 0 || n > 0x7fffffffLL) return NIF_ERR_INVALID_ARG;
    *bytes = align_up(sizeof(NifQueryScratch) + (size_t)NIF_MAX_BINS * 4 + (size_t)n * 8, 256) + 256;
    return NIF_OK;
}

void nif_query_ws_layout(const nif_bvh* bvh, int64_t n, void* workspace, NifQueryWs* ws)
{
    ws->scratch = (NifQueryScratch*)workspace;
    ws->bin_count = (uint32_t*)((char*)workspace + sizeof(NifQueryScratch));
    ws->rank = ws->bin_count + NIF_MAX_BINS;
    ws->hit_list = (int32_t*)(ws->rank + n);
    ws->bin_shift = 0;
    for (;;) {                                               // bricks of 2^s voxels until the bins fit
        ws->nvb = (bvh->nv + (1 << ws->bin_shift) - 1) >> ws->bin_shift;
        if ((unsigned long long)ws->nvb * ws->nvb * ws->nvb <= NIF_MAX_BINS) break;
        ++ws->bin_shift;
    }
    ws->n_bins = (uint32_t)(ws->nvb * ws->nvb * ws->nvb);
}

int nif_validate_query(const nif_bvh* bvh, const nif_net* net, const nif_ray_batch* rays,
                       const nif_query_out* out, unsigned flags);

static int validate_query(const nif_bvh* bvh, const nif_net* net, const nif_ray_batch* rays,
                          const nif_query_out* out, unsigned flags)
{
    if (!bvh || !rays || !out) return NIF_ERR_INVALID_ARG;
    if (rays->n < 0 || rays->n > 0x7fffffffLL) return NIF_ERR_INVALID_ARG;
    if (rays->n == 0) return NIF_OK;
    if (!rays->origin || !rays->dir) return NIF_ERR_INVALID_ARG;
    if (!out->voxel_id || !out->t_in || !out->t_out) return NIF_ERR_INVALID_ARG;
    if (flags & NIF_TRAVERSE_ONLY) return NIF_OK;
    if (!net || !out->occlusion) return NIF_ERR_INVALID_ARG;
    if (!(flags & NIF_OCCLUSION_ONLY) &&
        (!out->distance || !out->dist_total || !out->normal || !out->albedo || !out->material_logits))
        return NIF_ERR_INVALID_ARG;
    return NIF_OK;
}

int nif_validate_query(const nif_bvh* bvh, const nif_net* net, const nif_ray_batch* rays,
                       const nif_query_out* out, unsigned flags)
{
    return validate_query(bvh, net, rays, out, flags);
}

extern "C" int nif_query(const nif_bvh* bvh, const nif_net* net, const nif_ray_batch* rays,
                         const nif_query_out* out, void* workspace, size_t workspace_bytes,
                         unsigned flags, void* stream_)
{
    int rc = validate_query(bvh, net, rays, out, flags);
    if (rc != NIF_OK) return rc;
    if (rays->n == 0) return NIF_OK;
    size_t need = 0;
    nif_query_workspace_bytes(rays->n, &need);
    if (!workspace || ((uintptr_t)workspace & 255u) != 0 || workspace_bytes < need) return NIF_ERR_WORKSPACE;
    cudaStream_t stream = (cudaStream_t)stream_;
    NifQueryWs ws;
    nif_query_ws_layout(bvh, rays->n, workspace, &ws);
    NifQueryScratch* scratch = ws.scratch;
    int32_t* hit_list = ws.hit_list;
    const bool traverse_only = (flags & NIF_TRAVERSE_ONLY) != 0;
    NIF_CUDA_TRY(cudaMemsetAsync(workspace, 0, sizeof(NifQueryScratch) + (traverse_only ? 0 : (size_t)ws.n_bins * 4), stream));
    const int prof = nif_prof_begin(stream);                 // -1 unless nif_profile_enable(1)
    rc = nif_launch_traverse(bvh, rays, out, &ws, flags, nullptr, stream);
    if (rc == NIF_OK && !traverse_only) rc = nif_launch_bin_hits(bvh, rays, out, &ws, nullptr, stream);
    nif_prof_mark(prof, 1, stream);
    if (rc != NIF_OK || traverse_only) return rc;
    const bool use_tc = net->desc.dtype == NIF_F16 && net->tc_supported && !(flags & NIF_ENGINE_FFMA);
    if (use_tc) rc = nif_launch_fused_tc(bvh, net, rays, out, scratch, hit_list, flags, stream);
    else rc = nif_launch_ffma(bvh, net, rays, out, scratch, hit_list, flags, stream);
    nif_prof_mark(prof, 2, stream);
    return rc;
}

namespace {
// pose descriptors travel as a KERNEL PARAMETER (16 x 64 B per launch), not through a host-to-device copy:
// nif_query_poses stays enqueue-only and capturable in a CUDA graph (a captured memcpy would keep a pointer
// to the caller's stack); a replay uses the descriptors as they were at capture time
struct PoseDescPack { NifPoseDesc d[16]; };
__global__ void k_write_pose_desc(const PoseDescPack pack, NifPoseDesc* __restrict__ dst, int n)
{
    const int i = threadIdx.x >> 4, w = threadIdx.x & 15;            // 16 words of 4 bytes per descriptor
    if (i < n) reinterpret_cast<uint32_t*>(dst + i)[w] = reinterpret_cast<const uint32_t*>(&pack.d[i])[w];
}
}  // namespace

// Several poses of one object in ONE query: every ray names its pose (SURVEY 8(f) f2, B:9 "one BVH per pose ...
// network shared across all poses").  Hit rays are binned by rest-space voxel across poses, so the encode tiles
// mix rays of all poses that hit the same voxel: they look up the same table cells.
extern "C" int nif_query_poses_workspace_bytes(int64_t n, size_t* bytes)
{
    size_t q = 0;
    int rc = nif_query_workspace_bytes(n, &q);
    if (rc != NIF_OK) return rc;
    *bytes = align_up(q, 256) + align_up(sizeof(NifPoseDesc) * NIF_MAX_POSES, 256);
    return NIF_OK;
}

extern "C" int nif_query_poses(const nif_bvh* const* bvhs, int32_t n_poses, const nif_net* net,
                               const nif_ray_batch* rays, const int32_t* pose_id, const nif_query_out* out,
                               void* workspace, size_t workspace_bytes, unsigned flags, void* stream_)
{
    if (!bvhs || n_poses < 1 || n_poses > NIF_MAX_POSES || !pose_id) return NIF_ERR_INVALID_ARG;
    for (int i = 0; i < n_poses; ++i) {
        if (!bvhs[i]) return NIF_ERR_INVALID_ARG;
        if (bvhs[i]->nv != bvhs[0]->nv || bvhs[i]->local_inverse != bvhs[0]->local_inverse) return NIF_ERR_INVALID_ARG;
    }
    int rc = validate_query(bvhs[0], net, rays, out, flags);
    if (rc != NIF_OK) return rc;
    if (flags & NIF_PROBE_SKIP_GATHER) return NIF_ERR_INVALID_ARG;
    if (rays->n == 0) return NIF_OK;
    size_t need = 0, qbytes = 0;
    nif_query_poses_workspace_bytes(rays->n, &need);
    nif_query_workspace_bytes(rays->n, &qbytes);
    if (!workspace || ((uintptr_t)workspace & 255u) != 0 || workspace_bytes < need) return NIF_ERR_WORKSPACE;
    cudaStream_t stream = (cudaStream_t)stream_;
    NifQueryWs ws;
    nif_query_ws_layout(bvhs[0], rays->n, workspace, &ws);
    NifPoseDesc* d_desc = (NifPoseDesc*)((char*)workspace + align_up(qbytes, 256));
    for (int base = 0; base < n_poses; base += 16) {
        PoseDescPack pack;
        memset(&pack, 0, sizeof(pack));
        const int m = n_poses - base < 16 ? n_poses - base : 16;
        for (int i = 0; i < m; ++i) {
            const nif_bvh* b = bvhs[base + i];
            NifPoseDesc& d = pack.d[i];
            d.nodes = b->nodes; d.lat = b->lattice; d.root = b->root;
            for (int a = 0; a < 3; ++a) { d.lo[a] = b->lo[a]; d.hi[a] = b->hi[a]; }
            d.theta_max = b->theta_max; d.bend_k = b->bend_k; d.local_inverse = b->local_inverse;
        }
        k_write_pose_desc<<<1, 256, 0, stream>>>(pack, d_desc + base, m);
        nif_count_launch(1);
    }
    NIF_CUDA_TRY(cudaGetLastError());
    NifPoseBatch batch{d_desc, pose_id, n_poses};
    const bool traverse_only = (flags & NIF_TRAVERSE_ONLY) != 0;
    NIF_CUDA_TRY(cudaMemsetAsync(workspace, 0, sizeof(NifQueryScratch) + (traverse_only ? 0 : (size_t)ws.n_bins * 4), stream));
    const int prof = nif_prof_begin(stream);
    // the coherence vote looks at ray geometry only; its "extent" comes from the first pose
    rc = nif_launch_traverse(bvhs[0], rays, out, &ws, flags, nullptr, stream, &batch);
    if (rc == NIF_OK && !traverse_only) rc = nif_launch_bin_hits(bvhs[0], rays, out, &ws, nullptr, stream);
    nif_prof_mark(prof, 1, stream);
    if (rc != NIF_OK || traverse_only) return rc;
    const bool use_tc = net->desc.dtype == NIF_F16 && net->tc_supported && !(flags & NIF_ENGINE_FFMA);
    if (use_tc) rc = nif_launch_fused_tc(bvhs[0], net, rays, out, ws.scratch, ws.hit_list, flags, stream, &batch);
    else rc = nif_launch_ffma(bvhs[0], net, rays, out, ws.scratch, ws.hit_list, flags, stream, &batch);
    nif_prof_mark(prof, 2, stream);
    return rc;
}

extern "C" int nif_query_last_hit_count(const void* workspace, void* stream_, int64_t* n_hit)
{
    if (!workspace || !n_hit) return NIF_ERR_INVALID_ARG;
    NifQueryScratch h;
    cudaStream_t stream = (cudaStream_t)stream_;
    NIF_CUDA_TRY(cudaMemcpyAsync(&h, workspace, sizeof(h), cudaMemcpyDeviceToHost, stream));
    NIF_CUDA_TRY(cudaStreamSynchronize(stream));
    *n_hit = (int64_t)h.n_hit;
    // pad[3]: set by the traversal kernels if a per-ray stack ever overflowed (cannot happen for nv <= 512,
    // see STACK_MAX in nif_traverse.cu): the results of that query are not trustworthy
    return h.pad[3] ? NIF_ERR_INTERNAL : NIF_OK;
}

// ---------------------------------------------------------------------------------------------
// end-to-end with HOST buffers: chunked, NSLOT slots each on its own stream, so the H2D copy of
// chunk i+1, the kernels of chunk i and the D2H copy of chunk i-1 overlap (two copy engines).
// ---------------------------------------------------------------------------------------------
namespace { constexpr int NSLOT = 3; }

struct nif_stage {
    int64_t chunk;
    cudaStream_t stream[NSLOT];
    char* dev[NSLOT];            // one allocation per slot
    size_t slot_bytes, ws_bytes;
    // offsets inside a slot
    size_t o_origin, o_dir, o_vid, o_tin, o_tout, o_occ, o_dist, o_dtot, o_nrm, o_alb, o_mat, o_raw, o_hit, o_hitr, o_ws;
    // nif_query_host_compact: compacted head rows of the chunk's hit rays + their ray indices
    size_t c_ray, c_occ, c_dist, c_dtot, c_nrm, c_alb, c_mat;
    unsigned long long* h_count;     // pinned host, NSLOT hit counts
    cudaEvent_t ev[NSLOT];
};

extern "C" int nif_stage_create(int64_t chunk_rays, nif_stage** out)
{
    if (!out || chunk_rays < 1 || chunk_rays > 0x7fffffffLL) return NIF_ERR_INVALID_ARG;
    if (!nif_device_supported()) return NIF_ERR_UNSUPPORTED;
    nif_stage* s = new (std::nothrow) nif_stage();
    if (!s) return NIF_ERR_CUDA;
    memset(s, 0, sizeof(*s));
    s->chunk = chunk_rays;
    const size_t n = (size_t)chunk_rays;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
    s->o_origin = take(n * 12); s->o_dir = take(n * 12);
    s->o_vid = take(n * 4); s->o_tin = take(n * 4); s->o_tout = take(n * 4);
    s->o_occ = take(n * 4); s->o_dist = take(n * 4); s->o_dtot = take(n * 4);
    s->o_nrm = take(n * 12); s->o_alb = take(n * 12); s->o_mat = take(n * 16); s->o_raw = take(n * 48);
    s->o_hit = take(n * 12); s->o_hitr = take(n * 12);
    nif_query_workspace_bytes(chunk_rays, &s->ws_bytes);
    s->o_ws = take(s->ws_bytes);
    s->c_ray = take(n * 4); s->c_occ = take(n * 4); s->c_dist = take(n * 4); s->c_dtot = take(n * 4);
    s->c_nrm = take(n * 12); s->c_alb = take(n * 12); s->c_mat = take(n * 16);
    s->slot_bytes = off;
    if (cudaHostAlloc((void**)&s->h_count, NSLOT * sizeof(unsigned long long), cudaHostAllocDefault) != cudaSuccess) {
        (void)cudaGetLastError(); delete s; return NIF_ERR_CUDA;
    }
    for (int i = 0; i < NSLOT; ++i) {
        if (cudaStreamCreateWithFlags(&s->stream[i], cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&s->ev[i], cudaEventDisableTiming) != cudaSuccess ||
            cudaMalloc((void**)&s->dev[i], s->slot_bytes) != cudaSuccess) {
            (void)cudaGetLastError();
            nif_stage_destroy(s);
            return NIF_ERR_CUDA;
        }
    }
    *out = s;
    return NIF_OK;
}

extern "C" void nif_stage_destroy(nif_stage* s)
{
    if (!s) return;
    for (int i = 0; i < NSLOT; ++i) {
        if (s->dev[i]) cudaFree(s->dev[i]);
        if (s->ev[i]) cudaEventDestroy(s->ev[i]);
        if (s->stream[i]) cudaStreamDestroy(s->stream[i]);
    }
    if (s->h_count) cudaFreeHost(s->h_count);
    delete s;
}

static int query_host_enqueue(const nif_bvh* bvh, const nif_net* net, nif_stage* st,
                              const nif_ray_batch* rays, const nif_query_out* out, unsigned flags);

extern "C" int nif_query_host(const nif_bvh* bvh, const nif_net* net, nif_stage* st,
                              const nif_ray_batch* rays, const nif_query_out* out, unsigned flags)
{
    if (!st) return NIF_ERR_INVALID_ARG;
    int rc = validate_query(bvh, net, rays, out, flags);
    if (rc != NIF_OK) return rc;
    rc = query_host_enqueue(bvh, net, st, rays, out, flags);
    // success or not, nothing may still be copying into the caller's buffers when this returns
    for (int i = 0; i < NSLOT; ++i)
        if (cudaStreamSynchronize(st->stream[i]) != cudaSuccess) { (void)cudaGetLastError(); if (rc == NIF_OK) rc = NIF_ERR_CUDA; }
    return rc;
}

static int query_host_enqueue(const nif_bvh* bvh, const nif_net* net, nif_stage* st,
                              const nif_ray_batch* rays, const nif_query_out* out, unsigned flags)
{
    int rc = NIF_OK;
    const bool heads = !(flags & NIF_TRAVERSE_ONLY);
    const bool full = heads && !(flags & NIF_OCCLUSION_ONLY);
    int chunk_idx = 0;
    // the device->host copies (60 B per ray) are the bottleneck of the pipeline, so they should start as
    // early as possible: the first chunks are short (1/8, 1/4, 1/2 of the slot size), then full ones
    int64_t m = 0;
    for (int64_t begin = 0; begin < rays->n; begin += m, ++chunk_idx) {
        int64_t want = st->chunk;
        if (chunk_idx < 3 && rays->n > st->chunk) want = st->chunk >> (3 - chunk_idx);
        if (want < 1) want = 1;
        m = (rays->n - begin < want) ? rays->n - begin : want;
        const int slot = chunk_idx % NSLOT;
        cudaStream_t stream = st->stream[slot];
        char* d = st->dev[slot];
        NIF_CUDA_TRY(cudaMemcpyAsync(d + st->o_origin, rays->origin + 3 * begin, (size_t)m * 12, cudaMemcpyHostToDevice, stream));
        NIF_CUDA_TRY(cudaMemcpyAsync(d + st->o_dir, rays->dir + 3 * begin, (size_t)m * 12, cudaMemcpyHostToDevice, stream));
        nif_ray_batch rb; rb.n = m; rb.origin = (const float*)(d + st->o_origin); rb.dir = (const float*)(d + st->o_dir);
        nif_query_out qo;
        qo.voxel_id = (int32_t*)(d + st->o_vid); qo.t_in = (float*)(d + st->o_tin); qo.t_out = (float*)(d + st->o_tout);
        qo.occlusion = (float*)(d + st->o_occ); qo.distance = (float*)(d + st->o_dist);
        qo.dist_total = (float*)(d + st->o_dtot); qo.normal = (float*)(d + st->o_nrm);
        qo.albedo = (float*)(d + st->o_alb); qo.material_logits = (float*)(d + st->o_mat);
        qo.raw_logits = (heads && out->raw_logits) ? (float*)(d + st->o_raw) : nullptr;
        qo.hit_position = (full && out->hit_position) ? (float*)(d + st->o_hit) : nullptr;
        qo.hit_position_rest = (full && out->hit_position_rest) ? (float*)(d + st->o_hitr) : nullptr;
        rc = nif_query(bvh, net, &rb, &qo, d + st->o_ws, st->ws_bytes, flags, stream);
        if (rc != NIF_OK) return rc;
        auto back = [&](void* host, size_t host_off, size_t dev_off, size_t bytes) -> cudaError_t {
            return cudaMemcpyAsync((char*)host + host_off, d + dev_off, bytes, cudaMemcpyDeviceToHost, stream);
        };
        const size_t b = (size_t)begin, mm = (size_t)m;
        NIF_CUDA_TRY(back(out->voxel_id, b * 4, st->o_vid, mm * 4));
        NIF_CUDA_TRY(back(out->t_in, b * 4, st->o_tin, mm * 4));
        NIF_CUDA_TRY(back(out->t_out, b * 4, st->o_tout, mm * 4));
        if (heads) NIF_CUDA_TRY(back(out->occlusion, b * 4, st->o_occ, mm * 4));
        if (full) {
            NIF_CUDA_TRY(back(out->distance, b * 4, st->o_dist, mm * 4));
            NIF_CUDA_TRY(back(out->dist_total, b * 4, st->o_dtot, mm * 4));
            NIF_CUDA_TRY(back(out->normal, b * 12, st->o_nrm, mm * 12));
            NIF_CUDA_TRY(back(out->albedo, b * 12, st->o_alb, mm * 12));
            NIF_CUDA_TRY(back(out->material_logits, b * 16, st->o_mat, mm * 16));
        }
        if (heads && out->raw_logits) NIF_CUDA_TRY(back(out->raw_logits, b * 48, st->o_raw, mm * 48));
        if (qo.hit_position) NIF_CUDA_TRY(back(out->hit_position, b * 12, st->o_hit, mm * 12));
        if (qo.hit_position_rest) NIF_CUDA_TRY(back(out->hit_position_rest, b * 12, st->o_hitr, mm * 12));
    }
    return NIF_OK;
}


// ---------------------------------------------------------------------------------------------
// nif_query_host with a COMPACT return: ids and t for every ray, head outputs only for the rays that hit.
// A miss ray's heads are zeros by definition (R18); on a primary-ray frame 88 % of the 48 head bytes per ray
// that the dense entry point copies back over PCIe are those zeros.
// ---------------------------------------------------------------------------------------------
namespace {
struct CompactDst { int32_t* ray; float *occ, *dist, *dtot, *nrm, *alb, *mat; };

__global__ void __launch_bounds__(256)
k_compact_heads(const NifQueryScratch* __restrict__ scratch, const int32_t* __restrict__ hit_list, const nif_query_out dense,
                const CompactDst c, int32_t ray_base, unsigned flags)
{
    const long long n_hit = (long long)scratch->n_hit;
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n_hit; i += (long long)gridDim.x * 256) {
        const int32_t r = hit_list[i];
        c.ray[i] = r + ray_base;
        c.occ[i] = dense.occlusion[r];
        if (flags & NIF_OCCLUSION_ONLY) continue;
        c.dist[i] = dense.distance[r]; c.dtot[i] = dense.dist_total[r];
#pragma unroll
        for (int a = 0; a < 3; ++a) { c.nrm[3 * i + a] = dense.normal[3 * r + a]; c.alb[3 * i + a] = dense.albedo[3 * r + a]; }
#pragma unroll
        for (int a = 0; a < 4; ++a) c.mat[4 * i + a] = dense.material_logits[4 * r + a];
    }
}
}  // namespace

static int query_host_compact_enqueue(const nif_bvh* bvh, const nif_net* net, nif_stage* st, const nif_ray_batch* rays,
                                      const nif_query_out* out, int32_t* hit_ray, int64_t* n_hit_total, unsigned flags)
{
    const bool full = !(flags & NIF_OCCLUSION_ONLY);
    const int n_sm = nif_sm_count();
    if (n_sm <= 0) return NIF_ERR_CUDA;
    int64_t total = 0;
    int pending_slot = -1;
    // copies the compacted rows of the chunk in `slot` back once its hit count has arrived on the host
    auto finish = [&](int slot) -> int {
        NIF_CUDA_TRY(cudaEventSynchronize(st->ev[slot]));
        const size_t m = (size_t)st->h_count[slot], b = (size_t)total;
        cudaStream_t stream = st->stream[slot];
        char* d = st->dev[slot];
        if (m) {
            NIF_CUDA_TRY(cudaMemcpyAsync(hit_ray + b, d + st->c_ray, m * 4, cudaMemcpyDeviceToHost, stream));
            NIF_CUDA_TRY(cudaMemcpyAsync(out->occlusion + b, d + st->c_occ, m * 4, cudaMemcpyDeviceToHost, stream));
            if (full) {
                NIF_CUDA_TRY(cudaMemcpyAsync(out->distance + b, d + st->c_dist, m * 4, cudaMemcpyDeviceToHost, stream));
                NIF_CUDA_TRY(cudaMemcpyAsync(out->dist_total + b, d + st->c_dtot, m * 4, cudaMemcpyDeviceToHost, stream));
                NIF_CUDA_TRY(cudaMemcpyAsync(out->normal + 3 * b, d + st->c_nrm, m * 12, cudaMemcpyDeviceToHost, stream));
                NIF_CUDA_TRY(cudaMemcpyAsync(out->albedo + 3 * b, d + st->c_alb, m * 12, cudaMemcpyDeviceToHost, stream));
                NIF_CUDA_TRY(cudaMemcpyAsync(out->material_logits + 4 * b, d + st->c_mat, m * 16, cudaMemcpyDeviceToHost, stream));
            }
        }
        total += (int64_t)m;
        return NIF_OK;
    };
    int chunk_idx = 0;
    int64_t m = 0;
    for (int64_t begin = 0; begin < rays->n; begin += m, ++chunk_idx) {
        int64_t want = st->chunk;
        if (chunk_idx < 3 && rays->n > st->chunk) want = st->chunk >> (3 - chunk_idx);
        if (want < 1) want = 1;
        m = (rays->n - begin < want) ? rays->n - begin : want;
        const int slot = chunk_idx % NSLOT;
        cudaStream_t stream = st->stream[slot];
        char* d = st->dev[slot];
        NIF_CUDA_TRY(cudaMemcpyAsync(d + st->o_origin, rays->origin + 3 * begin, (size_t)m * 12, cudaMemcpyHostToDevice, stream));
        NIF_CUDA_TRY(cudaMemcpyAsync(d + st->o_dir, rays->dir + 3 * begin, (size_t)m * 12, cudaMemcpyHostToDevice, stream));
        nif_ray_batch rb; rb.n = m; rb.origin = (const float*)(d + st->o_origin); rb.dir = (const float*)(d + st->o_dir);
        nif_query_out qo;
        memset(&qo, 0, sizeof(qo));
        qo.voxel_id = (int32_t*)(d + st->o_vid); qo.t_in = (float*)(d + st->o_tin); qo.t_out = (float*)(d + st->o_tout);
        qo.occlusion = (float*)(d + st->o_occ); qo.distance = (float*)(d + st->o_dist);
        qo.dist_total = (float*)(d + st->o_dtot); qo.normal = (float*)(d + st->o_nrm);
        qo.albedo = (float*)(d + st->o_alb); qo.material_logits = (float*)(d + st->o_mat);
        int rc = nif_query(bvh, net, &rb, &qo, d + st->o_ws, st->ws_bytes, flags, stream);
        if (rc != NIF_OK) return rc;
        NifQueryWs ws;
        nif_query_ws_layout(bvh, m, d + st->o_ws, &ws);
        CompactDst c{(int32_t*)(d + st->c_ray), (float*)(d + st->c_occ), (float*)(d + st->c_dist), (float*)(d + st->c_dtot),
                     (float*)(d + st->c_nrm), (float*)(d + st->c_alb), (float*)(d + st->c_mat)};
        const long long blocks_want = (m + 255) / 256;
        k_compact_heads<<<(unsigned)(blocks_want < 4LL * n_sm ? blocks_want : 4LL * n_sm), 256, 0, stream>>>(ws.scratch, ws.hit_list, qo, c, (int32_t)begin, flags);
        nif_count_launch(1);
        NIF_CUDA_TRY(cudaGetLastError());
        NIF_CUDA_TRY(cudaMemcpyAsync(&st->h_count[slot], &ws.scratch->n_hit, sizeof(unsigned long long), cudaMemcpyDeviceToHost, stream));
        NIF_CUDA_TRY(cudaEventRecord(st->ev[slot], stream));
        const size_t b = (size_t)begin, mm = (size_t)m;
        NIF_CUDA_TRY(cudaMemcpyAsync(out->voxel_id + b, d + st->o_vid, mm * 4, cudaMemcpyDeviceToHost, stream));
        NIF_CUDA_TRY(cudaMemcpyAsync(out->t_in + b, d + st->o_tin, mm * 4, cudaMemcpyDeviceToHost, stream));
        NIF_CUDA_TRY(cudaMemcpyAsync(out->t_out + b, d + st->o_tout, mm * 4, cudaMemcpyDeviceToHost, stream));
        if (pending_slot >= 0) { rc = finish(pending_slot); if (rc != NIF_OK) return rc; }
        pending_slot = slot;
    }
    if (pending_slot >= 0) { int rc = finish(pending_slot); if (rc != NIF_OK) return rc; }
    *n_hit_total = total;
    return NIF_OK;
}

extern "C" int nif_query_host_compact(const nif_bvh* bvh, const nif_net* net, nif_stage* st, const nif_ray_batch* rays,
                                      const nif_query_out* out, int32_t* hit_ray, int64_t* n_hit, unsigned flags)
{
    if (!st || !hit_ray || !n_hit) return NIF_ERR_INVALID_ARG;
    if (flags & NIF_TRAVERSE_ONLY) return NIF_ERR_INVALID_ARG;
    int rc = validate_query(bvh, net, rays, out, flags);
    if (rc != NIF_OK) return rc;
    if (out->raw_logits || out->hit_position || out->hit_position_rest) return NIF_ERR_INVALID_ARG;
    *n_hit = 0;
    rc = query_host_compact_enqueue(bvh, net, st, rays, out, hit_ray, n_hit, flags);
    for (int i = 0; i < NSLOT; ++i)
        if (cudaStreamSynchronize(st->stream[i]) != cudaSuccess) { (void)cudaGetLastError(); if (rc == NIF_OK) rc = NIF_ERR_CUDA; }
    return rc;
}
