// nif_walk.cu -- nif_query_multi: the evaluation-time multi-voxel walk.
// PAPER.md:51 "explicitly determining the voxel face through which a ray exits, which allows correct
// selection of neighboring voxels"; P:53 the BVH gives the starting voxel and skips empty gaps;
// P:59-61 the distance is the sum of gaps and segments up to the first voxel k that contains a hit,
// plus the local distance t_k in it; "During evaluation, we reconstruct hit positions along
// the same segmented ray".  Readings R22/R23 of DESIGN.md section 3.
//
// Rounds: round 0 is the plain query over all rays; after each round k_walk_update looks at the
// occlusion the network predicted for every ray that hit a voxel, accepts (>= 0.5) or appends the
// ray to the list of rays that walk on; round j+1 traverses only those, looking for the successor
// of the voxel they evaluated last in (t_in, id) order, and evaluates the network on it.  Nothing
// synchronises: all `max_steps` rounds are enqueued and a round whose list is empty costs a few
// empty launches.  Per-ray walk state lives in the outputs themselves (t_in / voxel_id = the
// successor bound, dist_accum = the running sum, steps) plus one float per ray (previous exit).
#include "nif_common.cuh"

namespace {

struct WalkUpdateParams {
    nif_query_out out;
    nif_walk_out walk;
    const NifQueryScratch* scratch;      // n_hit of this round
    const int32_t* hit_list;
    float* prev_exit;                    // t_out of the voxel evaluated last; 0 = the ray origin (R13)
    int32_t* next_list;
    unsigned int* next_count;
    int max_steps;
    unsigned flags;
};

__global__ void __launch_bounds__(256)
k_walk_update(const WalkUpdateParams p)
{
    const long long n_hit = (long long)p.scratch->n_hit;
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n_hit; i += (long long)gridDim.x * 256) {
        const int32_t r = p.hit_list[i];
        const float ti = p.out.t_in[r], to = p.out.t_out[r];
        const int32_t k = p.walk.steps[r] + 1;
        p.walk.steps[r] = k;
        const float delta = __fsub_rn(ti, p.prev_exit[r]);           // signed gap (R23)
        const float ell = __fsub_rn(to, ti);
        const float acc = p.walk.dist_accum[r];
        if (p.out.occlusion[r] >= 0.5f) {                            // first voxel containing a hit
            const float tk = (p.flags & NIF_OCCLUSION_ONLY) ? 0.0f : p.out.distance[r];
            p.walk.dist_accum[r] = __fadd_rn(__fadd_rn(acc, delta), tk);
            p.walk.status[r] = NIF_WALK_HIT;
        } else {
            p.walk.dist_accum[r] = __fadd_rn(acc, __fadd_rn(delta, ell));
            p.prev_exit[r] = to;
            if (k >= p.max_steps) {
                p.walk.status[r] = NIF_WALK_MAX_STEPS;
            } else {
                p.next_list[atomicAdd(p.next_count, 1u)] = r;
            }
        }
    }
}

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
constexpr int WALK_MAX_STEPS = 4096;
inline size_t walk_header_bytes() { return align_up((size_t)(WALK_MAX_STEPS + 1) * 4, 256); }

}  // namespace

int nif_validate_query(const nif_bvh* bvh, const nif_net* net, const nif_ray_batch* rays,
                       const nif_query_out* out, unsigned flags);

extern "C" int nif_query_multi_workspace_bytes(int64_t n, size_t* bytes)
{
    size_t q = 0;
    int rc = nif_query_workspace_bytes(n, &q);
    if (rc != NIF_OK) return rc;
    *bytes = align_up(q, 256) + walk_header_bytes() + align_up((size_t)n * 4, 256) * 2;
    return NIF_OK;
}

extern "C" int nif_query_multi(const nif_bvh* bvh, const nif_net* net, const nif_ray_batch* rays,
                               const nif_query_out* out, const nif_walk_out* walk, int32_t max_steps,
                               void* workspace, size_t workspace_bytes, unsigned flags, void* stream_)
{
    if (flags & (NIF_TRAVERSE_ONLY | NIF_PROBE_SKIP_GATHER)) return NIF_ERR_INVALID_ARG;
    int rc = nif_validate_query(bvh, net, rays, out, flags);
    if (rc != NIF_OK) return rc;
    if (!walk || max_steps < 1 || max_steps > WALK_MAX_STEPS) return NIF_ERR_INVALID_ARG;
    if (rays->n == 0) return NIF_OK;
    if (!walk->status || !walk->steps || !walk->dist_accum) return NIF_ERR_INVALID_ARG;
    size_t need = 0, qbytes = 0;
    nif_query_multi_workspace_bytes(rays->n, &need);
    nif_query_workspace_bytes(rays->n, &qbytes);
    if (!workspace || ((uintptr_t)workspace & 255u) != 0 || workspace_bytes < need) return NIF_ERR_WORKSPACE;
    cudaStream_t stream = (cudaStream_t)stream_;
    const size_t n = (size_t)rays->n;

    NifQueryWs ws;
    nif_query_ws_layout(bvh, rays->n, workspace, &ws);
    char* extra = (char*)workspace + align_up(qbytes, 256);
    unsigned int* live_count = (unsigned int*)extra;                 // [round] rays entering round `round`
    int32_t* live_list = (int32_t*)(extra + walk_header_bytes());
    float* prev_exit = (float*)((char*)live_list + align_up(n * 4, 256));

    NIF_CUDA_TRY(cudaMemsetAsync(extra, 0, walk_header_bytes(), stream));
    NIF_CUDA_TRY(cudaMemsetAsync(prev_exit, 0, n * 4, stream));
    NIF_CUDA_TRY(cudaMemsetAsync(walk->status, 0, n * 4, stream));   // NIF_WALK_MISS until a round says otherwise
    NIF_CUDA_TRY(cudaMemsetAsync(walk->steps, 0, n * 4, stream));
    NIF_CUDA_TRY(cudaMemsetAsync(walk->dist_accum, 0, n * 4, stream));

    const int n_sm = nif_sm_count();
    if (n_sm <= 0) return NIF_ERR_CUDA;
    const bool use_tc = net->desc.dtype == NIF_F16 && net->tc_supported && !(flags & NIF_ENGINE_FFMA);
    for (int round = 0; round < max_steps; ++round) {
        NifWalkRound wr;
        wr.round = round; wr.ray_list = live_list; wr.n_list = &live_count[round]; wr.dist_accum = walk->dist_accum;
        // round 0 clears header + bins with one memset; later rounds clear the header and let a kernel clear the
        // bins only if some ray still walks, so that the rounds after the last live ray cost a few empty launches
        if (round == 0) NIF_CUDA_TRY(cudaMemsetAsync(workspace, 0, sizeof(NifQueryScratch) + (size_t)ws.n_bins * 4, stream));
        else {
            NIF_CUDA_TRY(cudaMemsetAsync(workspace, 0, sizeof(NifQueryScratch), stream));
            rc = nif_launch_clear_bins(&ws, &live_count[round], stream);
            if (rc != NIF_OK) return rc;
        }
        const int prof = nif_prof_begin(stream);
        rc = nif_launch_traverse(bvh, rays, out, &ws, flags, &wr, stream);
        if (rc == NIF_OK) rc = nif_launch_bin_hits(bvh, rays, out, &ws, &wr, stream);
        nif_prof_mark(prof, 1, stream);
        if (rc != NIF_OK) return rc;
        if (use_tc) rc = nif_launch_fused_tc(bvh, net, rays, out, ws.scratch, ws.hit_list, flags, stream);
        else rc = nif_launch_ffma(bvh, net, rays, out, ws.scratch, ws.hit_list, flags, stream);
        if (rc != NIF_OK) return rc;
        WalkUpdateParams up;
        up.out = *out; up.walk = *walk; up.scratch = ws.scratch; up.hit_list = ws.hit_list;
        up.prev_exit = prev_exit; up.next_list = live_list; up.next_count = &live_count[round + 1];
        up.max_steps = max_steps; up.flags = flags;
        const long long want = ((long long)n + 255) / 256;
        const long long cap = (long long)n_sm * 8;
        k_walk_update<<<(unsigned)(want < cap ? want : cap), 256, 0, stream>>>(up);
        nif_count_launch(1);
        NIF_CUDA_TRY(cudaGetLastError());
        nif_prof_mark(prof, 2, stream);
    }
    return NIF_OK;
}
