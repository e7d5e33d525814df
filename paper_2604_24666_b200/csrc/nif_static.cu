// nif_static.cu -- nif_query_static: the hot path (a1)-(a5) for callers that cannot allocate device memory
// (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  It is nif_query with
// ONE difference: the query scratch (header with the hit counter and tile counter, the hit-ray bins, the
// rank and hit-list arrays; layout in nif_common.cuh) does not come from the caller but from a file-scope
// device array of fixed size.  The kernels are the ones nif_query launches; this file adds no arithmetic.
//
// What a caller has to know (also in include/nif.h):
//   * the array serves batches of at most NIF_STATIC_MAX_RAYS rays; larger batches are rejected with
//     NIF_ERR_STATIC_LIMIT before anything is enqueued;
//   * every GPU that loads the library holds the array (NIF_STATIC_SCRATCH_BYTES, ~24 MiB) until the
//     process exits;
//   * every call on a device shares the one array and finds the previous call's contents in it: the
//     header and the bin counters -- the only parts that must start at zero -- are cleared on `stream`
//     at the start of every call; calls whose GPU work overlaps (different streams, no ordering) RACE;
//   * no cudaMalloc / cudaFree / allocating library routine is called: the work is a cudaMemsetAsync and
//     kernel launches.  The address of the array is looked up once per device (cudaGetSymbolAddress, with
//     that device current) on the first call made with that device current -- make that first call
//     outside a graph capture.
#include "nif_common.cuh"

#include <mutex>

namespace {

constexpr size_t static_scratch_bytes(size_t n)
{
    // same formula as nif_query_workspace_bytes (nif_api.cu); checked against it at run time below
    return ((sizeof(NifQueryScratch) + (size_t)NIF_MAX_BINS * 4 + n * 8 + 255) / 256) * 256 + 256;
}
static_assert(static_scratch_bytes(NIF_STATIC_MAX_RAYS) == NIF_STATIC_SCRATCH_BYTES,
              "include/nif.h states the size of the static scratch");

// In HOST code this name is a host-side stand-in for the device array, not a device address: it must never
// be handed to a kernel.  Host code below only ever passes it to cudaGetSymbolAddress.
static __device__ __align__(256) unsigned char g_static_scratch[NIF_STATIC_SCRATCH_BYTES];

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
void* g_scratch_ptr[MAX_DEVICES];          // device address of g_static_scratch, per device ordinal

// device address of the array on the CURRENT device (looked up once per device)
int static_scratch_address(void** out)
{
    int dev = -1;
    NIF_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) return NIF_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
        void* ptr = nullptr;
        NIF_CUDA_TRY(cudaGetSymbolAddress((void**)&ptr, g_static_scratch));
        if (!ptr || ((uintptr_t)ptr & 255u) != 0) return NIF_ERR_CUDA;
        g_scratch_ptr[dev] = ptr;
    }
    *out = g_scratch_ptr[dev];
    return NIF_OK;
}

}  // namespace

int nif_validate_query(const nif_bvh* bvh, const nif_net* net, const nif_ray_batch* rays,
                       const nif_query_out* out, unsigned flags);

extern "C" int nif_query_static(const nif_bvh* bvh, const nif_net* net, const nif_ray_batch* rays,
                                const nif_query_out* out, unsigned flags, void* stream_)
{
    int rc = nif_validate_query(bvh, net, rays, out, flags);
    if (rc != NIF_OK) return rc;
    if (rays->n > (int64_t)NIF_STATIC_MAX_RAYS) return NIF_ERR_STATIC_LIMIT;
    if (rays->n == 0) return NIF_OK;
    size_t need = 0;
    rc = nif_query_workspace_bytes(rays->n, &need);
    if (rc != NIF_OK) return rc;
    if (need > (size_t)NIF_STATIC_SCRATCH_BYTES) return NIF_ERR_STATIC_LIMIT;
    void* scratch_dev = nullptr;
    rc = static_scratch_address(&scratch_dev);
    if (rc != NIF_OK) return rc;

    cudaStream_t stream = (cudaStream_t)stream_;
    NifQueryWs ws;
    nif_query_ws_layout(bvh, rays->n, scratch_dev, &ws);
    const bool traverse_only = (flags & NIF_TRAVERSE_ONLY) != 0;
    // the array keeps the last call's contents: header (hit / tile counters, status) and bin counters restart at zero
    NIF_CUDA_TRY(cudaMemsetAsync(scratch_dev, 0, sizeof(NifQueryScratch) + (traverse_only ? 0 : (size_t)ws.n_bins * 4), stream));
    rc = nif_launch_traverse(bvh, rays, out, &ws, flags, nullptr, stream);
    if (rc == NIF_OK && !traverse_only) rc = nif_launch_bin_hits(bvh, rays, out, &ws, nullptr, stream);
    if (rc != NIF_OK || traverse_only) return rc;
    const bool use_tc = net->desc.dtype == NIF_F16 && net->tc_supported && !(flags & NIF_ENGINE_FFMA);
    if (use_tc) return nif_launch_fused_tc(bvh, net, rays, out, ws.scratch, ws.hit_list, flags, stream);
    return nif_launch_ffma(bvh, net, rays, out, ws.scratch, ws.hit_list, flags, stream);
}
