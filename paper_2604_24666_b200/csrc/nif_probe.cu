// nif_probe.cu -- measurement helpers of libnif.so (include/nif.h "diagnostics"):
//   * per-kernel timing of nif_query with CUDA events on the caller's stream, so bench.py can
//     report the dominant kernel's average launch duration from inside the timed region;
//   * the random-sector gather probe that gives the denominator of the gather roofline
//     (MEASURED_PEAKS.json has no L2 figure).
// None of this is on the query path unless profiling is switched on.
#include "nif_common.cuh"

#include <mutex>

namespace {

constexpr int PROF_RING = 512;             // queries remembered between two reads

struct ProfState {
    std::mutex mu;
    bool enabled = false;
    bool events_ready = false;
    cudaEvent_t ev[PROF_RING][3];          // before traverse, after traverse, after encode+MLP
    int kind[PROF_RING];                   // 1 = traverse only, 2 = traverse + network
    int count = 0;
};
ProfState g_prof;

bool ensure_events()
{
    if (g_prof.events_ready) return true;
    for (int i = 0; i < PROF_RING; ++i)
        for (int j = 0; j < 3; ++j)
            if (cudaEventCreate(&g_prof.ev[i][j]) != cudaSuccess) { (void)cudaGetLastError(); return false; }
    g_prof.events_ready = true;
    return true;
}

}  // namespace

// ---- hooks used by nif_query (nif_api.cu) ---------------------------------------------------
int nif_prof_begin(cudaStream_t stream)
{
    std::lock_guard<std::mutex> lk(g_prof.mu);
    if (!g_prof.enabled || g_prof.count >= PROF_RING) return -1;
    const int slot = g_prof.count++;
    g_prof.kind[slot] = 0;
    if (cudaEventRecord(g_prof.ev[slot][0], stream) != cudaSuccess) { (void)cudaGetLastError(); }
    return slot;
}

void nif_prof_mark(int slot, int which, cudaStream_t stream)
{
    if (slot < 0) return;
    std::lock_guard<std::mutex> lk(g_prof.mu);
    if (cudaEventRecord(g_prof.ev[slot][which], stream) != cudaSuccess) { (void)cudaGetLastError(); }
    g_prof.kind[slot] = which;
}

extern "C" int nif_profile_enable(int on)
{
    std::lock_guard<std::mutex> lk(g_prof.mu);
    if (on && !ensure_events()) return NIF_ERR_CUDA;
    g_prof.enabled = on != 0;
    g_prof.count = 0;
    return NIF_OK;
}

extern "C" int nif_profile_read(double* traverse_ms, double* network_ms, int64_t* n_queries)
{
    if (!traverse_ms || !network_ms || !n_queries) return NIF_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lk(g_prof.mu);
    double t = 0.0, m = 0.0;
    int64_t n = 0;
    for (int i = 0; i < g_prof.count; ++i) {
        if (g_prof.kind[i] < 1) continue;
        float a = 0.f, b = 0.f;
        NIF_CUDA_TRY(cudaEventSynchronize(g_prof.ev[i][g_prof.kind[i]]));
        NIF_CUDA_TRY(cudaEventElapsedTime(&a, g_prof.ev[i][0], g_prof.ev[i][1]));
        if (g_prof.kind[i] == 2) NIF_CUDA_TRY(cudaEventElapsedTime(&b, g_prof.ev[i][1], g_prof.ev[i][2]));
        t += a; m += b; ++n;
    }
    *traverse_ms = t; *network_ms = m; *n_queries = n;
    g_prof.count = 0;
    return NIF_OK;
}

// ---- gather probes: the denominators of the gather roofline ------------------------------------
namespace {

// Counter-based hash, no state.
__device__ __forceinline__ uint32_t mix32(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

// MODE 0 "divergent": every lane loads 4 bytes from its own pseudo-random 32-byte sector (its own 128-byte
//   line), 8 independent loads per batch: the access pattern of a hashed level, where no two lanes share a
//   sector.  A warp load is then 32 L1 wavefronts: this measures the L1/LSU divergent-access ceiling
//   (wavefronts per second), with the lines coming from L2 (or HBM for a large buffer).
// MODE 1 "coalesced sectors": the 32 lanes of a warp read one pseudo-random 128-byte line (4 bytes each: 4
//   sectors, 8 lanes per sector), 16 independent lines per batch: one L1 wavefront moves 4 sectors, so the
//   LSU is far from its limit and the rate is what L2 (or HBM) delivers to the SMs in 32-byte sectors.
template <int MODE>
__global__ void __launch_bounds__(512)
k_probe_gather(const uint32_t* __restrict__ buf, uint32_t mask, int iters, uint32_t* __restrict__ sink)
{
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t acc = 0;
    const uint32_t ctr = (MODE == 0 ? tid : (tid >> 5)) * 0x9e3779b9u;
    constexpr int NB = MODE == 0 ? 8 : 16;          // independent loads in flight per thread
    for (int it = 0; it < iters * 8 / NB; ++it) {
        uint32_t v[NB];
#pragma unroll
        for (int j = 0; j < NB; ++j) {
            const uint32_t s = mix32(ctr + (uint32_t)(it * NB + j)) & mask;
            if (MODE == 0) v[j] = __ldg(buf + (size_t)s * 8u + (tid & 7u));                 // s = sector index
            else v[j] = __ldg(buf + (size_t)s * 32u + (tid & 31u));                          // s = line index
        }
#pragma unroll
        for (int j = 0; j < NB; ++j) acc ^= v[j];
    }
    if (acc == 0x12345678u) sink[0] = acc;      // defeats dead-code elimination, never true in practice
}

}  // namespace

extern "C" int nif_probe_gather(const void* buf, size_t bytes, int iters, size_t smem_bytes, int mode, void* stream_,
                                double* sectors_per_s, double* ms)
{
    if (smem_bytes > 227u * 1024u || (mode != 0 && mode != 1)) return NIF_ERR_INVALID_ARG;
    if (!buf || !sectors_per_s || iters < 1 || bytes < 4096) return NIF_ERR_INVALID_ARG;
    if (!nif_device_supported()) return NIF_ERR_UNSUPPORTED;
    cudaStream_t stream = (cudaStream_t)stream_;
    size_t n_sectors = 1;
    while (n_sectors * 2 * 32 <= bytes) n_sectors *= 2;          // power of two that fits
    uint32_t* sink = nullptr;
    NIF_CUDA_TRY(cudaMalloc((void**)&sink, 256));
    cudaEvent_t e0, e1;
    NIF_CUDA_TRY(cudaEventCreate(&e0));
    NIF_CUDA_TRY(cudaEventCreate(&e1));
    const int sms = nif_sm_count();
    if (sms <= 0) return NIF_ERR_CUDA;
    // dynamic shared memory the probe does not touch: it only shrinks the L1 data cache to what a
    // kernel with that much shared memory is left with (one block per SM above ~113 KB)
    if (mode == 0) NIF_CUDA_TRY(cudaFuncSetAttribute(k_probe_gather<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes));
    else NIF_CUDA_TRY(cudaFuncSetAttribute(k_probe_gather<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes));
    const int per_sm = smem_bytes > 113u * 1024u ? 1 : (smem_bytes > 56u * 1024u ? 2 : 4);
    const int blocks = sms * per_sm, threads = 512;
    const uint32_t mask = (uint32_t)((mode == 0 ? n_sectors : n_sectors / 4) - 1);
    double best = 1e30;
    for (int rep = 0; rep < 4; ++rep) {                            // rep 0 warms L2 with the buffer
        NIF_CUDA_TRY(cudaEventRecord(e0, stream));
        if (mode == 0) k_probe_gather<0><<<blocks, threads, smem_bytes, stream>>>((const uint32_t*)buf, mask, iters, sink);
        else k_probe_gather<1><<<blocks, threads, smem_bytes, stream>>>((const uint32_t*)buf, mask, iters, sink);
        NIF_CUDA_TRY(cudaEventRecord(e1, stream));
        NIF_CUDA_TRY(cudaEventSynchronize(e1));
        nif_count_launch(1);
        float t = 0.f;
        NIF_CUDA_TRY(cudaEventElapsedTime(&t, e0, e1));
        if (rep > 0 && t < best) best = t;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    NIF_CUDA_TRY(cudaGetLastError());
    const double lane_loads = (double)blocks * threads * (double)iters * 8.0;
    *sectors_per_s = (mode == 0 ? lane_loads : lane_loads / 8.0) / (best * 1e-3);     // 8 lanes share a sector in mode 1
    if (ms) *ms = best;
    return NIF_OK;
}
