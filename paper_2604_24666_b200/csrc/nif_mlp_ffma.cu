// nif_mlp_ffma.cu -- steps (a2)-(a5) on the plain FP32 pipes: inverse deformation, composite
// encoding, MLP, head decode for the hit rays the traversal compacted.
//
// This engine serves (i) NIF_F32 networks (config 0: fp32 parameters and a 1e-5 tolerance rule
// out TF32/FP16 tensor cores, B:7) and (ii) an on-device cross-check of the tcgen05 kernel
// (flag NIF_ENGINE_FFMA).  One block handles a tile of 8 hit rays: activations stay in shared
// memory, weights stream through L1/L2, nothing intermediate touches HBM.
#include "nif_encode.cuh"

namespace {

constexpr int FF_THREADS = 128;
constexpr int FF_TILE = 8;          // rays per block iteration

struct FfmaParams {
    NifEnc enc;
    int d_in, hidden_layers, width, n_out;
    const void* table;
    const void* w[NIF_MAX_LAYERS];
    NifMapCtx map;
    NifPoseBatch batch;
    const float* origin; const float* dir;
    nif_query_out out;
    const NifQueryScratch* scratch;
    const int32_t* hit_list;
    unsigned flags;
};

template <typename T> __device__ __forceinline__ float to_f32(T v);
template <> __device__ __forceinline__ float to_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ float to_f32<__half>(__half v) { return __half2float(v); }

// out[r][n] = act( sum_k W[n][k] in[r][k] ), r < FF_TILE.  The K range is split over
// G = FF_THREADS / n_pad thread groups; partial sums are combined in a fixed order.
template <typename T>
__device__ void dense_layer(const float* __restrict__ in, int in_stride, int K, const T* __restrict__ W,
                            int n_out, int n_pad, float* __restrict__ part, float* __restrict__ outp,
                            int out_stride, bool relu)
{
    const int G = FF_THREADS / n_pad;
    const int g = threadIdx.x / n_pad, n = threadIdx.x % n_pad;
    if (g < G) {
        float acc[FF_TILE];
#pragma unroll
        for (int r = 0; r < FF_TILE; ++r) acc[r] = 0.0f;
        if (n < n_out) {
            const int kc = (K + G - 1) / G;
            const int k0 = g * kc, k1 = min(K, k0 + kc);
            const T* wrow = W + (size_t)n * K;
            for (int k = k0; k < k1; ++k) {
                const float w = to_f32<T>(wrow[k]);
#pragma unroll
                for (int r = 0; r < FF_TILE; ++r) acc[r] = fmaf(w, in[r * in_stride + k], acc[r]);
            }
        }
#pragma unroll
        for (int r = 0; r < FF_TILE; ++r) part[(g * FF_TILE + r) * n_pad + n] = acc[r];
    }
    __syncthreads();
    for (int i = threadIdx.x; i < FF_TILE * n_pad; i += FF_THREADS) {
        const int r = i / n_pad, nn = i % n_pad;
        float s = 0.0f;
        for (int gg = 0; gg < G; ++gg) s += part[(gg * FF_TILE + r) * n_pad + nn];
        if (relu) s = fmaxf(s, 0.0f);
        outp[r * out_stride + nn] = s;
    }
    __syncthreads();
}

template <typename T, int F>
__global__ void __launch_bounds__(FF_THREADS)
k_encode_mlp_ffma(const FfmaParams p)
{
    extern __shared__ float smem[];
    const bool concat = p.enc.mode == NIF_ENC_CONCAT;
    const int S = concat ? 1 : 1 + 2 * p.enc.bands, L = p.enc.levels;     // samples that go through the grid
    const int n_pe = concat ? 3 + 6 * p.enc.bands : 0;                    // gamma scalars handed to the MLP directly
    const int d_in = p.d_in, W = p.width;
    float* act0 = smem;                                  // [FF_TILE][d_in]
    float* actA = act0 + FF_TILE * d_in;                 // [FF_TILE][W]
    float* actB = actA + FF_TILE * W;                    // [FF_TILE][W]
    float* part = actB + FF_TILE * W;                    // [G][FF_TILE][n_pad] <= FF_THREADS*FF_TILE
    float* xn = part + FF_THREADS * FF_TILE;             // [FF_TILE][2][3]
    float* samp = xn + FF_TILE * 6;                      // [FF_TILE][2][S][3]
    float* tseg = samp + FF_TILE * 2 * S * 3;            // [FF_TILE][2]  t_in, t_out
    __shared__ long long ray_of[FF_TILE];

    const long long n_hit = (long long)p.scratch->n_hit;
    const long long n_tiles = (n_hit + FF_TILE - 1) / FF_TILE;
    const T* table = reinterpret_cast<const T*>(p.table);
    const size_t level_stride = ((size_t)1 << p.enc.log2_T) * F;
    const uint32_t t_mask = (1u << p.enc.log2_T) - 1u;

    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        // (a2) entry/exit points -> rest space -> [0,1]^3
        if (threadIdx.x < FF_TILE * 2) {
            const int r = threadIdx.x >> 1, e = threadIdx.x & 1;
            const long long h = tile * FF_TILE + r;
            long long ray = -1;
            float x = 0.f, y = 0.f, z = 0.f, ti = 0.f, to = 0.f;
            if (h < n_hit) {
                ray = p.hit_list[h];
                ti = p.out.t_in[ray]; to = p.out.t_out[ray];
                const float oo[3] = {p.origin[3 * ray], p.origin[3 * ray + 1], p.origin[3 * ray + 2]};
                const float dd[3] = {p.dir[3 * ray], p.dir[3 * ray + 1], p.dir[3 * ray + 2]};
                float ri[3], ro[3];
                const NifMapCtx m = nif_ray_map(p.map, p.batch, ray);
                if (p.map.local) nif_map_back_pair<true>(m, p.out.voxel_id[ray], oo, dd, ti, to, ri, ro);
                else nif_map_back_pair<false>(m, 0, oo, dd, ti, to, ri, ro);
                x = e ? ro[0] : ri[0]; y = e ? ro[1] : ri[1]; z = e ? ro[2] : ri[2];
            }
            xn[(r * 2 + e) * 3 + 0] = nif_normalise(x);
            xn[(r * 2 + e) * 3 + 1] = nif_normalise(y);
            xn[(r * 2 + e) * 3 + 2] = nif_normalise(z);
            if (e == 0) { ray_of[r] = ray; tseg[2 * r] = ti; tseg[2 * r + 1] = to; }
        }
        __syncthreads();
        // gamma: S three-vector samples per endpoint
        for (int i = threadIdx.x; i < FF_TILE * 2 * S * 3; i += FF_THREADS) {
            const int a = i % 3, s = (i / 3) % S, re = i / (3 * S);
            samp[i] = nif_pe_sample(xn[re * 3 + a], s);
        }
        __syncthreads();
        // NIF_ENC_CONCAT: input[e*per + j] = gamma scalar j, per = n_pe + L*F
        for (int i = threadIdx.x; i < FF_TILE * 2 * n_pe; i += FF_THREADS) {
            const int j = i % n_pe, re = i / n_pe;
            act0[(re >> 1) * d_in + (re & 1) * (n_pe + L * F) + j] = nif_pe_scalar(xn + re * 3, j, p.enc.bands);
        }
        // (a3) phi of every sample, flattened input[((e*S + s)*L + l)*F + f]  (concat: after the gamma scalars)
        for (int i = threadIdx.x; i < FF_TILE * 2 * S * L; i += FF_THREADS) {
            const int l = i % L, s = (i / L) % S, re = i / (L * S);
            const int r = re >> 1, e = re & 1;
            float feat[F];
            const float* sp = samp + (re * S + s) * 3;
            nif_level_features<T, F>(table + (size_t)l * level_stride, p.enc.res[l],
                                     (p.enc.dense_mask >> l) & 1u, t_mask, sp[0], sp[1], sp[2], feat);
#pragma unroll
            for (int f = 0; f < F; ++f) act0[r * d_in + n_pe * (e + 1) + ((e * S + s) * L + l) * F + f] = feat[f];
        }
        __syncthreads();
        // (a4) MLP
        const float* cur = act0; int cur_stride = d_in, K = d_in;
        float* nxt = actA;
        for (int layer = 0; layer < p.hidden_layers; ++layer) {
            dense_layer<T>(cur, cur_stride, K, reinterpret_cast<const T*>(p.w[layer]), W, W, part, nxt, W, true);
            cur = nxt; cur_stride = W; K = W;
            nxt = (nxt == actA) ? actB : actA;
        }
        dense_layer<T>(cur, cur_stride, K, reinterpret_cast<const T*>(p.w[p.hidden_layers]), p.n_out, 16,
                       part, nxt, 16, false);
        // (a5) heads
        if (threadIdx.x < FF_TILE && ray_of[threadIdx.x] >= 0) {
            const int r = threadIdx.x;
            float z[NIF_N_OUT];
#pragma unroll
            for (int a = 0; a < NIF_N_OUT; ++a) z[a] = a < p.n_out ? nxt[r * 16 + a] : 0.0f;
            if (p.map.local) nif_decode_store<true>(z, tseg[2 * r], tseg[2 * r + 1], ray_of[r], p.out, p.flags, NifDecodeCtx{p.origin, p.dir, p.map, p.batch});
            else nif_decode_store<false>(z, tseg[2 * r], tseg[2 * r + 1], ray_of[r], p.out, p.flags, NifDecodeCtx{p.origin, p.dir, p.map, p.batch});
        }
        __syncthreads();
    }
}

template <typename T>
int launch_t(const FfmaParams& p, int feat, size_t smem, int blocks, cudaStream_t stream)
{
#define NIF_FF_LAUNCH(FEAT)                                                                            \
    do {                                                                                               \
        NIF_CUDA_TRY(cudaFuncSetAttribute(k_encode_mlp_ffma<T, FEAT>,                                  \
                                          cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));    \
        k_encode_mlp_ffma<T, FEAT><<<blocks, FF_THREADS, smem, stream>>>(p);                           \
    } while (0)
    switch (feat) {
        case 1: NIF_FF_LAUNCH(1); break;
        case 2: NIF_FF_LAUNCH(2); break;
        case 4: NIF_FF_LAUNCH(4); break;
        default: return NIF_ERR_UNSUPPORTED;
    }
#undef NIF_FF_LAUNCH
    nif_count_launch(1);
    NIF_CUDA_TRY(cudaGetLastError());
    return NIF_OK;
}

}  // namespace

int nif_launch_ffma(const nif_bvh* bvh, const nif_net* net, const nif_ray_batch* rays,
                    const nif_query_out* out, const NifQueryScratch* scratch,
                    const int32_t* hit_list, unsigned flags, cudaStream_t stream, const NifPoseBatch* batch)
{
    if (rays->n == 0) return NIF_OK;
    FfmaParams p;
    p.batch = batch ? *batch : NifPoseBatch{nullptr, nullptr, 0};
    p.enc = net->enc;
    p.d_in = net->d_in; p.hidden_layers = net->desc.hidden_layers; p.width = net->desc.width;
    p.n_out = (flags & NIF_OCCLUSION_ONLY) ? 1 : NIF_N_OUT;
    p.table = net->table;
    for (int i = 0; i <= net->desc.hidden_layers; ++i) p.w[i] = net->w_plain[i];
    p.map = NifMapCtx{bvh->theta_max, bvh->bend_k, bvh->lattice, bvh->nv, bvh->local_inverse};
    p.origin = rays->origin; p.dir = rays->dir;
    p.out = *out; p.scratch = scratch; p.hit_list = hit_list; p.flags = flags;
    const int S = 1 + 2 * net->enc.bands;
    const size_t smem = sizeof(float) * ((size_t)FF_TILE * net->d_in + 2 * (size_t)FF_TILE * net->desc.width +
                                         (size_t)FF_THREADS * FF_TILE + FF_TILE * 6 + (size_t)FF_TILE * 2 * S * 3 +
                                         FF_TILE * 2);
    if (smem > 200 * 1024) return NIF_ERR_UNSUPPORTED;
    long long tiles = (rays->n + FF_TILE - 1) / FF_TILE;
    int blocks = (int)(tiles < 148 * 8 ? tiles : 148 * 8);
    if (net->desc.dtype == NIF_F32) return launch_t<float>(p, net->enc.feat, smem, blocks, stream);
    return launch_t<__half>(p, net->enc.feat, smem, blocks, stream);
}
