// nif_fused_tc.cu -- steps (a2)-(a5) for NIF_F16 networks as ONE persistent sm_100a kernel:
// inverse deformation -> composite encoding psi = phi o gamma (Eq. 1) -> MLP on
// tcgen05 tensor cores -> head decode, per tile of 128 hit rays, with no
// intermediate HBM round trip.
//
// Data flow of one tile (UMMA M = 128 rays, thread/TMEM lane r = ray r of the tile):
//   * every A operand lives in TENSOR MEMORY: the gather warps write the layer-1 features with
//     tcgen05.st (fp16 pairs, 32 columns per 64-feature K chunk, a ring of chunk slots), the tail
//     warps write the hidden activations the same way, and the MMAs are issued in the A-from-TMEM
//     form.  Shared memory holds only B operands (weights) and ray info, which keeps the L1 data
//     cache large for the table gathers and needs no proxy fences;
//   * layer-1 weights stay resident in shared memory when they fit the budget (config 1-3: 104 KB),
//     otherwise their K chunks stream through a ring (config 4: 416 KB); hidden/output weights are
//     resident for W <= 64 and stream through a 2-slot ring for W = 128;
//   * accumulators: a tile owns one TMEM accumulator buffer from its first layer-1 MMA to the read of its
//     output (the hidden/output layers accumulate into the drained layer-1 buffer); three buffers for
//     W <= 64 (layer 1 of tile t+1 runs while the two tail groups work on tiles t and t-1), two for
//     W = 128; the rest of the 512 TMEM columns is the A ring (8 / 6 chunk slots).
//
// Warp roles (one CTA per SM, 32 warps; setmaxnreg moves registers from the other roles to the
// gather warps, whose loop needs 80):
//   warps 0-3 / 4-7  tail groups 0 / 1, alternating tiles: drain the layer-1 accumulator (tcgen05.ld),
//                    ReLU -> fp16 -> tcgen05.st as the next A operand, one thread issues the hidden /
//                    output layer MMAs, finally decode and store the heads (a5).  Two groups keep two
//                    tiles' dependent layer chains in flight.
//   warp 8           issues the layer-1 MMAs chunk by chunk as ring slots fill (converged, elect.sync).
//   warp 9           lane 0 loads the resident weights once and streams layer-1 chunks when they are
//                    not resident; lane 1 streams hidden/output chunks (W = 128).
//   warps 10-11      "prep": draw tile ids from the global counter, fetch the tile's rays through
//                    hit_list and map entry/exit points back to rest space (a2) -> ray_buf (3 deep).
//   warps 12-31      gather warps: lane = ray of row group (warp % 4); one work item = (endpoint, PE
//                    sample): the L levels of that sample are interpolated (8 table gathers each, fp32,
//                    two batches of loads in flight) and written as fp16 into the chunk slot (a3).
// Template parameters: W, F; CONCAT = concatenation reading of the hybrid encoding (R1); LOCAL =
// voxel-local trilinear inverse for lattice-supplied deformations (R27); PROBE = the gathers are
// replaced by a constant A operand (the MLP-only probe of bench.py; its own instantiation, the product
// kernels carry no probe branch).
#include "nif_encode.cuh"

#include <type_traits>

namespace {

constexpr int TC_TILE = 128;                 // rays per tile = UMMA M
constexpr int TC_TAIL_WARPS = 8;             // two groups of 4
constexpr int TC_MMA_WARP = 8;
constexpr int TC_LOAD_WARP = 9;
constexpr int TC_PREP_WARP0 = 10;            // warps 10, 11
constexpr int TC_PREP_THREADS = 64;
constexpr int TC_GATHER_WARP0 = 12;
constexpr int TC_GATHER_WARPS = 20;          // 4 row groups x TC_GPR warps: as many as the register file allows at 80 each
constexpr int TC_GPR = TC_GATHER_WARPS / 4;
constexpr int TC_THREADS = 32 * (TC_GATHER_WARP0 + TC_GATHER_WARPS);      // 1024
constexpr int TC_RAY_BUFS = 3;               // ray_buf depth: prep runs up to two tiles ahead of the tails
constexpr int TC_RAY_FIELDS = 9;             // xi yi zi xo yo zo t_in t_out ray
constexpr int TC_MAX_A_SLOTS = 10;           // layer-1 A chunk slots in TMEM (32 columns each)
constexpr int TC_MAX_ACC = 3;                // layer-1 accumulator buffers (W <= 64: 3, W = 128: 2)
constexpr int TC_MAX_W1_SLOTS = 8;           // layer-1 weight chunk slots when W1 streams
constexpr int TC_HSLOTS = 2;                 // hidden/output weight chunk ring (W = 128)
constexpr int TC_NOUT_PAD = 16;              // output layer N (12 heads padded to the UMMA minimum)
// Launched with 64 registers per thread (1024 threads); setmaxnreg then moves registers from the roles that are off the
// critical path of the real (gather-bound) kernel to the gather warps, whose loop needs 80 and which are the kernel's
// memory-level parallelism: tails 40, small roles 24, gather 80 (8 x 40 + 4 x 24 + 20 x 80 = 2016 <= 32 x 64; a
// setmaxnreg.inc can only take what a dec released).  Measured: 16 gather warps (tails 72, small roles 40) 0.706 / 5.00 ms on
// config 1 / 4, 20 gather warps 0.673 / 4.87 ms; the tails and the prep warps spill ~150 B and do not care.
constexpr int TC_REGS_MISC = 24, TC_REGS_GATHER = 80, TC_REGS_TAIL = 40;

// ---- PTX wrappers -----------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    } while (!done);
}
// wait for the role warps whose waits are long: try_wait with a suspend-time hint parks the thread in
// hardware until the phase completes or the hint expires, so the wait takes (almost) no issue slots
// from the gather warps and still wakes up as soon as the barrier flips
__device__ __forceinline__ void mbar_wait_sleep(uint32_t bar, uint32_t parity, unsigned hint_ns = 20000)
{
    uint32_t done;
    do {
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}" : "=r"(done) : "r"(bar), "r"(parity), "r"(hint_ns) : "memory");
    } while (!done);
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

__device__ __forceinline__ void tmem_alloc(uint32_t dst_smem, uint32_t cols)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t cols)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }

// D[tmem] (+)= A[tmem] * B[smem]^T, fp16 operands, fp32 accumulate, M = 128.  A: lane = row, 16-bit
// elements packed two per 32-bit column (K = 16 -> 8 columns); B: K-major SWIZZLE_128B descriptor.
__device__ __forceinline__ void umma_f16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t"
        "}" ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
// One K chunk in ONE asm block, called by a CONVERGED warp: elect.sync picks the issuing lane, which issues NK
// UMMAs over consecutive K = 16 slices (A: +8 TMEM columns, B: +32 bytes = +2 in the descriptor's address
// field) and, if commit_bar != 0, the commit that releases the chunk.  Measured on B200: code
// that runs the MMA loop on one lane of a diverged warp makes ptxas wrap every tcgen05.mma in an elect-one loop
// and issues an M128 N64 K16 UMMA every 56 cycles (the tensor pipe needs 32); the warp-converged form below
// issues one every 32 cycles, i.e. the 64-wide layers run at the tensor pipe's rate.
template <int NK>
__device__ __forceinline__ void umma_chunk_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc,
                                              uint32_t accumulate_first, uint32_t commit_bar)
{
    static_assert(NK == 1 || NK == 2 || NK == 4, "K = 16, 32 or 64 per chunk");
    if constexpr (NK == 4) {
        // the K = 16 slices advance the descriptor's 14-bit address field by 2 (32 bytes): a 32-bit add on the low
        // word (a chunk never straddles the 256 KB field), the high word is shared
        asm volatile(
            "{\n\t"
            ".reg .pred p, pe, cq;\n\t"
            ".reg .b32 a1, a2, a3, lo, hi, l1, l2, l3;\n\t"
            ".reg .b64 b1, b2, b3;\n\t"
            "elect.sync _|pe, 0xffffffff;\n\t"
            "setp.ne.b32 p, %4, 0;\n\t"
            "setp.ne.and.b32 cq, %5, 0, pe;\n\t"
            "mov.b64 {lo, hi}, %2;\n\t"
            "add.u32 a1, %1, 8;\n\t"
            "add.u32 a2, %1, 16;\n\t"
            "add.u32 a3, %1, 24;\n\t"
            "add.u32 l1, lo, 2;\n\t"
            "add.u32 l2, lo, 4;\n\t"
            "add.u32 l3, lo, 6;\n\t"
            "mov.b64 b1, {l1, hi};\n\t"
            "mov.b64 b2, {l2, hi};\n\t"
            "mov.b64 b3, {l3, hi};\n\t"
            "@pe tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t"
            "@pe tcgen05.mma.cta_group::1.kind::f16 [%0], [a1], b1, %3, 1;\n\t"
            "@pe tcgen05.mma.cta_group::1.kind::f16 [%0], [a2], b2, %3, 1;\n\t"
            "@pe tcgen05.mma.cta_group::1.kind::f16 [%0], [a3], b3, %3, 1;\n\t"
            "@cq tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%5];\n\t"
            "}" ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate_first), "r"(commit_bar) : "memory");
    } else if constexpr (NK == 2) {
        asm volatile(
            "{\n\t"
            ".reg .pred p, pe, cq;\n\t"
            ".reg .b32 a1;\n\t"
            ".reg .b64 b1;\n\t"
            "elect.sync _|pe, 0xffffffff;\n\t"
            "setp.ne.b32 p, %4, 0;\n\t"
            "setp.ne.and.b32 cq, %5, 0, pe;\n\t"
            "add.u32 a1, %1, 8;\n\t"
            "add.u64 b1, %2, 2;\n\t"
            "@pe tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t"
            "@pe tcgen05.mma.cta_group::1.kind::f16 [%0], [a1], b1, %3, 1;\n\t"
            "@cq tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%5];\n\t"
            "}" ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate_first), "r"(commit_bar) : "memory");
    } else {
        asm volatile(
            "{\n\t"
            ".reg .pred p, pe, cq;\n\t"
            "elect.sync _|pe, 0xffffffff;\n\t"
            "setp.ne.b32 p, %4, 0;\n\t"
            "setp.ne.and.b32 cq, %5, 0, pe;\n\t"
            "@pe tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t"
            "@cq tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%5];\n\t"
            "}" ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate_first), "r"(commit_bar) : "memory");
    }
}
// the same for a lone commit (converged warp, one elected lane): all previously issued MMAs of the ELECTED lane
// arrive on `bar` when they complete.  elect.sync with a full mask always elects the same lane, so commits and
// MMAs come from one thread.
__device__ __forceinline__ void umma_commit_elect(uint32_t bar)
{
    asm volatile(
        "{\n\t"
        ".reg .pred pe;\n\t"
        "elect.sync _|pe, 0xffffffff;\n\t"
        "@pe tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n\t"
        "}" ::"r"(bar) : "memory");
}
// all previously issued MMAs of this thread arrive on `bar` when they complete (implies fence::before_thread_sync)
__device__ __forceinline__ void umma_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

// K-major SWIZZLE_128B shared-memory matrix descriptor: rows of 128 bytes, 8-row groups 1024 bytes
// apart (SBO), LBO unused (1), descriptor version 1 (sm_100), layout type 2 (cute::UMMA::SWIZZLE_128B)
__device__ __forceinline__ uint64_t smem_desc_sw128(uint32_t addr)
{
    return (uint64_t)((addr & 0x3ffffu) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) |
           ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
// instruction descriptor, kind::f16: D fp32 (bit 4), A/B fp16 (0), both K-major, N>>3 at bit 17, M>>4 at bit 24
__host__ __device__ constexpr uint32_t idesc_f16(int M, int N)
{
    return (1u << 4) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

// TMEM -> registers: this warp's 32 lanes x 32 consecutive fp32 columns (thread = lane = row)
__device__ __forceinline__ void tmem_ld_32x32(uint32_t taddr, uint32_t* v)
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld_32x16(uint32_t taddr, uint32_t* v)
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
// registers -> TMEM: this warp's 32 lanes x 4 / 16 consecutive 32-bit columns
__device__ __forceinline__ void tmem_st_32x4(uint32_t taddr, uint32_t a, uint32_t b, uint32_t c, uint32_t d)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ void tmem_st_32x16(uint32_t taddr, const uint32_t* v)
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
        ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
          "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ void named_bar_sync(int id, int threads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}

__device__ __forceinline__ uint32_t pack_half2(float a, float b)
{
    __half2 h = __floats2half2_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&h);
}

// byte offset of the 16-byte unit `unit` (0..7) of row `row` inside a [rows x 128 B] SWIZZLE_128B chunk
__host__ __device__ __forceinline__ uint32_t sw128_off(uint32_t row, uint32_t unit)
{
    return row * 128u + ((unit ^ (row & 7u)) << 4);
}

// ---- optional per-tile timestamps (compile with -DNIF_TC_TRACE; nif_debug_set_tc_trace hands in the buffer) ----
#ifdef NIF_TC_TRACE
__device__ unsigned int* g_tc_trace = nullptr;        // [cta][NIF_TC_TRACE_TILES][32] clock() samples
#define NIF_TC_TRACE_TILES 24
#define TC_TRACE(j, slot) do { if (g_tc_trace && (j) < NIF_TC_TRACE_TILES) \
        g_tc_trace[((size_t)blockIdx.x * NIF_TC_TRACE_TILES + (size_t)(j)) * 32 + (slot)] = (unsigned int)clock(); } while (0)
#else
#define TC_TRACE(j, slot) do { } while (0)
#endif

// ---- kernel parameters -------------------------------------------------------------------------
struct TcParams {
    NifEnc enc;
    int hidden_layers;            // H
    int n_chunks;                 // layer-1 K chunks of 64 columns = ceil(2 S L F / 64)
    int es_per_chunk;             // (endpoint, sample) pairs per chunk = 64 / (L F)
    int n_es;                     // 2 S
    const __half* table;
    const uint8_t* w_img;         // B-operand images: W1 chunks | hidden layers 2..H | output layer
    uint32_t w_bytes, w1_bytes;
    int w1_slots;                 // layer-1 weight chunk slots in shared memory
    int w1_resident;              // 1: w1_slots == n_chunks, loaded once; 0: ring
    float theta_max, bend_k;
    const float* origin;
    const float* dir;
    nif_query_out out;
    const NifQueryScratch* scratch;
    unsigned int* tile_counter;   // dynamic tile scheduler (scratch header, zeroed per query)
    int enc_mode;                 // NIF_ENC_COMPOSE | NIF_ENC_CONCAT
    NifMapCtx map;                // (a2): pose, or the lattice for the voxel-local inverse
    NifPoseBatch batch;           // nif_query_poses: per-ray pose (pose_id == NULL otherwise)
    const int32_t* hit_list;
    unsigned flags;
};

// shared memory: [hidden/output weights][layer-1 weight slots][ray_buf][barriers, tile ids, level constants]
struct TcSmemLayout {
    uint32_t w_hid, w1, ray_buf, bars, total;
};
__host__ __device__ inline uint32_t tc_hid_bytes(int W, int hidden_layers)
{
    const uint32_t KC = (uint32_t)(W + 63) / 64;
    if (W > 64) return TC_HSLOTS * (uint32_t)W * 128u;                                   // ring
    return (uint32_t)(hidden_layers - 1) * KC * (uint32_t)W * 128u + KC * TC_NOUT_PAD * 128u;   // resident
}
__host__ __device__ inline TcSmemLayout tc_smem_layout(int W, int hidden_layers, int w1_slots)
{
    TcSmemLayout L;
    uint32_t off = 0;
    L.w_hid = off;   off += (tc_hid_bytes(W, hidden_layers) + 1023u) & ~1023u;
    L.w1 = off;      off += (uint32_t)w1_slots * (uint32_t)W * 128u;
    L.ray_buf = off; off += (uint32_t)TC_RAY_BUFS * TC_RAY_FIELDS * TC_TILE * 4u;
    L.bars = off;    off += 1024;
    L.total = off + 1024;                       // slack for the manual 1024-byte alignment
    return L;
}

enum { BAR_A_FULL = 0, BAR_A_EMPTY = BAR_A_FULL + TC_MAX_A_SLOTS, BAR_W1_FULL = BAR_A_EMPTY + TC_MAX_A_SLOTS,
       BAR_W1_EMPTY = BAR_W1_FULL + TC_MAX_W1_SLOTS, BAR_ACC_FULL = BAR_W1_EMPTY + TC_MAX_W1_SLOTS,
       BAR_ACC_EMPTY = BAR_ACC_FULL + TC_MAX_ACC, BAR_RAY_FULL = BAR_ACC_EMPTY + TC_MAX_ACC, BAR_RAY_EMPTY = BAR_RAY_FULL + TC_RAY_BUFS,
       BAR_HID = BAR_RAY_EMPTY + TC_RAY_BUFS, BAR_HFULL = BAR_HID + 2, BAR_HEMPTY = BAR_HFULL + TC_HSLOTS,
       BAR_WRES = BAR_HEMPTY + TC_HSLOTS, BAR_COUNT = BAR_WRES + 1 };

// ---- (a3) gathers of one sample, software-pipelined in batches of 8/F levels (16 loads of 4 B for
// F = 2, 8 loads of 8 B for F = 4).  issue() computes the 8 table indices of each level of the batch
// (index rule and corner order of nif_level_features, R6) and issues the loads; consume()
// interpolates in fp32 and returns the batch's 4 features as two packed half2.  Two batches are in
// flight per thread: the next batch's loads are issued before the current one is consumed.
struct TcLevel {            // per-level constants, staged in shared memory (one LDS.128 per level)
    float fn;               // N
    uint32_t np1;           // N+1 for a dense level, 0 for a hashed one
    const void* base;       // &table[l][0][0].  Read back from shared memory on purpose: a base the compiler can
                            // prove warp-uniform stays in uniform registers and every gather address then costs an
                            // IADD3 + IADD3.X pair; a base in a vector register pair makes it ONE IMAD.WIDE.U32
};
static_assert(sizeof(TcLevel) == 16, "TcLevel is read with one LDS.128");

// L1 eviction priority of the table gathers.  Measured (cfg 1 / cfg 4 encode+MLP ms): plain __ldg 0.711 /
// 10.69; evict_last on every level 0.708 / 10.47; evict_first or no_allocate on the fine (hashed) levels
// 0.96 / 11.8 and 1.21 / 20.3 -- even the random fine-level gathers live on L1 reuse (the two x-corners of
// a cell share a sector half of the time, entry and exit points share cells), so nothing is streamed past L1.
#ifndef NIF_TC_FINE_FROM
#define NIF_TC_FINE_FROM 0             // levels >= this use the hint below
#endif
#ifndef NIF_TC_FINE_HINT
#define NIF_TC_FINE_HINT "L1::evict_last"
#endif
// OFF = immediate byte offset, so that the +x corner of a dense cell shares its neighbour's address register
template <bool FINE, int OFF = 0> __device__ __forceinline__ uint32_t ldg_hint(const uint32_t* p)
{
    uint32_t v;
    if constexpr (FINE) asm volatile("ld.global.nc." NIF_TC_FINE_HINT ".b32 %0, [%1+%2];" : "=r"(v) : "l"(p), "n"(OFF));
    else {
#ifdef NIF_TC_COARSE_HINT
        asm volatile("ld.global.nc." NIF_TC_COARSE_HINT ".b32 %0, [%1+%2];" : "=r"(v) : "l"(p), "n"(OFF));
#else
        asm volatile("ld.global.nc.b32 %0, [%1+%2];" : "=r"(v) : "l"(p), "n"(OFF));
#endif
    }
    return v;
}
template <bool FINE, int OFF = 0> __device__ __forceinline__ uint2 ldg_hint(const uint2* p)
{
    uint2 v;
    if constexpr (FINE) asm volatile("ld.global.nc." NIF_TC_FINE_HINT ".v2.b32 {%0, %1}, [%2+%3];" : "=r"(v.x), "=r"(v.y) : "l"(p), "n"(OFF));
    else asm volatile("ld.global.nc.v2.b32 {%0, %1}, [%2+%3];" : "=r"(v.x), "=r"(v.y) : "l"(p), "n"(OFF));
    return v;
}

// (a ^ b) & m as ONE LOP3 (left to itself the compiler folds the y/z hash xor into every corner and spends
// a second LOP3 per corner on the mask)
__device__ __forceinline__ uint32_t xor_and(uint32_t a, uint32_t b, uint32_t m)
{
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, 0x28;" : "=r"(d) : "r"(a), "r"(b), "r"(m));
    return d;
}

template <int F>
struct GatherBatch {
    static constexpr int NL = 4 / F;                          // levels per batch
    typedef typename std::conditional<F == 2, uint32_t, uint2>::type raw_t;
    raw_t raw[NL][8];
    float wx[NL], wy[NL], wz[NL];

    __device__ __forceinline__ void issue(const TcLevel* __restrict__ s_lvl, int log2_T, int l0, float px, float py, float pz)
    {
        if (l0 >= NIF_TC_FINE_FROM) issue_t<true>(s_lvl, log2_T, l0, px, py, pz);
        else issue_t<false>(s_lvl, log2_T, l0, px, py, pz);
    }
    template <bool FINE>
    __device__ __forceinline__ void issue_t(const TcLevel* __restrict__ s_lvl, int log2_T, int l0, float px, float py, float pz)
    {
        const uint32_t t_mask = (1u << log2_T) - 1u;
#pragma unroll
        for (int li = 0; li < NL; ++li) {
            const int l = l0 + li;
            const uint4 lv = *reinterpret_cast<const uint4*>(s_lvl + l);
            const float fn = __uint_as_float(lv.x), top = fn - 1.0f;
            const uint32_t np1 = lv.y;
            const raw_t* lvl = reinterpret_cast<const raw_t*>(((unsigned long long)lv.w << 32) | (unsigned long long)lv.z);
            const float posx = px * fn, posy = py * fn, posz = pz * fn;           // p in [0,1]: floor >= 0
            const float flx = fminf(floorf(posx), top), fly = fminf(floorf(posy), top), flz = fminf(floorf(posz), top);
            wx[li] = posx - flx; wy[li] = posy - fly; wz[li] = posz - flz;
            const uint32_t cx = (uint32_t)flx, cy = (uint32_t)fly, cz = (uint32_t)flz;
            // entry indices (32-bit) from the level's base: each gather address is one IMAD.WIDE.U32
            if (np1) {
                // dense: the +x corner is the next entry -> same address register, immediate offset
                const uint32_t o2 = np1 * np1;
                const uint32_t i00 = cx + np1 * cy + o2 * cz, i10 = i00 + np1, i01 = i00 + o2, i11 = i01 + np1;
                const raw_t *q00 = lvl + i00, *q10 = lvl + i10, *q01 = lvl + i01, *q11 = lvl + i11;
                constexpr int E = (int)sizeof(raw_t);
                raw[li][0] = ldg_hint<FINE, 0>(q00); raw[li][1] = ldg_hint<FINE, E>(q00);
                raw[li][2] = ldg_hint<FINE, 0>(q10); raw[li][3] = ldg_hint<FINE, E>(q10);
                raw[li][4] = ldg_hint<FINE, 0>(q01); raw[li][5] = ldg_hint<FINE, E>(q01);
                raw[li][6] = ldg_hint<FINE, 0>(q11); raw[li][7] = ldg_hint<FINE, E>(q11);
            } else {
                const uint32_t hy0 = cy * 2654435761u, hy1 = hy0 + 2654435761u;
                const uint32_t hz0 = cz * 805459861u, hz1 = hz0 + 805459861u;
                const uint32_t hyz[4] = {hy0 ^ hz0, hy1 ^ hz0, hy0 ^ hz1, hy1 ^ hz1};
                const uint32_t x1 = cx + 1u;
#pragma unroll
                for (int c = 0; c < 8; ++c) raw[li][c] = ldg_hint<FINE>(lvl + xor_and((c & 1) ? x1 : cx, hyz[c >> 1], t_mask));
            }
        }
    }

    __device__ __forceinline__ void consume(uint32_t& p0, uint32_t& p1) const
    {
        float f[4];
#pragma unroll
        for (int li = 0; li < NL; ++li) {
            const float x1 = wx[li], x0 = 1.0f - x1, y1 = wy[li], y0 = 1.0f - y1, z1 = wz[li], z0 = 1.0f - z1;
            const float xy[4] = {x0 * y0, x1 * y0, x0 * y1, x1 * y1};
            float acc[F];
#pragma unroll
            for (int k = 0; k < F; ++k) acc[k] = 0.0f;
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                const float w = xy[c & 3] * ((c >> 2) ? z1 : z0);
                if constexpr (F == 2) {
                    const float2 v = __half22float2(*reinterpret_cast<const __half2*>(&raw[li][c]));
                    acc[0] = fmaf(w, v.x, acc[0]); acc[1] = fmaf(w, v.y, acc[1]);
                } else {
                    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&raw[li][c].x));
                    const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&raw[li][c].y));
                    acc[0] = fmaf(w, a.x, acc[0]); acc[1] = fmaf(w, a.y, acc[1]);
                    acc[2] = fmaf(w, b.x, acc[2]); acc[3] = fmaf(w, b.y, acc[3]);
                }
            }
#pragma unroll
            for (int k = 0; k < F; ++k) f[li * F + k] = acc[k];
        }
        p0 = pack_half2(f[0], f[1]);
        p1 = pack_half2(f[2], f[3]);
    }
};

// drains N32*32 fp32 accumulator columns of this thread's row from TMEM, applies ReLU, rounds to fp16
// and writes them back to TMEM as the next layer's A operand (two fp16 per 32-bit column)
template <int W>
__device__ __forceinline__ void drain_relu_to_act(uint32_t tm_src_row, uint32_t tm_act_row)
{
    __syncwarp();                                          // tcgen05.ld / .st are .sync.aligned
#pragma unroll
    for (int cg = 0; cg < W / 32; ++cg) {
        uint32_t v[32], h[16];
        tmem_ld_32x32(tm_src_row + (uint32_t)(cg * 32), v);
        tmem_ld_wait();
#pragma unroll
        for (int i = 0; i < 16; ++i)
            h[i] = pack_half2(fmaxf(__uint_as_float(v[2 * i]), 0.0f), fmaxf(__uint_as_float(v[2 * i + 1]), 0.0f));
        tmem_st_32x16(tm_act_row + (uint32_t)(cg * 16), h);
    }
    tmem_st_wait();
}

template <int W, int F, bool CONCAT, bool LOCAL, bool PROBE>
__global__ void __launch_bounds__(TC_THREADS, 1)
k_fused_encode_mlp(const TcParams p)
{
    constexpr int NG = (W == 128) ? 1 : 2;                 // tail groups
    constexpr int KC = (W + 63) / 64;                      // K chunks of a hidden layer
    constexpr int K16 = (W < 64 ? W : 64) / 16;            // UMMA K steps per hidden chunk
    constexpr uint32_t HCHUNK = (uint32_t)W * 128u;        // one weight chunk: W rows x 64 fp16
    constexpr uint32_t OUTCHUNK = TC_NOUT_PAD * 128u;
    constexpr uint32_t ACT_COLS = W / 2;
    // TMEM columns: [accumulator x NACC][activations x NG][A ring].  A tile keeps ONE accumulator buffer from its first
    // layer-1 MMA to the read of its output: the hidden/output layers accumulate into the drained layer-1 buffer.  W <= 64:
    // three buffers, so that the layer-1 MMAs of tile t+1 never wait for the tails of tiles t and t-1 (one per tail
    // group), and 8 ring slots; W = 128: two buffers (one tail group), 6 ring slots.  (Round 2 first gave W <= 64 two
    // layer-1 buffers plus a hidden accumulator per tail group -- 6 ring slots; the deeper ring decouples the gather
    // warps better: config 1 0.670 -> 0.656 ms.)
    constexpr int NACC = (W == 128) ? 2 : 3;
    constexpr uint32_t C_ACT = (uint32_t)NACC * W;
    constexpr uint32_t C_RING = C_ACT + NG * ACT_COLS;
    constexpr int A_SLOTS = (512 - (int)C_RING) / 32 < TC_MAX_A_SLOTS ? (512 - (int)C_RING) / 32 : TC_MAX_A_SLOTS;
    constexpr uint32_t TMEM_COLS = 512;
    static_assert(A_SLOTS >= 2, "layer-1 A ring too short");

    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    const TcSmemLayout SL = tc_smem_layout(W, p.hidden_layers, p.w1_slots);
    const uint32_t s_whid = smem_base + SL.w_hid, s_w1 = smem_base + SL.w1;
    float* ray_buf = reinterpret_cast<float*>(smem_gen + SL.ray_buf);          // [TC_RAY_BUFS][TC_RAY_FIELDS][128]
    const uint32_t s_bar = smem_base + SL.bars;
    static_assert(8 * BAR_COUNT <= 480, "barrier block overlaps the tile-id / TMEM pointer slots");
    volatile int* s_tile = reinterpret_cast<volatile int*>(smem_gen + SL.bars + 480);    // [TC_RAY_BUFS]
    uint32_t* s_tmem_ptr = reinterpret_cast<uint32_t*>(smem_gen + SL.bars + 496);
    auto bar = [&](int i) { return s_bar + 8u * (uint32_t)i; };

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int L = p.enc.levels, S = 1 + 2 * p.enc.bands;
    const int epc = p.es_per_chunk, n_chunks = p.n_chunks;
    const uint32_t W1_SLOTS = (uint32_t)p.w1_slots;

    // ---- one-time setup ------------------------------------------------------------------------
    if (tid == 0) {
        for (int i = 0; i < TC_MAX_A_SLOTS; ++i) { mbar_init(bar(BAR_A_FULL + i), 4u * (uint32_t)epc); mbar_init(bar(BAR_A_EMPTY + i), 1); }
        for (int i = 0; i < TC_MAX_W1_SLOTS; ++i) { mbar_init(bar(BAR_W1_FULL + i), 1); mbar_init(bar(BAR_W1_EMPTY + i), 1); }
        for (int i = 0; i < TC_HSLOTS; ++i) { mbar_init(bar(BAR_HFULL + i), 1); mbar_init(bar(BAR_HEMPTY + i), 1); }
        for (int i = 0; i < TC_MAX_ACC; ++i) { mbar_init(bar(BAR_ACC_FULL + i), 1); mbar_init(bar(BAR_ACC_EMPTY + i), TC_TILE); }
        for (int i = 0; i < 2; ++i) mbar_init(bar(BAR_HID + i), 1);
        for (int i = 0; i < TC_RAY_BUFS; ++i) {
            mbar_init(bar(BAR_RAY_FULL + i), TC_PREP_THREADS); mbar_init(bar(BAR_RAY_EMPTY + i), TC_GATHER_WARPS + TC_TILE);
        }
        mbar_init(bar(BAR_WRES), 1);
        fence_barrier_init();
    }
    TcLevel* s_lvl = reinterpret_cast<TcLevel*>(smem_gen + SL.bars + 512);      // 16 levels x 16 B
    if (tid < NIF_MAX_LEVELS) {
        const int N = tid < L ? p.enc.res[tid] : 1;
        TcLevel lv;
        lv.fn = (float)N;
        lv.np1 = ((p.enc.dense_mask >> tid) & 1u) ? (uint32_t)N + 1u : 0u;
        lv.base = reinterpret_cast<const char*>(p.table) + ((size_t)tid << (p.enc.log2_T + (F == 2 ? 2 : 3)));
        s_lvl[tid] = lv;
    }
    if (warp == TC_MMA_WARP) tmem_alloc(smem_u32(s_tmem_ptr), TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *s_tmem_ptr;
    const uint32_t tm_acc1 = tmem_base, tm_ring = tmem_base + C_RING;

    const long long n_hit = (long long)p.scratch->n_hit;
    const long long n_tiles = (n_hit + TC_TILE - 1) / TC_TILE;

    if (warp < TC_TAIL_WARPS) {
        // ======================= tail groups: MLP layers 2.. and (a5), alternating tiles ===========
        reg_dec<TC_REGS_TAIL>();
        const int g = warp >> 2;
        if (g < NG) {
            const int tg = tid - g * TC_TILE;                              // row of the tile / TMEM lane
            const uint32_t t_row = (uint32_t)((warp & 3) * 32) << 16;
            const uint32_t tm_act = tmem_base + C_ACT + (uint32_t)g * ACT_COLS;
            uint32_t hid_phase = 0, hq = 0;
            const bool issuer = (warp & 3) == 0;                           // the group's first warp issues its MMAs (converged)
            if (W <= 64 && issuer) mbar_wait_sleep(bar(BAR_WRES), 0);     // resident hidden/output weights landed
            // one layer of this group's tile: A = the group's activations (TMEM), B = weight chunks, D = d_tmem
            auto run_layer = [&](uint32_t d_tmem, int N, int li) {
                tc_fence_after();
                const uint32_t idesc = idesc_f16(TC_TILE, N);
#pragma unroll
                for (int kc = 0; kc < KC; ++kc) {
                    uint32_t wchunk;
                    if constexpr (W <= 64) {
                        wchunk = s_whid + (uint32_t)(li * KC) * HCHUNK + (uint32_t)kc * (N == TC_NOUT_PAD ? OUTCHUNK : HCHUNK);
                    } else {
                        const uint32_t slot = hq % TC_HSLOTS;
                        mbar_wait_sleep(bar(BAR_HFULL + slot), (hq / TC_HSLOTS) & 1u);
                        tc_fence_after();
                        __syncwarp();
                        wchunk = s_whid + slot * HCHUNK;
                    }
                    // the chunk's commit releases the weight slot (W = 128) or, on the last chunk, signals the layer
                    const uint32_t cbar = (W > 64 && kc + 1 < KC) ? bar(BAR_HEMPTY + (hq % TC_HSLOTS)) : bar(BAR_HID + g);
                    umma_chunk_ts<K16>(d_tmem, tm_act + (uint32_t)(kc * 32), smem_desc_sw128(wchunk), idesc, (uint32_t)(kc != 0), cbar);
                    if constexpr (W > 64) { if (kc + 1 == KC) umma_commit_elect(bar(BAR_HEMPTY + (hq % TC_HSLOTS))); ++hq; }
                }
            };
            for (int j = g;; j += NG) {
                const int nb = j % TC_RAY_BUFS, b = j % NACC;
                mbar_wait_sleep(bar(BAR_RAY_FULL + nb), (uint32_t)((j / TC_RAY_BUFS) & 1));
                if (s_tile[nb] < 0) break;
                const float* rb = ray_buf + (size_t)nb * TC_RAY_FIELDS * TC_TILE + tg;
                const float cur_ti = rb[6 * TC_TILE], cur_to = rb[7 * TC_TILE];
                const long long cur_ray = (long long)__float_as_int(rb[8 * TC_TILE]);
                mbar_arrive(bar(BAR_RAY_EMPTY + nb));
                const uint32_t tm_l1 = tm_acc1 + (uint32_t)(b * W);
                const uint32_t tm_hid = tm_l1;
                if (tg == 0) TC_TRACE(j, 1);
                // layer 1 accumulator of tile j -> ReLU -> fp16 activations
                mbar_wait_sleep(bar(BAR_ACC_FULL + b), (uint32_t)((j / NACC) & 1));
                if (tg == 0) TC_TRACE(j, 2);
                tc_fence_after();
                drain_relu_to_act<W>(tm_l1 + t_row, tm_act + t_row);
                tc_fence_before();
                named_bar_sync(1 + g, TC_TILE);
                if (tg == 0) TC_TRACE(j, 3);
                // hidden layers 2..H
                for (int hl = 1; hl < p.hidden_layers; ++hl) {
                    if (issuer) run_layer(tm_hid, W, hl - 1);
                    mbar_wait_sleep(bar(BAR_HID + g), hid_phase); hid_phase ^= 1u;
                    tc_fence_after();
                    drain_relu_to_act<W>(tm_hid + t_row, tm_act + t_row);
                    tc_fence_before();
                    named_bar_sync(1 + g, TC_TILE);
                    if (tg == 0) TC_TRACE(j, 3 + hl);
                }
                // output layer (12 heads padded to N = 16) and (a5) decode
                if (issuer) run_layer(tm_hid, TC_NOUT_PAD, p.hidden_layers - 1);
                mbar_wait_sleep(bar(BAR_HID + g), hid_phase); hid_phase ^= 1u;
                if (tg == 0) TC_TRACE(j, 20);
                tc_fence_after();
                uint32_t zr[16];
                __syncwarp();
                tmem_ld_32x16(tm_hid + t_row, zr);
                tmem_ld_wait();
                tc_fence_before();
                mbar_arrive(bar(BAR_ACC_EMPTY + b));
                if (cur_ray >= 0) {
                    float z[NIF_N_OUT];
#pragma unroll
                    for (int a = 0; a < NIF_N_OUT; ++a) z[a] = __uint_as_float(zr[a]);
                    nif_decode_store<LOCAL>(z, cur_ti, cur_to, cur_ray, p.out, p.flags, NifDecodeCtx{p.origin, p.dir, p.map, p.batch});
                }
                if (tg == 0) TC_TRACE(j, 22);
            }
        }
    } else if (warp < TC_GATHER_WARP0) {
        reg_dec<TC_REGS_MISC>();
        if (warp == TC_MMA_WARP) {
            // ======================= layer-1 MMA issuer (whole warp converged, one elected lane issues) ====
            {
                const uint32_t idesc = idesc_f16(TC_TILE, W);
                if (p.w1_resident) mbar_wait_sleep(bar(BAR_WRES), 0);
                // one full/empty barrier pair per chunk slot (pairs per group of two chunks were measured: slower, 7.7)
                const uint64_t w1_desc0 = smem_desc_sw128(s_w1);
                // the loop body is instantiated per residency: this warp's instruction stream is what bounds the tensor
                // pipe on narrow layers, so nothing it can decide once is decided per chunk
                auto layer1 = [&](auto resident_tag) {
                    constexpr bool RES = decltype(resident_tag)::value;
                    uint32_t gs = 0, gph = 0, ws = 0, wph = 0;            // A slot + phase; streamed-W1 slot + phase
                    for (int j = 0;; ++j) {
                        const int nb = j % TC_RAY_BUFS, b = j % NACC;
                        mbar_wait_sleep(bar(BAR_RAY_FULL + nb), (uint32_t)((j / TC_RAY_BUFS) & 1));
                        if (s_tile[nb] < 0) break;
                        mbar_wait_sleep(bar(BAR_ACC_EMPTY + b), (uint32_t)(((j / NACC) & 1) ^ 1));
                        if (lane == 0) TC_TRACE(j, 25);
                        tc_fence_after();
                        __syncwarp();
                        const uint32_t d_tmem = tm_acc1 + (uint32_t)(b * W);
                        uint64_t bdesc = w1_desc0;
                        for (int c = 0; c < n_chunks; ++c) {
                            const uint32_t a_tmem = tm_ring + gs * 32u, a_empty = bar(BAR_A_EMPTY + gs);    // before the wait
                            mbar_wait_sleep(bar(BAR_A_FULL + gs), gph);
                            if (c == 0 && lane == 0) TC_TRACE(j, 26);
                            if constexpr (!RES) {
                                mbar_wait_sleep(bar(BAR_W1_FULL + ws), wph);
                                bdesc = w1_desc0 + (uint64_t)(ws * (HCHUNK >> 4));
                            }
                            tc_fence_after();
                            __syncwarp();
                            umma_chunk_ts<4>(d_tmem, a_tmem, bdesc, idesc, (uint32_t)(c != 0), a_empty);
                            if constexpr (RES) bdesc += (uint64_t)(HCHUNK >> 4);
                            else {
                                umma_commit_elect(bar(BAR_W1_EMPTY + ws));
                                if (++ws == W1_SLOTS) { ws = 0; wph ^= 1u; }
                            }
                            if (++gs == (uint32_t)A_SLOTS) { gs = 0; gph ^= 1u; }
                        }
                        umma_commit_elect(bar(BAR_ACC_FULL + b));
                        if (lane == 0) TC_TRACE(j, 27);
                    }
                };
                if (p.w1_resident) layer1(std::true_type{}); else layer1(std::false_type{});
            }
        } else if (warp == TC_LOAD_WARP) {
            // ======================= weights: global (L2) -> shared memory, cp.async.bulk ============
            if (lane == 0) {
                const uint32_t hid_total = (W <= 64) ? (p.w_bytes - p.w1_bytes) : 0u;
                const uint32_t res_bytes = hid_total + (p.w1_resident ? p.w1_bytes : 0u);
                if (res_bytes) {
                    mbar_expect_tx(bar(BAR_WRES), res_bytes);
                    for (uint32_t off = 0; off + 1u <= hid_total; off += 8192u) {
                        const uint32_t nbytes = hid_total - off < 8192u ? hid_total - off : 8192u;
                        bulk_g2s(s_whid + off, p.w_img + p.w1_bytes + off, nbytes, bar(BAR_WRES));
                    }
                    if (p.w1_resident)
                        for (int c = 0; c < n_chunks; ++c)
                            bulk_g2s(s_w1 + (uint32_t)c * HCHUNK, p.w_img + (size_t)c * HCHUNK, HCHUNK, bar(BAR_WRES));
                } else {
                    mbar_arrive(bar(BAR_WRES));
                }
                if (!p.w1_resident) {
                    // layer-1 weight chunks stream through the ring in the order the MMA warp consumes them
                    uint32_t q = 0;
                    for (int j = 0;; ++j) {
                        const int nb = j % TC_RAY_BUFS;
                        mbar_wait_sleep(bar(BAR_RAY_FULL + nb), (uint32_t)((j / TC_RAY_BUFS) & 1));
                        if (s_tile[nb] < 0) break;
                        for (int c = 0; c < n_chunks; ++c, ++q) {
                            const uint32_t ws = q % W1_SLOTS;
                            mbar_wait_sleep(bar(BAR_W1_EMPTY + ws), ((q / W1_SLOTS) & 1u) ^ 1u);
                            mbar_expect_tx(bar(BAR_W1_FULL + ws), HCHUNK);
                            bulk_g2s(s_w1 + ws * HCHUNK, p.w_img + (size_t)c * HCHUNK, HCHUNK, bar(BAR_W1_FULL + ws));
                        }
                    }
                }
            } else if (lane == 1 && W > 64) {
                // W = 128: hidden layers 2..H and the output layer, KC chunks each, per tile, in the order the
                // (single) tail group consumes them
                const uint8_t* wh = p.w_img + p.w1_bytes;
                uint32_t hq = 0;
                for (int j = 0;; ++j) {
                    const int nb = j % TC_RAY_BUFS;
                    mbar_wait_sleep(bar(BAR_RAY_FULL + nb), (uint32_t)((j / TC_RAY_BUFS) & 1));
                    if (s_tile[nb] < 0) break;
                    for (int l = 1; l <= p.hidden_layers; ++l) {
                        const bool is_out = l == p.hidden_layers;
                        const uint32_t bytes = is_out ? OUTCHUNK : HCHUNK;
                        const uint8_t* src = wh + (size_t)(l - 1) * (size_t)(KC * HCHUNK);
                        for (int kc = 0; kc < KC; ++kc, ++hq) {
                            const uint32_t slot = hq % TC_HSLOTS;
                            mbar_wait_sleep(bar(BAR_HEMPTY + slot), ((hq / TC_HSLOTS) & 1u) ^ 1u);
                            mbar_expect_tx(bar(BAR_HFULL + slot), bytes);
                            bulk_g2s(s_whid + slot * HCHUNK, src + (size_t)kc * bytes, bytes, bar(BAR_HFULL + slot));
                        }
                    }
                }
            }
        } else {
            // ======================= prep warps: tile ids, ray fetch, (a2) map back =====================
            const int pt = tid - TC_PREP_WARP0 * 32;                       // 0..63, two rays each
            unsigned next_t = 0;
            if (pt == 0) next_t = atomicAdd(p.tile_counter, 1u);
            int n_term = 0;
            for (int j = 0;; ++j) {
                const int nb = j % TC_RAY_BUFS;
                mbar_wait_sleep(bar(BAR_RAY_EMPTY + nb), (uint32_t)(((j / TC_RAY_BUFS) & 1) ^ 1));
                if (pt == 0) {
                    const int t = (long long)next_t < n_tiles ? (int)next_t : -1;
                    s_tile[nb] = t;
                    if (t >= 0) next_t = atomicAdd(p.tile_counter, 1u);    // next tile's id: latency hidden behind this tile's loads
                    TC_TRACE(j, 0);
                }
                named_bar_sync(3, TC_PREP_THREADS);
                const int tile = s_tile[nb];
                float* rbuf = ray_buf + (size_t)nb * TC_RAY_FIELDS * TC_TILE;
#pragma unroll 1
                for (int half = 0; half < 2; ++half) {
                    const int r = pt + TC_PREP_THREADS * half;
                    const long long h = tile < 0 ? n_hit : (long long)tile * TC_TILE + r;
                    float xi = 0.f, yi = 0.f, zi = 0.f, xo = 0.f, yo = 0.f, zo = 0.f, ti = 0.f, to = 0.f;
                    long long ray = -1;
                    if (PROBE && h < n_hit) {                // MLP-only probe: ray fetch only, no map back (a2)
                        ray = p.hit_list[h];
                        ti = p.out.t_in[ray]; to = p.out.t_out[ray];
                    } else if (h < n_hit) {
                        ray = p.hit_list[h];
                        ti = p.out.t_in[ray]; to = p.out.t_out[ray];
                        const float ox = p.origin[3 * ray], oy = p.origin[3 * ray + 1], oz = p.origin[3 * ray + 2];
                        const float dx = p.dir[3 * ray], dy = p.dir[3 * ray + 1], dz = p.dir[3 * ray + 2];
                        if constexpr (LOCAL) {           // deformation given as a lattice: voxel-local inverse (R27)
                            const float oo[3] = {ox, oy, oz}, dd[3] = {dx, dy, dz};
                            float ri[3], ro[3];
                            nif_map_back_pair<true>(nif_ray_map(p.map, p.batch, ray), p.out.voxel_id[ray], oo, dd, ti, to, ri, ro);
                            xi = ri[0]; yi = ri[1]; zi = ri[2]; xo = ro[0]; yo = ro[1]; zo = ro[2];
                        } else {
                            float th = p.theta_max, bk = p.bend_k;
                            if (p.batch.pose_id) {           // nif_query_poses: this ray's pose
                                const NifPoseDesc* pd = p.batch.poses + p.batch.pose_id[ray];
                                th = pd->theta_max; bk = pd->bend_k;
                            }
                            nif_inverse_deform(th, bk, fmaf(ti, dx, ox), fmaf(ti, dy, oy), fmaf(ti, dz, oz), xi, yi, zi);
                            nif_inverse_deform(th, bk, fmaf(to, dx, ox), fmaf(to, dy, oy), fmaf(to, dz, oz), xo, yo, zo);
                        }
                    }
                    rbuf[0 * TC_TILE + r] = nif_normalise(xi); rbuf[1 * TC_TILE + r] = nif_normalise(yi); rbuf[2 * TC_TILE + r] = nif_normalise(zi);
                    rbuf[3 * TC_TILE + r] = nif_normalise(xo); rbuf[4 * TC_TILE + r] = nif_normalise(yo); rbuf[5 * TC_TILE + r] = nif_normalise(zo);
                    rbuf[6 * TC_TILE + r] = ti; rbuf[7 * TC_TILE + r] = to; rbuf[8 * TC_TILE + r] = __int_as_float((int)ray);
                }
                mbar_arrive(bar(BAR_RAY_FULL + nb));
                if (tile < 0 && ++n_term == NG) break;                     // every tail group sees its own end marker
            }
        }
    } else {
        // ======================= gather warps: (a3) encode into the TMEM A ring =====================
        reg_inc<TC_REGS_GATHER>();
        const int gw = warp - TC_GATHER_WARP0;
        const int g = gw & 3, qr = gw >> 2;                                // row group (= TMEM lane quarter), rank in the group
        const uint32_t row = (uint32_t)(g * 32 + lane);
        const uint32_t t_row = (uint32_t)(g * 32) << 16;
        const int n_pairs = n_chunks * epc;                                // (endpoint, sample) slots per tile, padding included
        const int units_per_es = (L * F) / 8;                              // 16-byte units (4 TMEM columns) one sample fills
        for (int j = 0;; ++j) {
            const int nb = j % TC_RAY_BUFS;
            mbar_wait(bar(BAR_RAY_FULL + nb), (uint32_t)((j / TC_RAY_BUFS) & 1));
            if (s_tile[nb] < 0) break;
            const float* rb = ray_buf + (size_t)nb * TC_RAY_FIELDS * TC_TILE + row;
            const long long p0 = (long long)j * n_pairs;
            const int first = (int)(((long long)qr - p0 % TC_GPR + TC_GPR) % TC_GPR);
            for (int e = first; e < n_pairs; e += TC_GPR) {
                const int c = e / epc, esl = e - c * epc;
                const int es = e;
                const uint32_t gq = (uint32_t)j * (uint32_t)n_chunks + (uint32_t)c;                  // chunk counter
                const uint32_t slot = gq % (uint32_t)A_SLOTS;
                mbar_wait(bar(BAR_A_EMPTY + slot), ((gq / (uint32_t)A_SLOTS) & 1u) ^ 1u);
                __syncwarp();                                              // tcgen05.st is .sync.aligned
                tc_fence_after();
                const uint32_t a_dst = tm_ring + slot * 32u + (uint32_t)(esl * units_per_es) * 4u + t_row;
                if constexpr (PROBE) {
                    // MLP-only probe: synthetic features, no table access.  The constant is written on the first pass
                    // over the ring only (the MMAs do not modify A): afterwards an item is the slot hand-over alone, so
                    // that the probe measures the MLP pipeline and not the cost of faking its input
                    if (gq < (uint32_t)A_SLOTS)
                        for (int u = 0; u < units_per_es; ++u)
                            tmem_st_32x4(a_dst + (uint32_t)u * 4u, 0x2c002c00u, 0x2c002c00u, 0x2c002c00u, 0x2c002c00u);
                } else if (CONCAT && es >= 2 && es < p.n_es) {
                    // NIF_ENC_CONCAT: items 0, 1 are phi(entry), phi(exit); the rest carry the gamma scalars as
                    // they are: L*F = 32 -> two 32-column items per endpoint, L*F = 64 -> one 64-column item
                    const int pe_item = es - 2;
                    const int en = (L * F == 32) ? pe_item >> 1 : pe_item;
                    const int jbase = (L * F == 32) ? (pe_item & 1) * 32 : 0;
                    const float xr[3] = {rb[(3 * en) * TC_TILE], rb[(3 * en + 1) * TC_TILE], rb[(3 * en + 2) * TC_TILE]};
                    for (int u = 0; u < units_per_es; ++u) {
                        float v[8];
#pragma unroll
                        for (int i = 0; i < 8; ++i) v[i] = nif_pe_scalar(xr, jbase + 8 * u + i, p.enc.bands);
                        tmem_st_32x4(a_dst + (uint32_t)u * 4u, pack_half2(v[0], v[1]), pack_half2(v[2], v[3]),
                                     pack_half2(v[4], v[5]), pack_half2(v[6], v[7]));
                    }
                } else if (es < p.n_es) {
                    const int en = CONCAT ? es : (es >= S ? 1 : 0);
                    const int s = CONCAT ? 0 : es - en * S;
                    const float px = nif_pe_sample(rb[(3 * en) * TC_TILE], s), py = nif_pe_sample(rb[(3 * en + 1) * TC_TILE], s),
                                pz = nif_pe_sample(rb[(3 * en + 2) * TC_TILE], s);
                    GatherBatch<F> ba, bb;                                     // two batches in flight
                    constexpr int NL = GatherBatch<F>::NL;
                    ba.issue(s_lvl, p.enc.log2_T, 0, px, py, pz);
                    for (int u = 0; u < units_per_es; ++u) {
                        uint32_t pk[4];
                        bb.issue(s_lvl, p.enc.log2_T, (2 * u + 1) * NL, px, py, pz);
                        ba.consume(pk[0], pk[1]);
                        if (u + 1 < units_per_es) ba.issue(s_lvl, p.enc.log2_T, (2 * u + 2) * NL, px, py, pz);
                        bb.consume(pk[2], pk[3]);
                        __syncwarp();
                        tmem_st_32x4(a_dst + (uint32_t)u * 4u, pk[0], pk[1], pk[2], pk[3]);
                    }
                } else {
                    for (int u = 0; u < units_per_es; ++u) tmem_st_32x4(a_dst + (uint32_t)u * 4u, 0u, 0u, 0u, 0u);
                }
                tmem_st_wait();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(BAR_A_FULL + slot));
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(BAR_RAY_EMPTY + nb));
        }
    }

    // ---- teardown --------------------------------------------------------------------------------
    tc_fence_before();
    __syncthreads();
    if (warp == TC_MMA_WARP) { tc_fence_after(); __syncwarp(); tmem_dealloc(tmem_base, TMEM_COLS); }
}

// ---- weight repacking: row-major (fan_out, fan_in) fp16 -> K-major SWIZZLE_128B B-operand images ----
// image of one layer = ceil(K/64) chunks of [n_rows x 128 B]; element (n, k) sits in chunk k/64 at
// sw128_off(n, (k%64)/8) + (k%8)*2.  Rows/columns beyond the real matrix stay zero.
__global__ void k_pack_weights(const __half* __restrict__ w, int fan_out, int fan_in, int n_rows,
                               uint8_t* __restrict__ img, int concat_lf, int concat_npe)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= fan_out * fan_in) return;
    const int n = i / fan_in;
    int k = i - n * fan_in;
    if (concat_lf) {
        // NIF_ENC_CONCAT, layer 1: user column e*per + j (per = npe + L*F, gamma scalars first) -> K index of
        // the kernel's item layout: phi(e, j) at e*L*F + j, gamma(e, j) at 2*L*F + 64*e + j
        const int per = concat_npe + concat_lf, e = k / per, j = k - e * per;
        k = j < concat_npe ? 2 * concat_lf + 64 * e + j : e * concat_lf + (j - concat_npe);
    }
    const uint32_t off = (uint32_t)(k / 64) * (uint32_t)(n_rows * 128) + sw128_off((uint32_t)n, (uint32_t)((k % 64) / 8)) +
                         (uint32_t)(k % 8) * 2u;
    *reinterpret_cast<__half*>(img + off) = w[i];
}

struct TcShape {
    int S, n_es, lf, epc, n_chunks, KC;
    uint32_t w1_bytes, wh_bytes, wo_bytes, w_bytes;
};
TcShape tc_shape(const nif_net_desc* d)
{
    TcShape s{};
    s.S = 1 + 2 * d->pe_bands; s.n_es = 2 * s.S; s.lf = d->levels * d->feat;
    if (d->enc_mode == NIF_ENC_CONCAT) s.n_es = 2 + 128 / (s.lf > 0 ? s.lf : 128);     // phi(entry), phi(exit) + gamma items of lf columns
    s.epc = s.lf > 0 && s.lf <= 64 ? 64 / s.lf : 0;
    s.n_chunks = s.epc ? (s.n_es + s.epc - 1) / s.epc : 0;
    s.KC = (d->width + 63) / 64;
    s.w1_bytes = (uint32_t)s.n_chunks * (uint32_t)d->width * 128u;
    s.wh_bytes = (uint32_t)(d->hidden_layers - 1) * (uint32_t)s.KC * (uint32_t)d->width * 128u;
    s.wo_bytes = (uint32_t)s.KC * TC_NOUT_PAD * 128u;
    s.w_bytes = s.w1_bytes + s.wh_bytes + s.wo_bytes;
    return s;
}

// Shared-memory budget: 163 KB keeps the kernel inside the 164 KB carve-out, which leaves the L1 data cache
// large enough to keep the gathers' misses in flight.  Layer-1 weights are resident when
// everything fits that budget (config 1-3: 104 KB + 18 KB + 14 KB), otherwise they stream through as many
// chunk slots as fit (4..8).
#ifndef NIF_TC_SMEM_BUDGET
#define NIF_TC_SMEM_BUDGET (163u * 1024u)
#endif
struct TcW1Plan { int slots, resident; };
TcW1Plan tc_plan_w1(int W, int hidden_layers, int n_chunks)
{
    const uint32_t fixed = tc_smem_layout(W, hidden_layers, 0).total;
    const uint32_t chunk = (uint32_t)W * 128u;
#ifndef NIF_TC_FORCE_STREAM
    if (fixed + (uint32_t)n_chunks * chunk <= NIF_TC_SMEM_BUDGET) return TcW1Plan{n_chunks, 1};
#endif
    int slots = fixed < NIF_TC_SMEM_BUDGET ? (int)((NIF_TC_SMEM_BUDGET - fixed) / chunk) : 0;
    if (slots > TC_MAX_W1_SLOTS) slots = TC_MAX_W1_SLOTS;
    if (slots > n_chunks) slots = n_chunks;
    if (slots < 2 && slots < n_chunks) return TcW1Plan{0, 0};
    return TcW1Plan{slots, 0};
}

template <int W, int F, bool CONCAT, bool LOCAL, bool PROBE>
int launch_tc(const TcParams& p, uint32_t smem, int blocks, cudaStream_t stream)
{
    NIF_CUDA_TRY(cudaFuncSetAttribute(k_fused_encode_mlp<W, F, CONCAT, LOCAL, PROBE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_fused_encode_mlp<W, F, CONCAT, LOCAL, PROBE><<<blocks, TC_THREADS, smem, stream>>>(p);
    nif_count_launch(1);
    NIF_CUDA_TRY(cudaGetLastError());
    return NIF_OK;
}

}  // namespace

#ifdef NIF_TC_TRACE
extern "C" int nif_debug_set_tc_trace(void* buf)
{
    return cudaMemcpyToSymbol(g_tc_trace, &buf, sizeof(buf)) == cudaSuccess ? 0 : -5;
}
#endif

int nif_tc_supported(const nif_net_desc* d)
{
    if (d->dtype != NIF_F16) return 0;
    if (d->feat != 2 && d->feat != 4) return 0;
    if (d->width != 32 && d->width != 64 && d->width != 128) return 0;
    const int lf = d->levels * d->feat;
    if (lf != 8 && lf != 16 && lf != 32 && lf != 64) return 0;
    if (d->enc_mode == NIF_ENC_CONCAT && ((lf != 32 && lf != 64) || 3 + 6 * d->pe_bands > 64)) return 0;
    if (d->hidden_layers < 1) return 0;
    const TcShape s = tc_shape(d);
    if (d->width <= 64 && tc_smem_layout(d->width, d->hidden_layers, 2).total > NIF_TC_SMEM_BUDGET) return 0;   // resident hidden weights
    const TcW1Plan plan = tc_plan_w1(d->width, d->hidden_layers, s.n_chunks);
    return (plan.resident && plan.slots >= 1) || plan.slots >= 2 ? 1 : 0;
}

int nif_tc_pack_weights(nif_net* net, cudaStream_t stream)
{
    const nif_net_desc* d = &net->desc;
    const TcShape s = tc_shape(d);
    net->w_tc_bytes = s.w_bytes;
    NIF_CUDA_TRY(cudaMalloc(&net->w_tc, s.w_bytes));
    NIF_CUDA_TRY(cudaMemsetAsync(net->w_tc, 0, s.w_bytes, stream));
    uint8_t* img = (uint8_t*)net->w_tc;
    size_t off = 0;
    for (int i = 0; i <= d->hidden_layers; ++i) {
        const int fan_out = i == d->hidden_layers ? NIF_N_OUT : d->width;
        const int fan_in = i == 0 ? net->d_in : d->width;
        const int n_rows = i == d->hidden_layers ? TC_NOUT_PAD : d->width;
        net->w_tc_layer_off[i] = off;
        const int total = fan_out * fan_in;
        const bool cat = i == 0 && d->enc_mode == NIF_ENC_CONCAT;
        k_pack_weights<<<(total + 255) / 256, 256, 0, stream>>>((const __half*)net->w_plain[i], fan_out, fan_in, n_rows, img + off,
                                                                cat ? s.lf : 0, cat ? 3 + 6 * d->pe_bands : 0);
        nif_count_launch(1);
        off += i == 0 ? s.w1_bytes : (size_t)s.KC * n_rows * 128;
    }
    NIF_CUDA_TRY(cudaGetLastError());
    return NIF_OK;
}

int nif_launch_fused_tc(const nif_bvh* bvh, const nif_net* net, const nif_ray_batch* rays, const nif_query_out* out,
                        NifQueryScratch* scratch, const int32_t* hit_list, unsigned flags, cudaStream_t stream,
                        const NifPoseBatch* batch)
{
    if (rays->n == 0) return NIF_OK;
    const nif_net_desc* d = &net->desc;
    const TcShape s = tc_shape(d);
    TcParams p;
    p.enc = net->enc;
    p.hidden_layers = d->hidden_layers;
    p.n_chunks = s.n_chunks; p.es_per_chunk = s.epc; p.n_es = s.n_es;
    p.table = (const __half*)net->table;
    p.w_img = (const uint8_t*)net->w_tc; p.w_bytes = s.w_bytes; p.w1_bytes = s.w1_bytes;
    p.theta_max = bvh->theta_max; p.bend_k = bvh->bend_k;
    p.map = NifMapCtx{bvh->theta_max, bvh->bend_k, bvh->lattice, bvh->nv, bvh->local_inverse};
    p.batch = batch ? *batch : NifPoseBatch{nullptr, nullptr, 0};
    p.origin = rays->origin; p.dir = rays->dir;
    p.out = *out; p.scratch = scratch; p.tile_counter = &scratch->pad[4]; p.hit_list = hit_list; p.flags = flags;
    p.enc_mode = d->enc_mode;
    const TcW1Plan plan = tc_plan_w1(d->width, d->hidden_layers, s.n_chunks);
    p.w1_slots = plan.slots; p.w1_resident = plan.resident;
    const uint32_t smem = tc_smem_layout(d->width, d->hidden_layers, plan.slots).total;
    const int n_sm = nif_sm_count();
    if (n_sm <= 0) return NIF_ERR_CUDA;
    const long long max_tiles = (rays->n + TC_TILE - 1) / TC_TILE;
    const int blocks = (int)(max_tiles < n_sm ? max_tiles : n_sm);
    // the concatenation variant is its own instantiation so that the composition kernel's code is untouched
    // the MLP-only probe (NIF_PROBE_SKIP_GATHER) is its own instantiation of the composition kernel
#define NIF_TC_CASE(WW, FF) if (d->width == WW && d->feat == FF) { \
        if (flags & NIF_PROBE_SKIP_GATHER) \
            return d->enc_mode == NIF_ENC_CONCAT ? launch_tc<WW, FF, true, false, true>(p, smem, blocks, stream) \
                                                 : launch_tc<WW, FF, false, false, true>(p, smem, blocks, stream); \
        return d->enc_mode == NIF_ENC_CONCAT \
            ? (bvh->local_inverse ? launch_tc<WW, FF, true, true, false>(p, smem, blocks, stream) : launch_tc<WW, FF, true, false, false>(p, smem, blocks, stream)) \
            : (bvh->local_inverse ? launch_tc<WW, FF, false, true, false>(p, smem, blocks, stream) : launch_tc<WW, FF, false, false, false>(p, smem, blocks, stream)); }
    NIF_TC_CASE(32, 2); NIF_TC_CASE(64, 2); NIF_TC_CASE(128, 2);
    NIF_TC_CASE(32, 4); NIF_TC_CASE(64, 4); NIF_TC_CASE(128, 4);
#undef NIF_TC_CASE
    return NIF_ERR_UNSUPPORTED;
}
