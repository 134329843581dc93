// K2: E4M3 x E4M3 -> fp32 linear layers on the 5th-gen tensor cores (tcgen05.mma kind::f8f6f4,
// accumulators in TMEM, operands staged through shared memory by the TMA engine).
//
// Formulation ("swap-AB"): the WEIGHT matrix W[N][K] is the MMA's M-side operand (128 output
// channels per tile fill the 128 TMEM lanes) and the TOKENS X[M][K] are the MMA's N-side operand
// (TOK = 16..256 tokens per instruction, a run-time value).  Verify steps have few rows
// (M = B*T = 60..832) and many output channels: this keeps the tensor core full at any M, streams
// every weight byte once per token tile, and gives an epilogue in which the 32 lanes of a warp hold
// 32 consecutive output channels of one token, so global stores are coalesced without staging.
//
//   y[m][n] = (sum_k X[m][k] * W[n][k]) * s_x[m] * s_w[n]            (DESIGN.md R-accum)
//
// HBM layout of W (ours to choose: the library quantizes the weights): [N/128][K/128] tiles of
// 128 rows x 128 bytes, each tile 16 KiB CONTIGUOUS and already in the 128-byte-swizzled order the
// UMMA shared-memory descriptor expects.  One stage of weights is therefore one linear 16 KiB
// cp.async.bulk: full DRAM-page locality, no tensor-map walk (the row-major layout of v1 read 128
// scattered 128-byte rows per stage and reached 18-47 GB/s per SM; profiles/r1_launches_v1.md).
// X (activations, written row-major by the quantize kernels) comes through a 2-D tensor map.
//
// Persistent CTAs (grid = min(#SMs, work items)); a work item is (n_tile, m_tile, k_split), k_split
// fastest.  Warp roles (192 threads): warp 0 = TMA producer, warp 1 = TMEM owner + MMA issuer,
// warps 2..5 = epilogue.  Two TMEM accumulators alternate so the epilogue of item i overlaps the
// main loop of item i+1.  The epilogue of the layer GEMMs is deliberately trivial: raw fp32 accumulators
// go to out[split][m][n]; the kernel that consumes them (RMSNorm / RoPE / SwiGLU, each of which reads
// every element exactly once) sums the K-splits in split order and applies s_x[m] * s_w[n] (+ residual).
// That makes split-K free of any fix-up pass, fence or atomic, and deterministic (LinOut, ev_common.cuh).
// Only the LM head applies its scales here, because it reduces to an argmax in the epilogue.
// Canonical K cuts (batch invariance: verification must reproduce plain decoding bit for bit, so a token's
// result may not depend on how many other tokens share the launch).  Every layer matrix has ONE fixed set of K cuts,
// a function of its shape and of the model constant `cut_G` only: the K-blocks of the flattened (pair of 128-channel
// tiles, K-block) space are dealt out evenly to cut_G pieces, piece c = [floor(c U / G), floor((c+1) U / G)); each
// piece is accumulated from zero inside the tensor core and the pieces of a tile are added in K order with single
// rounded fp32 additions.  Few rows (one token tile): piece c IS the work of CTA pair c (stream-K), the pieces land
// in slabs the consumer adds (LinOut).  Many rows: a CTA pair owns whole (pair tile, token tile) items, switches the
// TMEM accumulator at the same cuts and its epilogue warps keep the running fp32 sum in registers - same additions,
// same order, one slab.  The LM head is never cut (1002 tiles).
// Programmatic dependent launch: barrier setup, TMEM allocation and the first STAGES weight tiles
// are issued BEFORE griddepcontrol.wait (weights do not depend on the previous kernel), so the
// weight stream of this GEMM starts while the previous (element-wise) kernel is still running.
#pragma once
#include "ev_common.cuh"

namespace ev {

enum GemmEpi { EPI_RAW = 0, EPI_ARGMAX = 2 };

constexpr int GEMM_THREADS = 192;        // warp 0 TMA, warp 1 MMA, 4 epilogue warps
constexpr int GEMM_THREADS_SUM = 320;    // the running-sum epilogue (CTA pairs, raw output): 8 epilogue warps
template <int EPI, bool PAIR> constexpr int gemm_threads() { return (PAIR && EPI == 0) ? GEMM_THREADS_SUM : GEMM_THREADS; }
constexpr int GEMM_BK = 128;          // bytes (= E4M3 elements) of K per stage: one swizzle row
constexpr int GEMM_WROWS = 128;       // output channels per tile = UMMA M
constexpr int GEMM_WTILE = GEMM_WROWS * GEMM_BK;  // 16 KiB
constexpr int GEMM_MAX_STAGES = 10;
constexpr int GEMM_SMEM_BUDGET = 200 * 1024;

struct GemmArgs {
    int M, N;
    int total_kb;       // ceil(K / 128) = K tiles of W
    int n_tiles, m_tiles, k_splits, kb_per_split;
    int sk_units;       // stream-K: U = tiles * total_kb K-blocks dealt out evenly (tile = n_tile * m_tiles + m_tile, or the
                        // same over PAIRS of n tiles with mc), CTA (pair) c gets [c U / G, (c+1) U / G); 0 = classic items
    int tok;            // tokens per tile (UMMA N), multiple of 16, <= 256
    int stages;
    const uint8_t* W;   // tiled + swizzled codes: [n_tiles][total_kb][16 KiB]
    const float* sx;    // [M]
    const float* sw;    // [N]
    float* out;         // EPI_RAW: [k_splits][M][ldo] raw accumulators; EPI_ARGMAX: optional logits [M][ldo]
    int ldo;
    unsigned long long* argmax_keys;  // EPI_ARGMAX: [M] packed (ordered logit, ~index)
    L2Prefetch pf;      // slice of the weight stream of the GEMMs that follow (ev_common.cuh)
    const void* warm[2];   // per-layer constants the CONSUMER kernel will read first thing after its wait (this
    int warm_bytes[2];     // matrix's s_w, the next RMSNorm's gain): touched here so they are L2 hits there
    int bal;            // balanced partition (several token tiles): the (n unit, 16-token block) space, n unit major, is dealt
                        // out evenly to the CTAs (CTA pairs); a CTA's contiguous range is cut at n-unit boundaries and into
                        // items of <= 256 tokens, so token tiles differ in size from item to item (GemmItem::tok) and no
                        // CTA idles in a partial last wave (896 tiles on 148 CTAs = 6.05 waves cost 7).  0 = uniform tiles
    int bal_blocks;     // 16-token blocks per n unit = ceil(M / 16)
    const CUtensorMap* tms;   // bal: activation tensor maps in global memory, box heights 8, 16, ..., 256 rows ([h / 8 - 1])
    int mc;             // 1 = work is indexed by PAIRS of CTAs (pair c = CTAs 2c, 2c+1; CTA rank r takes n tile 2 p + r of pair
                        // tile p).  The PAIR kernel (cluster of 2, tcgen05 cta_group::2) runs one 256-channel x tok MMA per pair,
                        // each CTA staging its own 128 channels of W and HALF of the token tile (see "CTA pairs" below); the
                        // single-CTA kernel uses the same indexing for stream-K so that both share the canonical K cuts
    int cut_G, cut_U;   // canonical K cuts for whole-tile items (PAIR kernel, raw output): pieces, K-block units; cut_U == 0 = none
};

// byte offset of element (row r, byte c) inside a 16 KiB weight tile (128-byte swizzle)
__host__ __device__ __forceinline__ int wtile_offset(int r, int c) {
    return r * 128 + ((((c >> 4) ^ (r & 7)) << 4) | (c & 15));
}

__device__ __forceinline__ uint32_t ordered_bits(float f) {
    const uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
            smem_u32(smem_dst)),
        "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void tmem_alloc_rt(uint32_t* smem_result, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(smem_result)), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_rt(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void epi_bar_sync() { asm volatile("bar.sync 1, 128;" ::: "memory"); }

__device__ __forceinline__ void bulk_load_plain(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// ---- CTA pairs (cta_group::2) ----
__device__ __forceinline__ void tmem_alloc_rt2(uint32_t* smem_result, uint32_t ncols) {   // one warp of EACH CTA of the pair
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(smem_result)), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_rt2(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
// D[tmem, 256 lanes over the pair] (+)= A[smem of both CTAs, 128 rows each] * B[smem of both CTAs, N/2 rows each]
__device__ __forceinline__ void umma_f8_2cta(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// all previously issued tcgen05.mma of this thread arrive on the mbarrier at this offset in BOTH CTAs of the pair
__device__ __forceinline__ void umma_commit_2cta(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(smem_u32(bar)),
                 "h"((uint16_t)3)
                 : "memory");
}
// arrive on the mbarrier at the same offset in CTA `rank` of the cluster
__device__ __forceinline__ void mbar_arrive_remote(uint64_t* bar, uint32_t rank) {
    // default (CTA-scope) semantics on purpose: the cluster-scope release / acquire forms compile to MEMBAR.ALL.GPU and
    // CCTL.IVALL around every arrive / wait (the pair ran at HALF the single-CTA speed with them).  What travels
    // through these barriers is ordered by the barriers' own completion: TMA-written shared memory read by the
    // tensor core, and tcgen05.ld -> tcgen05.fence::before_thread_sync -> arrive on the epilogue side.
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_map(bar, rank)) : "memory");
}
struct GemmItem { int n_tile, m_tile, split, tile, kb0, nkb, m0, tok; };   // m0, tok: first token row and token count of the item
__device__ __forceinline__ GemmItem gemm_item(const GemmArgs& a, int w) {
    GemmItem it;
    it.split = w % a.k_splits;
    it.tile = w / a.k_splits;
    it.m_tile = it.tile % a.m_tiles;
    it.n_tile = it.tile / a.m_tiles;
    it.kb0 = it.split * a.kb_per_split;
    it.nkb = min(a.kb_per_split, a.total_kb - it.kb0);
    it.m0 = it.m_tile * a.tok;
    it.tok = a.tok;
    return it;
}
// Work of one CTA, in order.  Classic: items blockIdx.x, +gridDim.x, ...  Stream-K: the contiguous range of
// K-blocks [c U / G, (c+1) U / G) of the flattened (n_tile, kb) space, cut at tile boundaries; the piece of a
// tile computed by the j-th CTA that touches it goes to slab j (sk_first_cta gives the first such CTA), so the
// consumer (LinOut) adds the pieces in K order: deterministic, and independent of M.
__host__ __device__ __forceinline__ int sk_first_cta(int unit, int G, int U) {  // largest c with floor(c U / G) <= unit
    return (int)(((long long)(unit + 1) * G + U - 1) / U) - 1;
}
struct GemmWork {
    int w, u, u_end;
    // c / G: this CTA's index and the CTA count, or - multicast pairs - the pair's index and the pair count
    __device__ __forceinline__ void init(const GemmArgs& a) {
        const int c = a.mc ? (int)(blockIdx.x >> 1) : (int)blockIdx.x, G = a.mc ? (int)(gridDim.x >> 1) : (int)gridDim.x;
        w = c;
        const long long U = a.bal ? (long long)(a.n_tiles / (a.mc ? 2 : 1)) * a.bal_blocks : a.sk_units;
        u = (int)((long long)c * U / G);
        u_end = (int)((long long)(c + 1) * U / G);
    }
    __device__ __forceinline__ bool next(const GemmArgs& a, GemmItem& it) {
        const int c = a.mc ? (int)(blockIdx.x >> 1) : (int)blockIdx.x, G = a.mc ? (int)(gridDim.x >> 1) : (int)gridDim.x;
        const int rank = a.mc ? (int)(blockIdx.x & 1) : 0, nmul = a.mc ? 2 : 1;   // pairs: tile = (pair of n tiles, m tile)
        if (a.bal) {   // u, u_end: 16-token blocks of the flattened (n unit, block) space
            if (u >= u_end) return false;
            const int p = u / a.bal_blocks, b0 = u - p * a.bal_blocks;
            const int len = min(u_end, (p + 1) * a.bal_blocks) - u;    // what is left of this CTA's piece of n unit p
            const int n_items = (len + 15) >> 4;                        // items of <= 16 blocks, as even as possible
            const int chunk = (len + n_items - 1) / n_items;
            it.tile = p; it.m_tile = 0; it.split = 0;
            it.n_tile = nmul * p + rank;
            it.kb0 = 0; it.nkb = a.total_kb;
            it.m0 = b0 * 16; it.tok = chunk * 16;
            u += chunk;
            return true;
        }
        if (a.sk_units) {
            if (u >= u_end) return false;
            it.tile = u / a.total_kb;
            it.m_tile = it.tile % a.m_tiles;
            it.n_tile = nmul * (it.tile / a.m_tiles) + rank;
            it.kb0 = u - it.tile * a.total_kb;
            it.nkb = min(a.total_kb - it.kb0, u_end - u);
            it.split = c - sk_first_cta(it.tile * a.total_kb, G, a.sk_units);
            it.m0 = it.m_tile * a.tok; it.tok = a.tok;
            u += it.nkb;
            return true;
        }
        if (a.mc) {  // pair item = (pair of adjacent n tiles, m tile), m fastest; this CTA takes n tile 2 * pair + rank
            if (w >= (a.n_tiles >> 1) * a.m_tiles) return false;
            it.split = 0;
            it.tile = w;
            it.m_tile = w % a.m_tiles;
            it.n_tile = 2 * (w / a.m_tiles) + rank;
            it.kb0 = 0;
            it.nkb = a.total_kb;
            it.m0 = it.m_tile * a.tok; it.tok = a.tok;
            w += G;
            return true;
        }
        if (w >= a.n_tiles * a.m_tiles * a.k_splits) return false;
        it = gemm_item(a, w);
        w += G;
        return true;
    }
    // K-blocks this CTA (pair) processes in total
    __device__ __forceinline__ long total_kb_iters(const GemmArgs& a) const {
        const int c = a.mc ? (int)(blockIdx.x >> 1) : (int)blockIdx.x, G = a.mc ? (int)(gridDim.x >> 1) : (int)gridDim.x;
        if (a.sk_units) return (long)((long long)(c + 1) * a.sk_units / G - (long long)c * a.sk_units / G);
        const int items = (a.mc ? (a.n_tiles >> 1) : a.n_tiles) * a.m_tiles * a.k_splits;
        return c < items ? (long)((items - c + G - 1) / G) * a.kb_per_split : 0;
    }
};

// chunk ends of a whole-tile item under the canonical K cuts: the K-blocks [kb, *end) of pair tile p that belong to piece cc
__device__ __forceinline__ int cut_end(const GemmArgs& a, int p, int cc) {
    return min(a.total_kb, (int)((long long)(cc + 1) * a.cut_U / a.cut_G) - p * a.total_kb);
}

// PAIR: the kernel contains cta_group::2 instructions and must be launched in clusters of 2 (a.mc == 1)
template <int EPI, bool PAIR>
__global__ void __launch_bounds__((gemm_threads<EPI, PAIR>()), 1) gemm_e4m3_kernel(const __grid_constant__ CUtensorMap tmX, const __grid_constant__ CUtensorMap tmXh, GemmArgs a) {
    constexpr bool SUM = PAIR && EPI == EPI_RAW;   // running-sum epilogue: 8 epilogue warps, canonical K cuts inside an item
    constexpr int EPI_WARPS = SUM ? 8 : 4;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    // CTA pairs (many token rows; PAIR): the pair runs ONE tcgen05.mma.cta_group::2 of 256 channels x tok tokens per
    // K step.  Each CTA stages its own 128 channels of W and HALF of the token tile; the tensor cores read both
    // halves across the pair.  Per K-block a CTA then receives 16 KiB + tok/2 x 128 B instead of 16 KiB + tok x 128 B:
    // a third less L2 -> SM traffic per flop and 6 instead of 4 stages in flight at tok = 208, which is what bounded
    // the single-CTA form (tensor pipe 61 % busy; multicasting the token tile to both CTAs changed nothing, because
    // every CTA still had to RECEIVE the whole tile).  Rank 0 issues the MMAs and commits to both CTAs' barriers;
    // rank 1's MMA warp only relays "my stage has landed" to rank 0; each CTA's epilogue drains its own 128 lanes.
    const int rank = PAIR ? (int)(blockIdx.x & 1) : 0;
    const int x_rows = PAIR ? a.tok / 2 : a.tok;
    const int x_bytes = x_rows * GEMM_BK;
    const int stage_bytes = GEMM_WTILE + x_bytes;
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + a.stages * stage_bytes);
    uint64_t* empty_bar = full_bar + GEMM_MAX_STAGES;
    uint64_t* peer_full_bar = empty_bar + GEMM_MAX_STAGES;    // rank 0: rank 1's stage has landed
    uint64_t* tmem_full_bar = peer_full_bar + GEMM_MAX_STAGES;   // [2]
    uint64_t* tmem_empty_bar = tmem_full_bar + 2;            // [2]
    uint32_t* tmem_base_smem = reinterpret_cast<uint32_t*>(tmem_empty_bar + 2);
    float* sx_smem = reinterpret_cast<float*>(tmem_base_smem + 4);  // [2][256] per-token scales of the current / next item
    unsigned long long* keys_smem = reinterpret_cast<unsigned long long*>(sx_smem + 512);  // [4 warps][256] argmax keys

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    pdl_launch_dependents();  // the consumer kernel's CTAs may become resident (they block in griddepcontrol.wait)
    l2_prefetch_issue(a.pf, 64);  // warp 2 (an epilogue warp, idle until the first accumulator is ready)
    if (warp >= 2) {  // epilogue warps are idle until the first accumulator is ready: one 128-byte line per thread
#pragma unroll
        for (int s = 0; s < 2; ++s)
            for (int ln = blockIdx.x * (32 * EPI_WARPS) + (int)threadIdx.x - 64; ln * 128 < a.warm_bytes[s]; ln += gridDim.x * (32 * EPI_WARPS)) {
                unsigned tmp;
                asm volatile("ld.global.cg.u32 %0, [%1];" : "=r"(tmp) : "l"(reinterpret_cast<const char*>(a.warm[s]) + (size_t)ln * 128));
            }
    }
    uint32_t tmem_cols = 32;
    while ((int)tmem_cols < 2 * a.tok) tmem_cols <<= 1;

    // ---- prologue.  The producer thread initialises the barriers and immediately starts the weight stream of
    // its first work item (weights do not depend on the previous kernel: this runs before griddepcontrol.wait,
    // i.e. while the previous kernel is still executing when launched with programmatic serialization). ----
    int pre = 0;
    GemmItem it0;
    {
        GemmWork w0;
        w0.init(a);
        if (!w0.next(a, it0)) { it0.n_tile = it0.m_tile = it0.kb0 = it0.nkb = it0.m0 = 0; it0.tok = a.tok; }
    }
    if (warp == 0 && lane == 0) {
        for (int s = 0; s < a.stages; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); mbar_init(&peer_full_bar[s], 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(&tmem_full_bar[i], 1); mbar_init(&tmem_empty_bar[i], (PAIR ? 2 : 1) * EPI_WARPS); }
        fence_barrier_init();
        pre = min(a.stages, it0.nkb);
        const uint8_t* wsrc = a.W + ((size_t)it0.n_tile * a.total_kb + it0.kb0) * GEMM_WTILE;
        const uint32_t tx0 = GEMM_WTILE + (PAIR ? it0.tok / 2 : it0.tok) * GEMM_BK;   // W tile + this CTA's token rows of the item
        for (int i = 0; i < pre; ++i) {
            mbar_arrive_expect_tx(&full_bar[i], tx0);
            bulk_load_plain(smem + i * stage_bytes, wsrc + (size_t)i * GEMM_WTILE, GEMM_WTILE, &full_bar[i]);
        }
        tma_prefetch_desc(&tmX);
    }
    if (warp == 1) { if (PAIR) tmem_alloc_rt2(tmem_base_smem, tmem_cols); else tmem_alloc_rt(tmem_base_smem, tmem_cols); }
    tc_fence_before();
    __syncthreads();
    if (PAIR) cluster_barrier();   // the peer's barriers exist before any commit or relayed arrive targets them
    tc_fence_after();
    const uint32_t tmem_base = *tmem_base_smem;
    const bool cuts = SUM && a.cut_U > 0;

    if (warp == 0) {
        if (lane == 0) {  // ===== producer: weights by linear bulk copy, activations by 2-D TMA =====
            const uint64_t pol_w = policy_evict_first();   // weights are streamed once per step
            const uint64_t pol_x = policy_evict_last();    // activations are re-read by every tile
            pdl_wait();  // activations come from the previous kernel
            trace_past_wait(a.pf);
            // pairs: this CTA fetches only its half of the item's token rows (rows rank * tok / 2 ...), into its own stage
            auto ld_x = [&](uint8_t* st, uint64_t* bar, int kb_abs, const GemmItem& item) {
                const int rows = PAIR ? item.tok / 2 : item.tok;
                const CUtensorMap* tm = a.bal ? a.tms + (rows / 8 - 1) : (PAIR ? &tmXh : &tmX);
                tma_load_2d_hint(st + GEMM_WTILE, tm, bar, kb_abs * GEMM_BK, item.m0 + rank * rows, pol_x);
            };
            for (int i = 0; i < pre; ++i) ld_x(smem + i * stage_bytes, &full_bar[i], it0.kb0 + i, it0);
#ifdef EV_GEMM_PROBE   // bring-up (-DEV_GEMM_PROBE): phase marks of the step trace (profiles/r2_step_timeline.md), last CTA each
            trace_phase_any(a.pf, 0);   // activations of the prefilled stages requested
#endif
            int s = pre;
            uint32_t ph = 0;
            if (s == a.stages) { s = 0; ph ^= 1; }
            GemmWork wk;
            wk.init(a);
            GemmItem it;
            for (bool first = true; wk.next(a, it); first = false) {
                const uint32_t tx = GEMM_WTILE + (PAIR ? it.tok / 2 : it.tok) * GEMM_BK;
                for (int kb = (first ? pre : 0); kb < it.nkb; ++kb) {
                    mbar_wait(&empty_bar[s], ph ^ 1);
                    mbar_arrive_expect_tx(&full_bar[s], tx);
                    uint8_t* st = smem + s * stage_bytes;
                    bulk_load(st, a.W + ((size_t)it.n_tile * a.total_kb + it.kb0 + kb) * GEMM_WTILE, GEMM_WTILE, &full_bar[s], pol_w);
                    ld_x(st, &full_bar[s], it.kb0 + kb, it);
                    if (++s == a.stages) { s = 0; ph ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        {   // ===== MMA issuer.  The WHOLE warp runs the loop and one elected lane issues: addresses and descriptors are
            // then provably warp-uniform and stay in uniform registers.  Under `if (lane == 0)` the compiler wrapped
            // every tcgen05.mma and commit in an ELECT / R2UR.BROADCAST / BRA.U.ANY loop (~100 cycles each, five per
            // K-block: more than the 416 cycles of tensor work of a 208-token K-block). =====
            const bool leader = elect_one();
            const uint32_t smem_base = smem_u32(smem);
            int s = 0;
            uint32_t ph = 0;
            GemmWork wk;
            wk.init(a);
            GemmItem it;
            if (rank == 1) {
                // pair, rank 1: no MMAs here; tell rank 0 when a stage of THIS CTA has landed
                while (wk.next(a, it)) {
                    for (int kb = 0; kb < it.nkb; ++kb) {
                        mbar_wait(&full_bar[s], ph);
                        if (leader) mbar_arrive_remote(&peer_full_bar[s], 0);
                        __syncwarp();
                        if (++s == a.stages) { s = 0; ph ^= 1; }
                    }
                }
            } else {
                int n_acc = 0;   // accumulators handed to the epilogue so far (one per item, or one per K piece of an item)
                while (wk.next(a, it)) {
                    const uint32_t idesc = umma_idesc_e4m3(PAIR ? 2 * GEMM_WROWS : GEMM_WROWS, it.tok);
                    const int p = it.n_tile >> 1;
                    int cc = cuts ? sk_first_cta(p * a.total_kb, a.cut_G, a.cut_U) : 0;
                    for (int kb = 0; kb < it.nkb; ++cc, ++n_acc) {
                        const int kb_end = cuts ? cut_end(a, p, cc) : it.nkb;
                        const int buf = n_acc & 1;
                        mbar_wait(&tmem_empty_bar[buf], ((n_acc >> 1) & 1) ^ 1);   // the epilogue (of both CTAs of a pair) has drained this accumulator
                        tc_fence_after();
                        const uint32_t d_tmem = tmem_base + (uint32_t)(buf * a.tok);
                        for (const int kb0 = kb; kb < kb_end; ++kb) {
                            mbar_wait(&full_bar[s], ph);
                            if (PAIR) mbar_wait(&peer_full_bar[s], ph);
                            tc_fence_after();
#ifdef EV_GEMM_PROBE
                            if (leader && n_acc == 0 && kb == kb0) trace_phase_any(a.pf, 1);          // first stage complete
                            if (leader && n_acc == 0 && kb == kb_end - 1) trace_phase_any(a.pf, 2);   // last stage of the first accumulator complete
#endif
                            const uint32_t wa = smem_base + (uint32_t)(s * stage_bytes);
                            const uint64_t adesc = umma_desc_k128(wa);
                            const uint64_t bdesc = umma_desc_k128(wa + GEMM_WTILE);
                            if (leader) {
                                if (PAIR) {
#pragma unroll
                                    for (int k = 0; k < GEMM_BK / 32; ++k)
                                        umma_f8_2cta(d_tmem, adesc + 2 * k, bdesc + 2 * k, idesc, ((kb - kb0) | k) != 0);
                                    umma_commit_2cta(&empty_bar[s]);
                                } else {
#pragma unroll
                                    for (int k = 0; k < GEMM_BK / 32; ++k)  // UMMA K = 32 E4M3 elements = 2 x 16 B
                                        umma_f8(d_tmem, adesc + 2 * k, bdesc + 2 * k, idesc, ((kb - kb0) | k) != 0);
                                    umma_commit(&empty_bar[s]);
                                }
                            }
                            __syncwarp();
                            if (++s == a.stages) { s = 0; ph ^= 1; }
                        }
                        if (leader) { if (PAIR) umma_commit_2cta(&tmem_full_bar[buf]); else umma_commit(&tmem_full_bar[buf]); }
                        __syncwarp();
                    }
                }
            }
        }
    } else if (SUM) {
        // ===== running-sum epilogue (CTA pairs, raw output): warps 2..9; warp w may touch TMEM lanes 32*(w%4) .. +31 and
        // takes one half of the item's token columns.  Every K piece of the item arrives as a fresh accumulator; the
        // pieces are added in K order with single rounded fp32 additions - the additions the consumer of the stream-K
        // slabs performs (lin_acc, ev_common.cuh) - and the item's sum is stored once. =====
        pdl_wait();
        const int q = warp & 3, half = (warp - 2) >> 2;
        const int n_loc = q * 32 + lane;
        int n_acc = 0;
        GemmWork wk;
        wk.init(a);
        GemmItem it;
        while (wk.next(a, it)) {
            const int n = it.n_tile * GEMM_WROWS + n_loc;
            const int ch = ((it.tok + 31) >> 5) << 4;            // columns per half, multiple of 16, <= 128
            const int c_lo = half * ch;
            const int ncols = max(0, min(it.tok, c_lo + ch) - c_lo);
            const int p = it.n_tile >> 1;
            int cc = cuts ? sk_first_cta(p * a.total_kb, a.cut_G, a.cut_U) : 0;
            float acc[128];
            bool first = true;
            for (int kb = 0; kb < it.nkb; ++cc, ++n_acc, first = false) {
                kb = cuts ? cut_end(a, p, cc) : it.nkb;
                const int buf = n_acc & 1;
                mbar_wait(&tmem_full_bar[buf], (n_acc >> 1) & 1);
                tc_fence_after();
                const uint32_t t_addr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * a.tok + c_lo);
#pragma unroll
                for (int g = 0; g < 4; ++g) {   // 32 columns per batch of loads
                    uint32_t v[32];
#pragma unroll
                    for (int u = 0; u < 2; ++u)
                        if (g * 32 + u * 16 < ncols) tmem_ld16(t_addr + (uint32_t)(g * 32 + u * 16), v + u * 16);
                    tmem_ld_wait();
                    if (g == 3) {  // accumulator fully read: hand it back to the MMA warp
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) { if (rank == 0) mbar_arrive(&tmem_empty_bar[buf]); else mbar_arrive_remote(&tmem_empty_bar[buf], 0); }
                    }
#pragma unroll
                    for (int j = 0; j < 32; ++j)
                        if (g * 32 + (j & ~15) < ncols) acc[g * 32 + j] = first ? __uint_as_float(v[j]) : __fadd_rn(acc[g * 32 + j], __uint_as_float(v[j]));
                }
            }
            if (n < a.N) {
                float* outp = a.out + (size_t)(it.m0 + c_lo) * a.ldo + n;
#pragma unroll
                for (int j = 0; j < 128; ++j)
                    if (j < ncols && it.m0 + c_lo + j < a.M) outp[(size_t)j * a.ldo] = acc[j];
            }
        }
    } else {  // ===== epilogue: warps 2..5; warp w may touch TMEM lanes 32*(w%4) .. +31 =====
        pdl_wait();
        const int q = warp & 3;
        const int et = (int)threadIdx.x - 64;  // 0..127 among the epilogue threads
        const int n_loc = q * 32 + lane;
        int n_it = 0;
        GemmWork wk;
        wk.init(a);
        GemmItem it;
        for (; wk.next(a, it); ++n_it) {
            const int buf = n_it & 1;
            const int n = it.n_tile * GEMM_WROWS + n_loc;
            const int m0 = it.m0, tok = it.tok;
            const bool n_ok = n < a.N;
            constexpr int GC = 32;                    // columns (tokens) handled per register group
            const int n_groups = (tok + GC - 1) / GC;
            float swn = 0.f;
            float* sxs = sx_smem + buf * 256;
            if (EPI == EPI_ARGMAX) {  // scales are fetched BEFORE waiting for the MMAs
                swn = n_ok ? __ldg(a.sw + n) : 0.f;
                for (int i = et; i < tok; i += 128) sxs[i] = (m0 + i < a.M) ? __ldg(a.sx + m0 + i) : 0.f;
                epi_bar_sync();
            }
            mbar_wait(&tmem_full_bar[buf], (n_it >> 1) & 1);
            tc_fence_after();
#ifdef EV_GEMM_PROBE
            if (et == 0 && n_it == 0) trace_phase_any(a.pf, 3);   // the epilogue holds the first accumulator
#endif
            const uint32_t t_addr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * a.tok);
            float* outp = a.out + (size_t)it.split * a.M * a.ldo;
            for (int g = 0; g < n_groups; ++g) {
                uint32_t v[GC];
                tmem_ld16(t_addr + (uint32_t)(g * GC), v);
                if (g * GC + 16 < tok) tmem_ld16(t_addr + (uint32_t)(g * GC + 16), v + 16);
                tmem_ld_wait();
                if (g == n_groups - 1) {  // accumulator fully read: hand it back to the MMA warp
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) { if (rank == 0) mbar_arrive(&tmem_empty_bar[buf]); else mbar_arrive_remote(&tmem_empty_bar[buf], 0); }
                }
                if (EPI == EPI_ARGMAX) {
                    // per token: max over the tile's 128 channels of (ordered logit, ~index).  Two warp-wide integer
                    // reductions per token (redux.sync: max of the ordered logit bits, then min of the channel index
                    // among the lanes that hold that maximum = lowest id on ties) instead of a 5-round shuffle tree
                    // on 64-bit keys (the shuffle tree made the LM head's epilogue, not its MMAs, the bound at M = 832);
                    // lane j keeps token j's key, then the 4 warps meet in shared memory and ONE atomicMax per
                    // (token, tile) goes to global memory
                    uint32_t kmx = 0u, kmn = 0xFFFFFFFFu;
#pragma unroll
                    for (int j = 0; j < GC; ++j) {
                        const int col = g * GC + j;
                        const int m = m0 + col;
                        const float y = mul_rn(mul_rn(__uint_as_float(v[j]), sxs[col < tok ? col : 0]), swn);
                        const bool ok = n_ok && col < tok && m < a.M;
                        const uint32_t ob = ok ? ordered_bits(y) : 0u;      // ordered_bits of a non-NaN value is never 0
                        const uint32_t mx = __reduce_max_sync(0xffffffffu, ob);
                        const uint32_t mn = __reduce_min_sync(0xffffffffu, (ok && ob == mx) ? (uint32_t)n : 0xFFFFFFFFu);
                        if (lane == j) { kmx = mx; kmn = mn; }
                        if (ok && a.out) __stcs(a.out + (size_t)m * a.ldo + n, y);
                    }
                    if (g * GC + lane < tok)   // no valid lane: (0, ~0xFFFFFFFF) = key 0, below every real key
                        keys_smem[q * 256 + g * GC + lane] = ((unsigned long long)kmx << 32) | (0xFFFFFFFFu - kmn);
                } else {
#pragma unroll
                    for (int j = 0; j < GC; ++j) {
                        const int col = g * GC + j;
                        const int m = m0 + col;
                        if (n_ok && col < tok && m < a.M) outp[(size_t)m * a.ldo + n] = __uint_as_float(v[j]);
                    }
                }
            }
            if (EPI == EPI_ARGMAX) {
                epi_bar_sync();
                for (int col = et; col < tok; col += 128) {
                    const int m = m0 + col;
                    if (m < a.M) {
                        unsigned long long k0 = keys_smem[col], k1 = keys_smem[256 + col], k2 = keys_smem[512 + col], k3 = keys_smem[768 + col];
                        k0 = k1 > k0 ? k1 : k0; k2 = k3 > k2 ? k3 : k2; k0 = k2 > k0 ? k2 : k0;
                        atomicMax(a.argmax_keys + m, k0);
                    }
                }
                epi_bar_sync();  // keys_smem is rewritten by the next item
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (PAIR) cluster_barrier();   // no CTA of the pair exits (or frees its TMEM) while the pair's MMAs or arrives may still target it
    if (warp == 1) { if (PAIR) tmem_dealloc_rt2(tmem_base, tmem_cols); else tmem_dealloc_rt(tmem_base, tmem_cols); }
    trace_exit(a.pf);
}

// tiled+swizzled codes -> row-major [rows][cols] (ev_model_get_quantized)
__global__ void __launch_bounds__(256) untile_weight_kernel(const uint8_t* __restrict__ Wt, int total_kb, long row_off, long rows,
                                                            long cols, uint8_t* __restrict__ out) {
    const long r = blockIdx.x;
    const long n = row_off + r;
    for (long k = threadIdx.x; k < cols; k += 256)
        out[r * cols + k] = Wt[((size_t)(n >> 7) * total_kb + (k >> 7)) * GEMM_WTILE + wtile_offset((int)(n & 127), (int)(k & 127))];
}

}  // namespace ev
