// K5 (tcgen05 version): tree-masked GQA attention over the paged bf16 KV cache on the 5th-gen tensor
// cores ("tree attention"; BASELINE.json:north_star (2)).  Same decomposition and outputs
// as tree_attn_partial_kernel (ev_attention.cuh): one CTA = (sequence, kv head, 128-row tile, key split);
// rows = tree nodes x GQA group; partial (O, max, sum) per split, merged by attn_merge_quant_kernel.
//
// Data flow per 64-key tile j (a CTA walks its key range tile by tile):
//   TMA warp      : 4 pages x {K,V} boxes, each a whole (page, K|V, head) block of 16 tokens x D -> 128-byte-swizzled
//                   smem as [page][8-token group][d half][8 x 128 B] (read in place through one 4-D tensor map)
//   MMA thread    : S[j&1]  = Q . K_j^T   (tcgen05.mma kind::f16, A = Q from TMEM, B = K tile, D in TMEM)
//                   Oc      = P[j&1] . V_j (A = P from TMEM, B = V tile MN-major, D in TMEM, from zero)
//   8 softmax warps (thread = one query row x half of the tile's keys):
//                   S -> registers (tcgen05.ld), tree mask, online max (the two halves of a row meet in shared
//                   memory behind a 64-thread named barrier), p = 2^(s k - m k), k = log2(e)/sqrt(d), one FFMA +
//                   one MUFU per key, P -> hi|lo fp16 -> TMEM (tcgen05.st); publishes the tile's rescale
//                   factor c = exp(m_old - m_new) in shared memory
//   8 correction warps (thread = one query row x half of d): Oc -> registers and
//                   O = O * c + Oc with ONE rounded fp32 operation per tile, concurrently with the softmax of
//                   the next tile (the two used to be serial in the same threads: 3,700 cycles per tile against
//                   a tensor floor of 1,536; profiles/r1_attention_v2.md).
// Precision (DESIGN.md section 6 "attention precision"): Q and P are fp32 values split into hi+lo fp16 parts
// (2 x 11 significand bits: x = hi + lo to 2^-22 relative, the size of one fp32 rounding of the sum), K and V
// are bf16 VALUES in binary16 containers (ev_common.cuh "KV pool containers"): kind::f16 wants A and B in the same
// format (fp16 A with bf16 B is an illegal instruction on sm_100a; converting the tiles in shared memory inside
// this kernel made the converting warps the bottleneck), so rope_kvwrite_kernel and the import path store them
// that way.  Every product is then exact (11 + 8 bits) and the tensor core only accumulates (small parts first).  Both are
// scaled by a power of two before the split so that the lo parts stay out of fp16's subnormals: Q by 2^6 (undone
// exactly in the 1/sqrt(d) multiply), P by 2^15 (p <= 1; the row sum and the running output carry the factor and
// drop it, exactly, when the partial is written).  The first version used three bf16 parts (exact, 3x the
// tensor work): the tensor pipe bounded the kernel at batch 32.  The running output lives in registers, not in
// TMEM, because long tensor-core accumulation chains truncate.
#pragma once
#include <cuda_fp16.h>
#include "ev_common.cuh"
#include "ev_attention.cuh"

namespace ev {

constexpr int TCA_THREADS = 576;  // warp 0 TMA producer, warp 1 MMA issuer, warps 2..9 softmax, warps 10..17 correction
constexpr int TCA_BN = 64;        // keys per tile (= ATT_CH: the split plan is shared with the legacy kernel)
constexpr int TCA_KS = 6;        // K ring depth (a K tile is released by Q.K^T, early)
constexpr int TCA_VS = 5;        // V ring depth (a V tile is released by P.V)
constexpr int TCA_PAGE = 16;      // tokens per page this kernel is built for

// FP8 = the pool holds E4M3 codes (ev_config.kv_dtype 1; "quantizing the KV cache to FP8 halves the storage"):
// raw 2-KiB page blocks arrive by linear bulk copies into raw rings, two extra warps (18: K, 19: V) turn each 64-key tile
// into the fp16, 128-byte-swizzled tile the MMAs read (E4M3 -> fp16 is exact; the static per-tensor scales are applied in
// fp32: K's in the score multiply, V's when the chunk's partial output is written), everything downstream is unchanged.
// SMALL = launches whose CTAs walk at most 8 key tiles (batch 1: 256-key chunks): rings of 3 + 3 tiles instead of 6 + 5.
// The arithmetic is the same; what changes is how much of the SM's 228 KiB is left as L1: the unified carve-out follows the
// dynamic shared memory a kernel asks for, and with 223 KiB asked for, the 64-KiB Q tile and the partial outputs went through
// ~5 KiB of L1 (a handful of lines in flight: 4,000 - 6,000 cycles each at batch 1; profiles/r2_attention_issue.md section 5).
template <int D, bool FP8 = false, bool SMALL = false>
struct TcaCfg {
    static constexpr int KS = FP8 ? 4 : (SMALL ? 3 : TCA_KS);          // fp16 K tiles in flight
    static constexpr int VS = FP8 ? 4 : (SMALL ? 3 : TCA_VS);          // fp16 V tiles in flight
    static constexpr int RS = FP8 ? 4 : 0;               // raw E4M3 tiles in flight, per K and per V
    static constexpr int RAW_BYTES = TCA_BN * D;         // one raw tile: 64 keys x D bytes
    // bf16 pool: Q.K^T and P.V have separate issuing warps (1 and 18).  FP8 pool: one issuer (warp 1) - a 21st warp would put six
    // warps on one scheduler (80 registers per thread, 216 B of spills) and the converter warps set the pace there anyway.
    static constexpr bool TWO_ISSUERS = !FP8;
    static constexpr int PV_WARP = FP8 ? -1 : 18;
    static constexpr int THREADS = FP8 ? TCA_THREADS + 64 : TCA_THREADS + 32;
    static constexpr int NH = D / 64;                    // 128-byte (64-element) halves of a head row
    static constexpr int Q_PART = NH * 128 * 128;        // bytes of one bf16 part of the 128 x D query tile
    static constexpr int Q_BYTES = 2 * Q_PART;
    static constexpr int KV_HALF = TCA_BN * 128;         // 8 KiB: 64 keys x 128 B
    static constexpr int K_BYTES = NH * KV_HALF;
    static constexpr int SBO = NH * 1024;               // 8-token groups of one d half: [page][group][half][1 KiB]
    static constexpr int PAGE_BYTES = 2 * SBO;          // one 16-token (page, K|V, head) block
    static constexpr int BAR_BYTES = 512;
    static constexpr int XCH_BYTES = (2 * 2 * 128 + 2 * 128 + 8 * 128) * 4;  // max exchange (double buffered) + sum exchange + rescale factors (8 tiles deep)
    // a chunk's partial output leaves through shared memory: a correction thread holds one ROW (TMEM lane), so its own stores hit
    // 32 different lines per instruction (5,000 cycles per chunk at batch 1: profiles/r2_attention_issue.md section 5); staged
    // OPW columns at a time in a [32 rows][OSTR] tile per warp, a store instruction writes whole rows (128-bit accesses: few instructions,
    // the chunk's end is a single warp's serial instruction stream)
    static constexpr int OPW = FP8 ? 16 : 32;
    // the same region stages the Q tile on its way in (bf16 pool variant): 16 warps x [32 rows][D/8 + 1] words per fp16 part
    static constexpr int QST_BYTES = FP8 ? 0 : 16 * 32 * (D / 8 + 1) * 4;
    static constexpr int OSTR = OPW + 4;     // floats between rows of the staging tile: 16-byte aligned rows, conflict-free 128-bit accesses
    static constexpr int OST_BYTES = (8 * 32 * OSTR * 4 > QST_BYTES) ? 8 * 32 * OSTR * 4 : QST_BYTES;
    static constexpr int SMEM = 1024 + (KS + VS) * K_BYTES + 2 * RS * RAW_BYTES + BAR_BYTES + XCH_BYTES + OST_BYTES;   // Q lives in TMEM
    // TMEM columns
    // S[2] and P[2] share two 64-column regions: S(j) = 64 fp32 columns, P(j) = 2 parts x 32 columns (64 fp16
    // pairs) written over it once both halves of the row have read S(j) (the pair barrier orders that).  (Three
    // regions with Q.K^T two tiles ahead measured the same: the tensor pipe, not the S hand-off, set the period.)
    // TWO O chunks, so P.V of tile j+1 does not wait for the correction warps to read chunk j.  The Q tile (hi | lo
    // fp16 parts, D/2 columns of pairs each) sits in TMEM too and is the A operand of Q.K^T straight from there:
    // from shared memory every N = 64 MMA read 4 KiB of Q + 2 KiB of K, 48 cycles against 32 of math.
    static constexpr int NSP = 2;
    static constexpr int NO = 2;            // O chunks in TMEM
    static constexpr int TS = 0;
    static constexpr int TP = 0;
    static constexpr int SP = 64;           // columns per S/P region
    static constexpr int TO = NSP * SP;     // O chunks: 2 x D fp32 columns
    static constexpr int TQ = TO + NO * D;  // Q: 2 parts x D/2 columns
    static_assert(TQ + D <= 512, "TMEM budget");
    static constexpr int DH = D / 2;        // output columns per softmax warpgroup
};

__device__ __forceinline__ void umma_bf16_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void umma_bf16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem),
        "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// instruction descriptor, kind::f16: D fp32 (bit 4), A format bits 7..9 = B format bits 10..12 = fp16 (0),
// A K-major, B K-major (0) or MN-major (1)
__host__ __device__ constexpr uint32_t umma_idesc_f16(int M, int N, int b_mn_major) {
    return (1u << 4) | ((uint32_t)b_mn_major << 16) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
// MN-major operand tile, 128-byte swizzle: 64 contiguous elements along MN per 128-byte row, rows = K index,
// 8-row groups SBO apart, next 64 elements along MN LBO apart
__device__ __forceinline__ uint64_t umma_desc_mn128(uint32_t smem_addr, uint32_t lbo, uint32_t sbo) {
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);
    d |= (uint64_t)((lbo >> 4) & 0x3FFFu) << 16;
    d |= (uint64_t)((sbo >> 4) & 0x3FFFu) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t* v) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
          "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
          "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* v) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
        "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
        "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
        : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t* v) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]),
                 "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7])
                 : "memory");
}
__device__ __forceinline__ void pair_bar_sync(int id) { asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory"); }
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void softmax_bar_sync() { asm volatile("bar.sync 1, 256;" ::: "memory"); }
__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// (x0, x1) -> packed fp16 pairs hi, lo with x = hi + lo up to 2^-22 |x| (x0 in the low half): hi = RN16(x),
// lo = RN16(x - hi); x - hi is exact in fp32.  |x| must stay below 65504 (the callers scale: see the header).
__device__ __forceinline__ void split2_pack(float x0, float x1, uint32_t& hi, uint32_t& lo) {
    const __half2 h = __floats2half2_rn(x0, x1);
    const float2 hf = __half22float2(h);
    const __half2 l = __floats2half2_rn(x0 - hf.x, x1 - hf.y);
    hi = *reinterpret_cast<const uint32_t*>(&h);
    lo = *reinterpret_cast<const uint32_t*>(&l);
}
constexpr float TCA_QSCALE = 64.f;        // 2^6
constexpr float TCA_PSCALE_LOG2 = 15.f;   // P is scaled by 2^15

struct TcAttnArgs {
    AttnArgs a;       // same fields as tree_attn_partial_kernel (pool pointer unused here)
    int row0;         // first row of this layer in the pool tensor map: layer * n_pages * 2 * Hkv * 16
    const uint8_t* pool8;   // FP8: the whole pool as bytes (row r of D codes at pool8 + r * D)
    float k_scale, v_scale; // FP8: this layer's static K / V cache scales (1 otherwise)
    L2Prefetch pf;
};
__device__ __forceinline__ void bulk_load_1d(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// 16 E4M3 codes (one 16-byte chunk) -> 16 fp16 values (two 16-byte chunks); exact
__device__ __forceinline__ void e4m3x16_to_f16(const uint4& in, uint4& lo, uint4& hi) {
    auto cv = [](uint32_t w, uint32_t& a, uint32_t& b) {
        asm("{\n\t.reg .b16 l, h;\n\tmov.b32 {l, h}, %2;\n\tcvt.rn.f16x2.e4m3x2 %0, l;\n\tcvt.rn.f16x2.e4m3x2 %1, h;\n\t}" : "=r"(a), "=r"(b) : "r"(w));
    };
    cv(in.x, lo.x, lo.y); cv(in.y, lo.z, lo.w); cv(in.z, hi.x, hi.y); cv(in.w, hi.z, hi.w);
}

// Bring-up probe (-DEV_ATTN_PROBE, never in the product build): every role of CTA (0, 0, 0) adds up the cycles it spends in
// each of its barrier waits and prints them for the first launches with >= 48 key tiles (profiles/r2_attention_issue.md).
#ifdef EV_ATTN_PROBE
__device__ int tca_probe_count = 0;
#define TCA_WAIT(bar, ph, acc) do { const long long t0_ = clock64(); mbar_wait(bar, ph); acc += clock64() - t0_; } while (0)
#define TCA_PROBE(...) __VA_ARGS__
__device__ int tca_tl_count = 0;
#define TCA_TL(id) do { if (lane == 0) tca_tl[id] = clock64() - t_kernel0; } while (0)
#define TCA_PROBE_ON (lane == 0 && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && n_tiles >= 48 && tca_probe_count < 4)
#else
#define TCA_WAIT(bar, ph, acc) mbar_wait(bar, ph)
#define TCA_PROBE(...)
#define TCA_TL(id)
#endif
template <int D, bool FP8, bool SMALL = false>
__global__ void __launch_bounds__((TcaCfg<D, FP8, SMALL>::THREADS), 1) tree_attn_tc_kernel(const __grid_constant__ CUtensorMap tmKV, TcAttnArgs ta) {
    using C = TcaCfg<D, FP8, SMALL>;
    constexpr int TCA_KS = C::KS, TCA_VS = C::VS;         // ring depths of this variant (shadow the bf16 defaults)
    const AttnArgs& a = ta.a;
    extern __shared__ uint8_t tca_smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(tca_smem_raw) + 1023) & ~(uintptr_t)1023);
    uint8_t* kv_s = smem;                                 // K ring [KS][NH x 8 KiB] | V ring [VS][NH x 8 KiB]
    uint8_t* raw_s = kv_s + (TCA_KS + TCA_VS) * C::K_BYTES;   // FP8: raw K ring [RS][64 x D B] | raw V ring [RS][64 x D B]
    uint64_t* bars = reinterpret_cast<uint64_t*>(raw_s + 2 * C::RS * C::RAW_BYTES);
    uint64_t* k_full = bars;                              // [KS]
    uint64_t* k_empty = k_full + TCA_KS;                  // [KS]
    uint64_t* v_full = k_empty + TCA_KS;                  // [VS]
    uint64_t* v_empty = v_full + TCA_VS;                  // [VS]
    uint64_t* s_full = v_empty + TCA_VS;                  // [3]
    uint64_t* p_full = s_full + C::NSP;                   // [3]
    uint64_t* o_full = p_full + C::NSP;                   // [2]
    uint64_t* o_empty = o_full + 2;                       // [2]
    uint64_t* sp_free = o_empty + 2;                      // [NSP] P.V has read P(j): the S/P region may take S(j + NSP)
    uint64_t* raw_full = sp_free + C::NSP;                // FP8: [2][RS] raw tile landed (K ring, then V ring)
    uint64_t* raw_empty = raw_full + 8;                   // FP8: [2][RS] raw tile converted
    uint32_t* tmem_base_smem = reinterpret_cast<uint32_t*>(raw_empty + 8);
    float* xmax = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(bars) + C::BAR_BYTES);  // [2 buf][2 wg][128]
    float* xsum = xmax + 2 * 2 * 128;                     // [2 wg][128]
    float* xc = xsum + 2 * 128;                           // [8 tiles][128] rescale factor of tile j at [j & 7]
    float* ostage = xc + 8 * 128;                         // [8 correction warps][32 rows][OSTR] staging of a chunk's partial output (and of the Q tile)

    TCA_PROBE(const long long t_kernel0 = clock64(); __shared__ long long tca_tl[24];)
    // grid (kv head x row group, chunk column, sequence): CTAs start in x-fastest order, so the columns beyond the live context
    // (they leave at once, below) come after every live CTA of the sequence instead of between them
    const int split = blockIdx.y;
    const int kvh = blockIdx.x % a.Hkv, rg = blockIdx.x / a.Hkv;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int R = a.T * a.G;

    // ---- prologue that does not depend on the previous kernel (overlaps it under PDL): barriers, TMEM ----
    pdl_launch_dependents();
    l2_prefetch_issue(ta.pf);
    // What tree_prep_kernel wrote at the head of the step is read BEFORE griddepcontrol.wait, and first of all: the kernel launched
    // right after tree_prep_kernel carries no programmatic-serialization attribute (ev_api.cu), so no later kernel of the step can
    // be resident before tree_prep_kernel has completed; __ldcg: an L1 line left over from the previous step must not serve.
    // The wait itself guards what the PRECEDING kernel (RoPE + K/V write) produced: Q, and the K/V of the tree's own slots.
    const int b = a.order ? __ldcg(a.order + blockIdx.z) : (int)blockIdx.z;
    const int nn = __ldcg(a.nn_eff + b);
    const int L = __ldcg(a.Lsnap + b);
    const int seq_slot = __ldcg(a.seq_slots + b);
    const int n_keys = __ldcg(a.kend_seq + b);         // one past the last bulk key slot of the sequence (tree_prep_kernel)
    // The grid covers the chunk columns of the longest context the model may see (a power of two of them for short chunks, so that
    // a growing context does not re-capture the graph): a CTA whose chunks lie beyond this sequence's keys leaves at once, before it
    // takes barriers or tensor memory - with max_ctx well above the live context there are more such CTAs than SMs, and each used
    // to hold an SM for its whole set-up (config[1] in a model sized for 2,900 tokens: 256 CTAs, 144 live, attention 426 us per
    // step against 329 with a tight max_ctx).
    if (nn == 0 || (long)split * a.cpg * a.chunk >= n_keys) {
        trace_exit(ta.pf);
        return;
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < TCA_KS; ++s) { mbar_init(&k_full[s], 1); mbar_init(&k_empty[s], 1); }
        for (int s = 0; s < TCA_VS; ++s) { mbar_init(&v_full[s], 1); mbar_init(&v_empty[s], 1); }
        for (int i = 0; i < C::NSP; ++i) { mbar_init(&s_full[i], 1); mbar_init(&p_full[i], 8); mbar_init(&sp_free[i], 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(&o_full[i], 1); mbar_init(&o_empty[i], 8); }
        if (FP8) for (int i = 0; i < 8; ++i) { mbar_init(&raw_full[i], 1); mbar_init(&raw_empty[i], 1); }   // [K|V][slot], stride 4
        fence_barrier_init();
        tma_prefetch_desc(&tmKV);
    }
    if (warp == 1) tmem_alloc<512>(tmem_base_smem);
    tc_fence_before();
    __syncthreads();       // barriers and the TMEM base are visible to every warp (still before the wait)
    tc_fence_after();
    const uint32_t tmem_base = *tmem_base_smem;
    if (warp == 2) TCA_TL(0);     // prologue done (barriers, TMEM, plan): at the wait
    if (warp != 0) {
        pdl_wait();
        trace_past_wait(ta.pf, 32);
    }
    if (warp == 2) TCA_TL(1);     // past the wait
    // This CTA walks a.cpg consecutive chunks; chunks sit at absolute key positions and each is reduced from a fresh
    // softmax state (batch-invariant, ev_attention.cuh), so how many chunks a CTA takes changes no result: the K/V
    // stream and the MMAs simply run on across chunk boundaries, the softmax / correction warps restart their state.
    const int chunk0 = split * a.cpg;
    const int tpc = a.chunk / TCA_BN;                  // tiles per chunk
    const int k_begin = chunk0 * a.chunk;
    const bool active = nn != 0 && k_begin < n_keys;   // uniform over the CTA
    const int k_end = min(k_begin + a.cpg * a.chunk, n_keys);
    const int n_tiles = active ? (k_end - k_begin + TCA_BN - 1) / TCA_BN : 0;
    // ---- Q tile -> TMEM (fp32 x 2^6 -> hi | lo fp16 pairs).  Softmax and correction threads stage it: a warp owns the
    // TMEM lanes of its 32 rows.  Warps 1..17 meet behind named barrier 5; warp 0 goes straight to its K/V
    // loads, which run under the staging (~1.5 us of a 15 us launch at batch 1). ----
    if (!FP8 && active && warp >= 2 && warp < 18) {
        // softmax AND correction warps: warp = (32 rows, quarter of d).  The rows are read with the lanes ALONG d (whole 128-byte
        // row quarters per access: a thread per row, the layout tcgen05.st wants, made every load instruction touch 32 lines and
        // the 64-KiB tile took 6,000 cycles to arrive at batch 1; profiles/r2_attention_issue.md section 5), split into hi | lo
        // fp16 pairs where they land, and turned through shared memory into the thread-per-row layout, one part at a time.
        constexpr int FPR = D / 4;         // floats of a row this warp handles
        constexpr int L4 = FPR / 4;        // lanes per row (one float4 each)
        constexpr int RPI = 32 / L4;       // rows per load instruction
        constexpr int NIT = 32 / RPI;      // load instructions (= D / 16)
        constexpr int WPR = FPR / 2;       // words (fp16 pairs) per row and part
        const int qd = (warp - 2) >> 2;   // 0..3
        const int r = (warp & 3) * 32 + lane;
        const int row = rg * 128 + r;
        const int node = row / a.G, gi = row % a.G;
        const bool valid = row < R && node < nn;
        const int my_off = valid ? (int)((size_t)(b * a.T + node) * a.q_ld + (size_t)(kvh * a.G + gi) * D) : -1;   // this thread's own row
        const uint32_t q_addr = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + C::TQ + qd * (D / 8);
        uint32_t* qst = reinterpret_cast<uint32_t*>(ostage) + (warp - 2) * 32 * (WPR + 1);
        const int rsub = lane / L4, c4 = lane % L4;
        float4 u[NIT];
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const int off = __shfl_sync(0xffffffffu, my_off, it * RPI + rsub);
            u[it] = off >= 0 ? *reinterpret_cast<const float4*>(a.q + off + qd * FPR + c4 * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
        uint32_t hw[2 * NIT], lw[2 * NIT];
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            split2_pack(u[it].x * TCA_QSCALE, u[it].y * TCA_QSCALE, hw[2 * it], lw[2 * it]);
            split2_pack(u[it].z * TCA_QSCALE, u[it].w * TCA_QSCALE, hw[2 * it + 1], lw[2 * it + 1]);
        }
#pragma unroll
        for (int part = 0; part < 2; ++part) {
#pragma unroll
            for (int it = 0; it < NIT; ++it) {
                uint32_t* dst = qst + (it * RPI + rsub) * (WPR + 1) + 2 * c4;
                dst[0] = part ? lw[2 * it] : hw[2 * it];
                dst[1] = part ? lw[2 * it + 1] : hw[2 * it + 1];
            }
            __syncwarp();
            uint32_t w[WPR];
#pragma unroll
            for (int j = 0; j < WPR; ++j) w[j] = qst[lane * (WPR + 1) + j];
            if (WPR == 16) tmem_st16(q_addr + part * (D / 2), w);
            else tmem_st8(q_addr + part * (D / 2), w);
            __syncwarp();
        }
        tmem_st_wait();
        tc_fence_before();
    }
    if (FP8 && active && warp >= 2 && warp < 18) {
        // FP8 pool variant (no room for the staging tile beside the raw rings): thread = (row, quarter of d)
        const int qd = (warp - 2) >> 2;   // 0..3
        const int r = (warp & 3) * 32 + lane;
        const int row = rg * 128 + r;
        const int node = row / a.G, gi = row % a.G;
        const bool valid = row < R && node < nn;
        const float* qp = a.q + (size_t)(b * a.T + (valid ? node : 0)) * a.q_ld + (size_t)(kvh * a.G + (valid ? gi : 0)) * D + qd * (D / 4);
        const uint32_t q_addr = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + C::TQ + qd * (D / 8);
        float4 u[D / 16];
#pragma unroll
        for (int i = 0; i < D / 16; ++i) u[i] = valid ? *reinterpret_cast<const float4*>(qp + i * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int g = 0; g < D / 64; ++g) {   // 16 elements = 8 columns of pairs per group
            uint32_t h[8], l[8];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                split2_pack(u[4 * g + i].x * TCA_QSCALE, u[4 * g + i].y * TCA_QSCALE, h[2 * i], l[2 * i]);
                split2_pack(u[4 * g + i].z * TCA_QSCALE, u[4 * g + i].w * TCA_QSCALE, h[2 * i + 1], l[2 * i + 1]);
            }
            tmem_st8(q_addr + g * 8, h);
            tmem_st8(q_addr + D / 2 + g * 8, l);
        }
        tmem_st_wait();
        tc_fence_before();
    }
    if (warp != 0 && warp < 18) {
        if (warp == 2) TCA_TL(2);     // this warp's part of Q is in TMEM
        asm volatile("bar.sync 5, %0;" ::"n"(TCA_THREADS - 32) : "memory");
        tc_fence_after();
        if (warp == 2) TCA_TL(3);     // Q staged (all warps)
    }

    if (!active) {
        // nothing to do for this (sequence, split): fall through to the TMEM release
    } else if (warp == 0) {
        // ===== TMA producer: lane i issues box i of the tile (K|V, page, half) =====
        constexpr int OPS = 2 * 4;
        const int32_t* pt = a.page_table + (size_t)seq_slot * a.max_pages;
        const int kv = lane >> 2, pg = lane & 3;
        // K and V tiles travel in separate rings: a K tile is released as soon as Q.K^T of its tile has run, a V
        // tile only after P.V.  Page ids are looked up one iteration ahead (off the critical path).  An L2 look-ahead (cp.async.bulk.prefetch.tensor
        // of tile j + 8) was tried and removed: the extra boxes go through the same TMA unit as the loads and made
        // IT the bottleneck (profiles/r1_attention_v2.md); for the same reason a block is ONE box, not one per half.
        auto box_row = [&](int j) {
            const int pid = pt[min((k_begin + j * TCA_BN) / TCA_PAGE + pg, a.max_pages - 1)];
            return (ta.row0 + ((pid * 2 + kv) * a.Hkv + kvh) * TCA_PAGE) >> 3;   // 8-row group index
        };
        // Lanes 0..3 stream the K tiles, lanes 4..7 the V tiles, as two INDEPENDENT loops (divergent lanes of one warp):
        // each stream runs as far ahead as its own ring allows.  In one common loop a full V ring (V tiles are
        // released by P.V, two tiles behind Q.K^T) also held back the K loads, and the MMA warp waited ~420 cycles per
        // tile for K.  The lane that owns page 0 arms the tile's full barrier (arrive + expected bytes); a box of
        // another lane may complete first - the phase still cannot complete before that arrive.
        const int dst_off = pg * C::PAGE_BYTES;
        // tiles that lie entirely in the committed context [0, L) were written by earlier steps: their loads start before
        // griddepcontrol.wait, under the tail of the RoPE kernel (at batch 1 the first K/V tile used to arrive ~4 us after the wait)
        const int n_old = min(n_tiles, max(0, L - k_begin) / TCA_BN);
        if (FP8) {
            // raw E4M3 page blocks: one linear 16-token x D-byte copy per (K|V, page) into the raw ring; lanes 0..3 stream K, 4..7 V
            if (lane < OPS) {
                uint64_t* full = raw_full + 4 * kv;
                uint64_t* empty = raw_empty + 4 * kv;
                uint8_t* ring = raw_s + kv * C::RS * C::RAW_BYTES;
                int row_next = box_row(0);
                for (int j = 0; j < n_tiles; ++j) {
                    if (j == n_old) pdl_wait();
                    const int row_cur = row_next;
                    if (j + 1 < n_tiles) row_next = box_row(j + 1);
                    const int sl = j % C::RS;
                    mbar_wait(&empty[sl], ((j / C::RS) & 1) ^ 1);
                    if (pg == 0) mbar_arrive_expect_tx(&full[sl], C::RAW_BYTES);
                    bulk_load_1d(ring + sl * C::RAW_BYTES + pg * (TCA_PAGE * D), ta.pool8 + (size_t)row_cur * 8 * D, TCA_PAGE * D, &full[sl]);
                }
            }
        } else if (lane < OPS) {
            uint64_t* full = kv ? v_full : k_full;
            uint64_t* empty = kv ? v_empty : k_empty;
            const int depth = kv ? TCA_VS : TCA_KS;
            uint8_t* ring = kv_s + (kv ? TCA_KS * C::K_BYTES : 0);
            int row_next = box_row(0);
            for (int j = 0; j < n_tiles; ++j) {
                if (j == n_old) pdl_wait();
                const int row_cur = row_next;
                if (j + 1 < n_tiles) row_next = box_row(j + 1);
                const int sl = j % depth;
                mbar_wait(&empty[sl], ((j / depth) & 1) ^ 1);
                if (pg == 0) mbar_arrive_expect_tx(&full[sl], C::K_BYTES);
                tma_load_4d(ring + sl * C::K_BYTES + dst_off, &tmKV, &full[sl], 0, 0, 0, row_cur);
            }
        }
    } else if (warp == 1 || warp == C::PV_WARP) {
        // ===== MMA issuers.  The WHOLE warp runs the loop (so addresses and descriptors are provably warp-uniform and
        // live in uniform registers); one elected lane issues.  Under `if (lane == 0)` the compiler wrapped every
        // tcgen05.mma in an ELECT / R2UR / BRA.U.ANY loop: ~100 cycles per instruction (profiles/r1_attention_v2.md).
        // A tcgen05.mma holds its issuing thread until the tensor pipe takes it: with ONE issuer the thread's time per tile
        // was the pipe's 1,024 cycles + ~350 of barrier round trips and commits + its waits, during which the pipe drained
        // (1,900 cycles per tile; profiles/r2_attention_issue.md).  With TWO_ISSUERS warp 1 issues Q.K^T and warp PV_WARP
        // issues P.V, so one warp's waits run under the other's MMAs; the pipe then no longer orders S(j) behind
        // P.V(j - NSP) by itself: sp_free says so. =====
        constexpr uint32_t idesc_qk = umma_idesc_f16(128, TCA_BN, 0);
        constexpr uint32_t idesc_pv = umma_idesc_f16(128, D, 1);
        const bool leader = elect_one();
        const uint32_t q_tmem = tmem_base + C::TQ;
        const uint32_t kv_addr = smem_u32(kv_s);
        TCA_PROBE(long long pw[5] = {0, 0, 0, 0, 0}; const long long t_begin = clock64();)
        auto issue_pv = [&](int i) {
            const int s = i % TCA_VS;
            TCA_WAIT(&v_full[s], (i / TCA_VS) & 1, pw[2]);
            TCA_WAIT(&o_empty[i % C::NO], ((i / C::NO) & 1) ^ 1, pw[3]);   // the correction warps have read chunk i - NO
            TCA_WAIT(&p_full[i % C::NSP], (i / C::NSP) & 1, pw[4]);
            tc_fence_after();
            const uint64_t vdesc = umma_desc_mn128(kv_addr + (TCA_KS + s) * C::K_BYTES, 1024, C::SBO);
            const uint32_t d_addr = tmem_base + C::TO + (i % C::NO) * D;
            const uint32_t p_addr = tmem_base + C::TP + (i % C::NSP) * C::SP;
            if (leader) {
#pragma unroll
                for (int part = 1; part >= 0; --part) {
#pragma unroll
                    for (int t = 0; t < TCA_BN / 16; ++t)
                        umma_bf16_ts(d_addr, p_addr + part * 32 + t * 8, vdesc + (uint64_t)(t * (C::PAGE_BYTES >> 4)), idesc_pv,
                                     (part == 1 && t == 0) ? 0u : 1u);
                }
                if (C::TWO_ISSUERS) umma_commit(&sp_free[i % C::NSP]);
                umma_commit(&v_empty[s]);
                umma_commit(&o_full[i % C::NO]);
            }
            __syncwarp();
        };
        auto issue_qk = [&](int j) {
            const int s = j % TCA_KS;
            TCA_WAIT(&k_full[s], (j / TCA_KS) & 1, pw[0]);
            if (C::TWO_ISSUERS) TCA_WAIT(&sp_free[j % C::NSP], ((j / C::NSP) & 1) ^ 1, pw[1]);   // P.V(j - NSP) has read the region S(j) goes into
            tc_fence_after();
            const uint32_t k_addr = kv_addr + s * C::K_BYTES;
            const uint32_t s_addr = tmem_base + C::TS + (j % C::NSP) * C::SP;
            if (leader) {
#pragma unroll
                for (int part = 1; part >= 0; --part) {
#pragma unroll
                    for (int h = 0; h < C::NH; ++h) {
                        const uint64_t bdesc = umma_desc_k128(k_addr + h * 1024, C::SBO);
#pragma unroll
                        for (int ks = 0; ks < 4; ++ks)  // UMMA K = 16 elements: 8 TMEM columns of Q pairs, 32 B of a K row
                            umma_bf16_ts(s_addr, q_tmem + part * (D / 2) + (h * 4 + ks) * 8, bdesc + 2 * ks, idesc_qk,
                                         (part == 1 && h == 0 && ks == 0) ? 0u : 1u);
                    }
                }
                umma_commit(&k_empty[s]);
                umma_commit(&s_full[j % C::NSP]);
            }
            __syncwarp();
        };
        if (C::TWO_ISSUERS) {
            if (warp == 1) for (int j = 0; j < n_tiles; ++j) issue_qk(j);
            else for (int i = 0; i < n_tiles; ++i) issue_pv(i);
        } else {
            // one issuer: Q.K^T runs NSP - 1 tiles ahead of P.V; S(j + NSP - 1) goes into the region P(j-1) was read from by
            // P.V(j-1), issued one iteration earlier (the tensor pipe executes one thread's MMAs in issue order)
            constexpr int LA = C::NSP - 1;
            for (int j = 0; j < min(LA, n_tiles); ++j) issue_qk(j);
            for (int j = 0; j < n_tiles; ++j) {
                if (j + LA < n_tiles) issue_qk(j + LA);
                issue_pv(j);
            }
        }
        TCA_PROBE(if (TCA_PROBE_ON) printf("mma warp %d: tiles %d total %lld | waits k_full %lld sp_free %lld v_full %lld o_empty %lld p_full %lld\n", warp, n_tiles,
                                          clock64() - t_begin, pw[0], pw[1], pw[2], pw[3], pw[4]);)
    } else if (warp >= 18) {
        // ===== FP8 converters (warp 18: K tiles, warp 19: V tiles): raw [64 keys][D codes] -> fp16 tile in the layout the
        // 4-D TMA box of the bf16 path produces: [8-key group][d half][8 rows x 128 B], 16-byte chunks XOR-swizzled by row =====
        if (FP8 && warp < 20) {
            const int kv = warp - 18;
            uint64_t* rfull = raw_full + 4 * kv;
            uint64_t* rempty = raw_empty + 4 * kv;
            uint64_t* tfull = kv ? v_full : k_full;
            uint64_t* tempty = kv ? v_empty : k_empty;
            const int depth = kv ? TCA_VS : TCA_KS;
            const uint8_t* raw = raw_s + kv * C::RS * C::RAW_BYTES;
            uint8_t* ring = kv_s + (kv ? TCA_KS * C::K_BYTES : 0);
            constexpr int CPR = D / 16;               // 16-code chunks per key row
            for (int j = 0; j < n_tiles; ++j) {
                const int rs = j % C::RS, ts = j % depth;
                mbar_wait(&rfull[rs], (j / C::RS) & 1);
                mbar_wait(&tempty[ts], ((j / depth) & 1) ^ 1);     // the MMAs that read this slot's previous tile have finished
                const uint8_t* src = raw + rs * C::RAW_BYTES;
                uint8_t* dst = ring + ts * C::K_BYTES;
                for (int c0 = 0; c0 < TCA_BN * CPR; c0 += 8 * 32) {   // 8 chunks per lane in flight: loads first, then convert + store
                    uint4 in[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const int c = c0 + u * 32 + lane;
                        in[u] = *reinterpret_cast<const uint4*>(src + (c / CPR) * D + (c % CPR) * 16);
                    }
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const int c = c0 + u * 32 + lane;
                        const int r = c / CPR, j8 = c % CPR;           // key row, chunk of 16 dims
                        uint4 lo, hi;
                        e4m3x16_to_f16(in[u], lo, hi);
                        const int h = j8 >> 2, jj = (j8 & 3) * 2;      // d half (64 dims), first of the two 16-byte chunks inside the 128-byte row
                        uint8_t* rowp = dst + (r >> 3) * C::SBO + h * 1024 + (r & 7) * 128;
                        *reinterpret_cast<uint4*>(rowp + ((jj ^ (r & 7)) << 4)) = lo;
                        *reinterpret_cast<uint4*>(rowp + (((jj + 1) ^ (r & 7)) << 4)) = hi;
                    }
                }
                fence_proxy_async();      // generic-proxy stores -> visible to the tensor core's async-proxy reads
                __syncwarp();
                if (lane == 0) { mbar_arrive(&tfull[ts]); mbar_arrive(&rempty[rs]); }
            }
        }
    } else if (warp < 10) {
        // ===== softmax: thread = (row, wg); wg handles keys [32 wg, +32) of every tile.  Warp w may touch TMEM
        // lanes 32 (w % 4) .. +31; the two warps of a row quarter meet behind named barrier 1 + (w % 4). =====
        const int wg = (warp - 2) >> 2;
        const int r = (warp & 3) * 32 + lane;
        const int row = rg * 128 + r;
        const int node = row / a.G, gi = row % a.G;
        const bool valid = row < R && node < nn;
        const bool warp_valid = __any_sync(0xffffffffu, valid);   // the same for both warps of a row quarter
        const unsigned long long ab = valid ? a.anc_bulk[b * a.T + node] : 0ull;   // tree slots among this row's bulk keys
        const int erow = valid ? a.erow[b * a.T + node] : 0;                       // cached positions below erow are bulk keys
        const uint32_t lane_addr = tmem_base + ((uint32_t)((warp & 3) * 32) << 16);
        constexpr float LOG2E = 1.4426950408889634f;
        float m_run = -INFINITY, l_run = 0.f;   // l_run carries P's factor 2^15
        // Scores stay RAW in the loop (S = 2^6 q . k): s = rn(S * qk_scale) is the method's rounded score and rounding is monotone,
        // so the chunk's max is rn(max(S) * qk_scale), taken once when the chunk ends; the exponent (S - M) * k2 is one FFMA per key.
        const float qk_scale = FP8 ? mul_rn(a.scale * (1.f / TCA_QSCALE), ta.k_scale) : a.scale * (1.f / TCA_QSCALE);   // FP8: the K cache's static scale rides along
        const float k2 = mul_rn(qk_scale, LOG2E);

        // (max, sum) of a finished chunk go to its partial slot (the two halves of a row meet in shared memory) and the
        // state restarts: t_left counts the tiles left in the current chunk
        float2* mlp = reinterpret_cast<float2*>(a.ml_part) + ((size_t)(b * a.T + (valid ? node : 0)) * a.Hq + kvh * a.G + (valid ? gi : 0)) * a.n_chunks + chunk0;
        int t_left = tpc;
        TCA_PROBE(long long pw[4] = {0, 0, 0, 0}; const long long t_begin = clock64();)
        for (int j = 0; j < n_tiles; ++j) {
            TCA_WAIT(&s_full[j % C::NSP], (j / C::NSP) & 1, pw[0]);
            tc_fence_after();
            if (warp == 2 && j < 4) TCA_TL(4 + j);    // S(j) ready
            if (!warp_valid) {   // no live row in this warp (chain drafts: 16 of 128 rows): keep the barrier protocol only
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&p_full[j % C::NSP]);
                continue;
            }
            uint32_t sv[32];
            TCA_PROBE(const long long tA = clock64();)
            tmem_ld32(lane_addr + C::TS + (j % C::NSP) * C::SP + wg * 32, sv);
            tmem_ld_wait();
            const int kb = k_begin + j * TCA_BN + wg * 32;
            if (kb + 32 > L - ATT_TAIL_R) {   // tile half reaches the end of some row's bulk (warp-uniform)
#pragma unroll
                for (int e = 0; e < 32; ++e)
                    if (!bulk_key(kb + e, L, erow, ab)) sv[e] = 0xFF800000u;  // -inf
            }
            float mx0 = fmaxf(__uint_as_float(sv[0]), __uint_as_float(sv[1])), mx1 = fmaxf(__uint_as_float(sv[2]), __uint_as_float(sv[3]));
#pragma unroll
            for (int e = 4; e < 32; e += 2) {
                mx0 = fmaxf(mx0, __uint_as_float(sv[e]));
                mx1 = fmaxf(mx1, __uint_as_float(sv[e + 1]));
            }
            float mx = fmaxf(mx0, mx1);
            xmax[((j & 1) * 2 + wg) * 128 + r] = mx;
            TCA_PROBE(const long long tB = clock64(); pw[1] += tB - tA;)
            pair_bar_sync(1 + (warp & 3));
            TCA_PROBE(const long long tC = clock64(); pw[2] += tC - tB;)
            mx = fmaxf(mx, xmax[((j & 1) * 2 + (wg ^ 1)) * 128 + r]);
            const float mn = fmaxf(m_run, mx);
            const float mu = (mn == -INFINITY) ? 0.f : mn;
            const float c = ex2_approx((m_run - mu) * k2);  // 2^-inf = 0 on the first tile
            m_run = mn;
            if (wg == 0) xc[(j & 7) * 128 + r] = c;
            const float nmk = fmaf(-mu, k2, TCA_PSCALE_LOG2);   // p' = 2^15 p
            float ls0 = 0.f, ls1 = 0.f;
            const uint32_t p_addr = lane_addr + C::TP + (j % C::NSP) * C::SP + wg * 16;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                uint32_t ph[8], pl[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const float p0 = ex2_approx(fmaf(__uint_as_float(sv[16 * h + 2 * e]), k2, nmk));
                    const float p1 = ex2_approx(fmaf(__uint_as_float(sv[16 * h + 2 * e + 1]), k2, nmk));
                    ls0 += p0;
                    ls1 += p1;
                    split2_pack(p0, p1, ph[e], pl[e]);
                }
                tmem_st8(p_addr + h * 8, ph);
                tmem_st8(p_addr + 32 + h * 8, pl);
            }
            l_run = fmaf(l_run, c, ls0 + ls1);
            tmem_st_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(&p_full[j % C::NSP]);
            TCA_PROBE(pw[3] += clock64() - tC;)
            if (--t_left == 0 || j == n_tiles - 1) {   // chunk finished (CTA-uniform)
                xsum[wg * 128 + r] = l_run * exp2f(-TCA_PSCALE_LOG2);   // exact
                pair_bar_sync(1 + (warp & 3));
                if (valid && wg == 0) *mlp = make_float2(mul_rn(m_run, qk_scale), xsum[r] + xsum[128 + r]);
                ++mlp;
                m_run = -INFINITY; l_run = 0.f;
                t_left = tpc;
            }
        }
        if (warp == 2) TCA_TL(8);     // softmax done
        TCA_PROBE(if ((warp == 2 || warp == 6) && TCA_PROBE_ON) printf("softmax warp %d: tiles %d total %lld | wait s_full %lld | ld + max %lld pair barrier %lld exp + split + st + arrive %lld\n",
                                                                      warp, n_tiles, clock64() - t_begin, pw[0], pw[1], pw[2], pw[3]);)
    } else {
        // ===== correction: thread = (row, half of d).  O = O * c(i) + Oc(i), one rounded fp32 operation per tile;
        // c(i) was published by the softmax warps before they released P(i), which Oc(i) depends on. =====
        const int hh = (warp - 10) >> 2;
        const int r = (warp & 3) * 32 + lane;
        const int row = rg * 128 + r;
        const int node = row / a.G, gi = row % a.G;
        const bool valid = row < R && node < nn;
        const bool warp_valid = __any_sync(0xffffffffu, valid);
        const uint32_t lane_addr = tmem_base + ((uint32_t)((warp & 3) * 32) << 16);
        float o[C::DH];
#pragma unroll
        for (int i = 0; i < C::DH; ++i) o[i] = 0.f;
        float* op = a.o_part + (((size_t)(b * a.T + (valid ? node : 0)) * a.Hq + kvh * a.G + (valid ? gi : 0)) * a.n_chunks + chunk0) * D + hh * C::DH;
        int t_left = tpc;
        const float oscale = FP8 ? mul_rn(exp2f(-TCA_PSCALE_LOG2), ta.v_scale) : exp2f(-TCA_PSCALE_LOG2);   // P's 2^15 out (exact); FP8: V's static scale in
        float* ost = ostage + (warp - 10) * 32 * C::OSTR;
        TCA_PROBE(long long pw = 0; const long long t_begin = clock64();)
        for (int i = 0; i < n_tiles; ++i) {
            TCA_WAIT(&o_full[i % C::NO], (i / C::NO) & 1, pw);
            if (warp == 10 && i == n_tiles - 1) TCA_TL(9);   // last P.V result ready
            tc_fence_after();
            if (!warp_valid) {   // no live row in this warp: release the chunk, nothing to add
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&o_empty[i % C::NO]);
                continue;
            }
            const bool last = --t_left == 0 || i == n_tiles - 1;   // the key chunk ends with this tile (CTA-uniform)
            const float c = xc[(i & 7) * 128 + r];
#pragma unroll
            for (int cb = 0; cb < C::DH / 16; ++cb) {
                uint32_t ov[16];
                tmem_ld16(lane_addr + C::TO + (i % C::NO) * D + hh * C::DH + cb * 16, ov);
                tmem_ld_wait();
                if (cb == C::DH / 16 - 1) {
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&o_empty[i % C::NO]);
                }
#pragma unroll
                for (int e = 0; e < 16; ++e) o[cb * 16 + e] = fmaf(o[cb * 16 + e], c, __uint_as_float(ov[e]));
            }
            if (last) {   // the chunk's partial output goes out (P's factor 2^15 taken out exactly), fresh accumulator
                const unsigned vmask = __ballot_sync(0xffffffffu, valid);
                const unsigned long long opa = reinterpret_cast<unsigned long long>(op);
                constexpr int L4 = C::OPW / 4;       // lanes per row (one float4 each)
                constexpr int RPI = 32 / L4;         // rows per store instruction
#pragma unroll
                for (int ps = 0; ps < C::DH / C::OPW; ++ps) {
#pragma unroll
                    for (int e = 0; e < C::OPW; e += 4)
                        *reinterpret_cast<float4*>(ost + lane * C::OSTR + e) = make_float4(o[ps * C::OPW + e] * oscale, o[ps * C::OPW + e + 1] * oscale,
                                                                                          o[ps * C::OPW + e + 2] * oscale, o[ps * C::OPW + e + 3] * oscale);
                    __syncwarp();
#pragma unroll
                    for (int it = 0; it < 32 / RPI; ++it) {
                        const int rr = it * RPI + lane / L4, c4 = lane % L4;
                        const float4 v = *reinterpret_cast<const float4*>(ost + rr * C::OSTR + c4 * 4);
                        const unsigned long long pa = __shfl_sync(0xffffffffu, opa, rr);
                        if ((vmask >> rr) & 1u) *reinterpret_cast<float4*>(reinterpret_cast<float*>(pa) + ps * C::OPW + c4 * 4) = v;
                    }
                    __syncwarp();
                }
#pragma unroll
                for (int e = 0; e < C::DH; ++e) o[e] = 0.f;
                op += D; t_left = tpc;
            }
        }
        if (warp == 10) TCA_TL(10);   // partials written
        TCA_PROBE(if (warp == 10 && TCA_PROBE_ON) printf("correction warp 10: tiles %d total %lld | wait o_full %lld\n", n_tiles, clock64() - t_begin, pw);)
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc<512>(tmem_base);
    TCA_PROBE(if (threadIdx.x == 0 && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && n_tiles >= 48) atomicAdd(&tca_probe_count, 1);)
    TCA_PROBE(if (threadIdx.x == 0 && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && n_tiles > 0 && n_tiles <= 8) {
        // short launches (batch 1): one CTA's timeline in cycles from kernel entry, printed for a few launches after warm-up
        if (tca_tl_count >= 400 && tca_tl_count < 404)
            printf("timeline (%d tiles): at wait %lld | past wait %lld | own Q part in TMEM %lld | Q staged %lld | S ready %lld %lld %lld %lld | softmax done %lld | "
                   "last P.V ready %lld | partials written %lld | end %lld\n", n_tiles, tca_tl[0], tca_tl[1], tca_tl[2], tca_tl[3], tca_tl[4], tca_tl[5], tca_tl[6],
                   tca_tl[7], tca_tl[8], tca_tl[9], tca_tl[10], clock64() - t_kernel0);
        atomicAdd(&tca_tl_count, 1);
    })
    trace_exit(ta.pf);
}

}  // namespace ev
