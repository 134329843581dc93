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
// main loop of item i+1.  Split-K (few tiles, small M) is deterministic: every split writes its raw
// fp32 partial, the split that arrives last at the tile's counter sums ALL partials in split order.
// Programmatic dependent launch: barrier setup, TMEM allocation and the first STAGES weight tiles
// are issued BEFORE griddepcontrol.wait (weights do not depend on the previous kernel), so the
// weight stream of this GEMM starts while the previous (element-wise) kernel is still running.
#pragma once
#include "ev_common.cuh"

namespace ev {

enum GemmEpi { EPI_STORE = 0, EPI_RESID = 1, EPI_ARGMAX = 2 };

constexpr int GEMM_THREADS = 192;
constexpr int GEMM_BK = 128;          // bytes (= E4M3 elements) of K per stage: one swizzle row
constexpr int GEMM_WROWS = 128;       // output channels per tile = UMMA M
constexpr int GEMM_WTILE = GEMM_WROWS * GEMM_BK;  // 16 KiB
constexpr int GEMM_MAX_STAGES = 10;
constexpr int GEMM_SMEM_BUDGET = 200 * 1024;

struct GemmArgs {
    int M, N;
    int total_kb;       // ceil(K / 128) = K tiles of W
    int n_tiles, m_tiles, k_splits, kb_per_split;
    int tok;            // tokens per tile (UMMA N), multiple of 16, <= 256
    int stages;
    const uint8_t* W;   // tiled + swizzled codes: [n_tiles][total_kb][16 KiB]
    const float* sx;    // [M]
    const float* sw;    // [N]
    float* out;         // [M][ldo]; EPI_RESID: out += y in place; EPI_ARGMAX: optional logits
    int ldo;
    float* partial;     // split-K: [tile][split][tok][128] raw fp32
    int* tile_counter;  // split-K: [tile], zero on entry and on exit
    unsigned long long* argmax_keys;  // EPI_ARGMAX: [M] packed (ordered logit, ~index)
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

struct GemmItem { int n_tile, m_tile, split, tile, kb0, nkb; };
__device__ __forceinline__ GemmItem gemm_item(const GemmArgs& a, int w) {
    GemmItem it;
    it.split = w % a.k_splits;
    it.tile = w / a.k_splits;
    it.m_tile = it.tile % a.m_tiles;
    it.n_tile = it.tile / a.m_tiles;
    it.kb0 = it.split * a.kb_per_split;
    it.nkb = min(a.kb_per_split, a.total_kb - it.kb0);
    return it;
}

template <int EPI>
__global__ void __launch_bounds__(GEMM_THREADS, 1) gemm_e4m3_kernel(const __grid_constant__ CUtensorMap tmX, GemmArgs a) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    const int x_bytes = a.tok * GEMM_BK;
    const int stage_bytes = GEMM_WTILE + x_bytes;
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + a.stages * stage_bytes);
    uint64_t* empty_bar = full_bar + GEMM_MAX_STAGES;
    uint64_t* tmem_full_bar = empty_bar + GEMM_MAX_STAGES;   // [2]
    uint64_t* tmem_empty_bar = tmem_full_bar + 2;            // [2]
    uint32_t* tmem_base_smem = reinterpret_cast<uint32_t*>(tmem_empty_bar + 2);
    int* flag_smem = reinterpret_cast<int*>(tmem_base_smem + 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int total_items = a.n_tiles * a.m_tiles * a.k_splits;
    uint32_t tmem_cols = 32;
    while ((int)tmem_cols < 2 * a.tok) tmem_cols <<= 1;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmX);
        for (int s = 0; s < a.stages; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(&tmem_full_bar[i], 1); mbar_init(&tmem_empty_bar[i], 4); }
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc_rt(tmem_base_smem, tmem_cols);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_base_smem;

    if (warp == 0) {
        if (lane == 0) {  // ===== producer: weights by linear bulk copy, activations by 2-D TMA =====
            const uint64_t pol_w = policy_evict_first();   // weights are streamed once per step
            const uint64_t pol_x = policy_evict_last();    // activations are re-read by every tile
            int s = 0;
            uint32_t ph = 0;
            int w = blockIdx.x;
            int pre = 0;
            GemmItem it0;
            if (w < total_items) {  // weight tiles of the first item: no dependency on the previous kernel
                it0 = gemm_item(a, w);
                pre = min(a.stages, it0.nkb);
                for (int i = 0; i < pre; ++i) {
                    mbar_arrive_expect_tx(&full_bar[i], stage_bytes);
                    bulk_load(smem + i * stage_bytes, a.W + ((size_t)it0.n_tile * a.total_kb + it0.kb0 + i) * GEMM_WTILE,
                              GEMM_WTILE, &full_bar[i], pol_w);
                }
            }
            pdl_wait();  // activations (and everything the epilogue reads) come from the previous kernel
            for (int i = 0; i < pre; ++i)
                tma_load_2d_hint(smem + i * stage_bytes + GEMM_WTILE, &tmX, &full_bar[i], (it0.kb0 + i) * GEMM_BK,
                                 it0.m_tile * a.tok, pol_x);
            s = pre;
            if (s == a.stages) { s = 0; ph ^= 1; }
            for (; w < total_items; w += gridDim.x) {
                const GemmItem it = gemm_item(a, w);
                for (int kb = (w == (int)blockIdx.x ? pre : 0); kb < it.nkb; ++kb) {
                    mbar_wait(&empty_bar[s], ph ^ 1);
                    mbar_arrive_expect_tx(&full_bar[s], stage_bytes);
                    uint8_t* st = smem + s * stage_bytes;
                    bulk_load(st, a.W + ((size_t)it.n_tile * a.total_kb + it.kb0 + kb) * GEMM_WTILE, GEMM_WTILE, &full_bar[s], pol_w);
                    tma_load_2d_hint(st + GEMM_WTILE, &tmX, &full_bar[s], (it.kb0 + kb) * GEMM_BK, it.m_tile * a.tok, pol_x);
                    if (++s == a.stages) { s = 0; ph ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {  // ===== MMA issuer =====
            const uint32_t idesc = umma_idesc_e4m3(GEMM_WROWS, a.tok);
            int s = 0;
            uint32_t ph = 0;
            int n_it = 0;
            for (int w = blockIdx.x; w < total_items; w += gridDim.x, ++n_it) {
                const GemmItem it = gemm_item(a, w);
                const int buf = n_it & 1;
                mbar_wait(&tmem_empty_bar[buf], ((n_it >> 1) & 1) ^ 1);  // epilogue has drained this accumulator
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + (uint32_t)(buf * a.tok);
                for (int kb = 0; kb < it.nkb; ++kb) {
                    mbar_wait(&full_bar[s], ph);
                    tc_fence_after();
                    const uint32_t wa = smem_u32(smem + s * stage_bytes);
                    const uint64_t adesc = umma_desc_k128(wa);
                    const uint64_t bdesc = umma_desc_k128(wa + GEMM_WTILE);
#pragma unroll
                    for (int k = 0; k < GEMM_BK / 32; ++k)  // UMMA K = 32 E4M3 elements = 2 x 16 B
                        umma_f8(d_tmem, adesc + 2 * k, bdesc + 2 * k, idesc, (kb | k) != 0);
                    umma_commit(&empty_bar[s]);
                    if (++s == a.stages) { s = 0; ph ^= 1; }
                }
                umma_commit(&tmem_full_bar[buf]);
            }
        }
    } else {  // ===== epilogue: warps 2..5; warp w may touch TMEM lanes 32*(w%4) .. +31 =====
        pdl_wait();
        const int q = warp & 3;
        const int et = (int)threadIdx.x - 64;  // 0..127 among the epilogue threads
        int n_it = 0;
        for (int w = blockIdx.x; w < total_items; w += gridDim.x, ++n_it) {
            const GemmItem it = gemm_item(a, w);
            const int buf = n_it & 1;
            const int n_loc = q * 32 + lane;
            const int n = it.n_tile * GEMM_WROWS + n_loc;
            const int m0 = it.m_tile * a.tok;
            const bool n_ok = n < a.N;
            const float swn = n_ok ? a.sw[n] : 0.f;
            mbar_wait(&tmem_full_bar[buf], (n_it >> 1) & 1);
            tc_fence_after();
            const uint32_t t_addr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * a.tok);
            const int n_chunks = a.tok / 16;
            bool reduce_here = true;
            float* part = nullptr;
            if (a.k_splits > 1) {
                // ---- split-K: publish the raw partial, last arriver reduces all of them in split order ----
                part = a.partial + (size_t)it.tile * a.k_splits * a.tok * GEMM_WROWS;
                float* mine = part + (size_t)it.split * a.tok * GEMM_WROWS;
                for (int c = 0; c < n_chunks; ++c) {
                    uint32_t v[16];
                    tmem_ld16(t_addr + (uint32_t)(c * 16), v);
                    tmem_ld_wait();
#pragma unroll
                    for (int j = 0; j < 16; ++j) mine[(size_t)(c * 16 + j) * GEMM_WROWS + n_loc] = __uint_as_float(v[j]);
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&tmem_empty_bar[buf]);
                __threadfence();
                epi_bar_sync();
                if (et == 0) {
                    const int old = atomicAdd(a.tile_counter + it.tile, 1);
                    *flag_smem = (old == a.k_splits - 1);
                    if (old == a.k_splits - 1) a.tile_counter[it.tile] = 0;  // ready for the next launch
                }
                epi_bar_sync();
                reduce_here = *flag_smem != 0;
                epi_bar_sync();  // flag is rewritten by the next item
                if (reduce_here) __threadfence();
            }
            if (reduce_here) {
                for (int c = 0; c < n_chunks; ++c) {
                    float acc[16];
                    if (a.k_splits > 1) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) acc[j] = __ldcg(part + (size_t)(c * 16 + j) * GEMM_WROWS + n_loc);
                        for (int sp = 1; sp < a.k_splits; ++sp) {
                            const float* ps = part + (size_t)sp * a.tok * GEMM_WROWS;
#pragma unroll
                            for (int j = 0; j < 16; ++j) acc[j] = add_rn(acc[j], __ldcg(ps + (size_t)(c * 16 + j) * GEMM_WROWS + n_loc));
                        }
                    } else {
                        uint32_t v[16];
                        tmem_ld16(t_addr + (uint32_t)(c * 16), v);
                        tmem_ld_wait();
#pragma unroll
                        for (int j = 0; j < 16; ++j) acc[j] = __uint_as_float(v[j]);
                        if (c == n_chunks - 1) {  // accumulator fully read: hand it back to the MMA warp
                            tc_fence_before();
                            __syncwarp();
                            if (lane == 0) mbar_arrive(&tmem_empty_bar[buf]);
                        }
                    }
                    const int mc = m0 + c * 16;
                    if (mc >= a.M) continue;  // warp-uniform
                    const int m_lane = mc + (lane & 15);
                    const float sx_lane = (m_lane < a.M) ? __ldg(a.sx + m_lane) : 0.f;
                    float res[16];
                    if (EPI == EPI_RESID) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) res[j] = (n_ok && mc + j < a.M) ? __ldcg(a.out + (size_t)(mc + j) * a.ldo + n) : 0.f;
                    }
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const float sxm = __shfl_sync(0xffffffffu, sx_lane, j);
                        const int m = mc + j;
                        const float y = mul_rn(mul_rn(acc[j], sxm), swn);
                        if (EPI == EPI_ARGMAX) {
                            unsigned long long key = (n_ok && m < a.M) ? (((unsigned long long)ordered_bits(y) << 32) | (0xFFFFFFFFu - (uint32_t)n)) : 0ull;
#pragma unroll
                            for (int o = 16; o > 0; o >>= 1) {
                                const unsigned long long other = __shfl_xor_sync(0xffffffffu, key, o);
                                key = other > key ? other : key;
                            }
                            if (lane == 0 && m < a.M) atomicMax(a.argmax_keys + m, key);
                            if (n_ok && m < a.M && a.out) __stcs(a.out + (size_t)m * a.ldo + n, y);
                        } else if (n_ok && m < a.M) {
                            a.out[(size_t)m * a.ldo + n] = (EPI == EPI_RESID) ? add_rn(res[j], y) : y;
                        }
                    }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc_rt(tmem_base, tmem_cols);
}

// debug / bring-up reference: same contraction on CUDA cores from the tiled weight layout
// (exact products, fp32 accumulation).  Used only when EV_NAIVE_GEMM=1 to bisect tensor-core issues.
__global__ void __launch_bounds__(128) gemm_e4m3_naive_kernel(const uint8_t* __restrict__ X, const uint8_t* __restrict__ Wt,
                                                              int M, int N, int K, int total_kb, const float* sx,
                                                              const float* sw, float* out, int ldo, int add_resid) {
    const int n = blockIdx.x * 128 + threadIdx.x, m = blockIdx.y;
    if (n >= N) return;
    float acc = 0.f;
    for (int k = 0; k < K; ++k) {
        const uint8_t wc = Wt[((size_t)(n >> 7) * total_kb + (k >> 7)) * GEMM_WTILE + wtile_offset(n & 127, k & 127)];
        const __half_raw hx = __nv_cvt_fp8_to_halfraw(X[(size_t)m * K + k], __NV_E4M3);
        const __half_raw hw = __nv_cvt_fp8_to_halfraw(wc, __NV_E4M3);
        acc = fmaf(__half2float(__half(hx)), __half2float(__half(hw)), acc);
    }
    const float y = mul_rn(mul_rn(acc, sx[m]), sw[n]);
    float* p = out + (size_t)m * ldo + n;
    *p = add_resid ? add_rn(*p, y) : y;
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
