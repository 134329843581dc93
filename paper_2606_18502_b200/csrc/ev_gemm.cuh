// K2: E4M3 x E4M3 -> fp32 linear layers on the 5th-gen tensor cores (tcgen05.mma kind::f8f6f4,
// accumulator in TMEM, operands staged by TMA with 128-byte swizzle).
//
// Formulation ("swap-AB"): the WEIGHT matrix W[N][K] is the MMA's M-side operand (128 output
// channels per CTA fill the 128 TMEM lanes) and the TOKENS X[M][K] are the MMA's N-side operand
// (TOK = 16..256 tokens per instruction).  Verify steps have few rows (M = B*T = 60..832) and many
// output channels, so this keeps the tensor core full at any M, streams each weight byte exactly
// once per token tile, and gives an epilogue in which the 32 lanes of a warp hold 32 consecutive
// output channels of one token: global stores are coalesced with no shared-memory staging.
//
//   y[m][n] = (sum_k X[m][k] * W[n][k]) * s_x[m] * s_w[n]            (DESIGN.md R-accum)
//
// Warp roles (192 threads): warp 0 = TMA producer (one lane), warp 1 = TMEM owner + MMA issuer
// (one lane), warps 2..5 = epilogue (TMEM -> registers -> scales -> global).
// grid = (ceil(N/128), ceil(M/TOK), k_splits).
#pragma once
#include "ev_common.cuh"

namespace ev {

enum GemmEpi { EPI_STORE = 0, EPI_RESID = 1, EPI_PARTIAL = 2, EPI_ARGMAX = 3 };

struct GemmArgs {
    int M, N, K;
    const float* sx;   // [M] per-token activation scales
    const float* sw;   // [N] per-output-channel weight scales
    float* out;        // [M][ldo]  (EPI_STORE / EPI_RESID: out = resid + y, in place; EPI_ARGMAX: optional logits)
    int ldo;
    int kb_per_split;  // 128-byte K blocks per grid.z slice
    float* partial;    // EPI_PARTIAL: [splits][M][N] raw fp32 accumulators
    unsigned long long* argmax_keys;  // EPI_ARGMAX: [M] packed (ordered logit, ~index), atomicMax
};

constexpr int GEMM_THREADS = 192;
constexpr int GEMM_BK = 128;        // bytes (= E4M3 elements) of K per pipeline stage: one swizzle row
constexpr int GEMM_WROWS = 128;     // output channels per CTA = UMMA M

template <int TOK>
struct GemmSmem {
    static constexpr int W_BYTES = GEMM_WROWS * GEMM_BK;
    static constexpr int X_BYTES = TOK * GEMM_BK;
    static constexpr int STAGE_BYTES = W_BYTES + X_BYTES;
    static constexpr int STAGES = (200 * 1024 / STAGE_BYTES) > 10 ? 10 : (200 * 1024 / STAGE_BYTES);
    static constexpr int BAR_BYTES = 256;
    static constexpr int TOTAL = STAGES * STAGE_BYTES + BAR_BYTES + 1024;  // +1024: manual alignment
    static constexpr int TMEM_COLS = TOK < 32 ? 32 : TOK;
};

// order-preserving map fp32 -> u32 (larger float => larger unsigned)
__device__ __forceinline__ uint32_t ordered_bits(float f) {
    const uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

template <int TOK, int EPI>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
gemm_e4m3_kernel(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmX, GemmArgs a) {
    using S = GemmSmem<TOK>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + S::STAGES * S::STAGE_BYTES);
    uint64_t* empty_bar = full_bar + S::STAGES;
    uint64_t* tmem_full_bar = empty_bar + S::STAGES;
    uint32_t* tmem_base_smem = reinterpret_cast<uint32_t*>(tmem_full_bar + 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n0 = blockIdx.x * GEMM_WROWS;
    const int m0 = blockIdx.y * TOK;
    const int total_kb = (a.K + GEMM_BK - 1) / GEMM_BK;
    const int kb0 = blockIdx.z * a.kb_per_split;
    const int nkb = min(a.kb_per_split, total_kb - kb0);

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmW);
        tma_prefetch_desc(&tmX);
        for (int s = 0; s < S::STAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
        mbar_init(tmem_full_bar, 1);
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc<S::TMEM_COLS>(tmem_base_smem);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_base_smem;

    if (warp == 0) {
        if (lane == 0) {  // ===== TMA producer =====
            for (int kb = 0; kb < nkb; ++kb) {
                const int s = kb % S::STAGES;
                const uint32_t ph = (kb / S::STAGES) & 1;
                mbar_wait(&empty_bar[s], ph ^ 1);
                mbar_arrive_expect_tx(&full_bar[s], S::STAGE_BYTES);
                uint8_t* ws = smem + s * S::STAGE_BYTES;
                tma_load_2d(ws, &tmW, &full_bar[s], (kb0 + kb) * GEMM_BK, n0);
                tma_load_2d(ws + S::W_BYTES, &tmX, &full_bar[s], (kb0 + kb) * GEMM_BK, m0);
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {  // ===== MMA issuer =====
            constexpr uint32_t idesc = umma_idesc_e4m3(GEMM_WROWS, TOK);
            for (int kb = 0; kb < nkb; ++kb) {
                const int s = kb % S::STAGES;
                const uint32_t ph = (kb / S::STAGES) & 1;
                mbar_wait(&full_bar[s], ph);
                tc_fence_after();
                const uint32_t wa = smem_u32(smem + s * S::STAGE_BYTES);
                const uint64_t adesc = umma_desc_k128(wa);
                const uint64_t bdesc = umma_desc_k128(wa + S::W_BYTES);
#pragma unroll
                for (int k = 0; k < GEMM_BK / 32; ++k)  // UMMA K = 32 E4M3 elements = 32 bytes = 2 x 16 B
                    umma_f8(tmem_base, adesc + 2 * k, bdesc + 2 * k, idesc, (kb | k) != 0);
                umma_commit(&empty_bar[s]);  // frees the stage when these MMAs have read it
            }
            umma_commit(tmem_full_bar);
        }
    } else {  // ===== epilogue: warps 2..5; warp w may touch TMEM lanes 32*(w%4) .. +31 =====
        const int q = warp & 3;
        const int n = n0 + q * 32 + lane;
        mbar_wait(tmem_full_bar, 0);
        tc_fence_after();
        const bool n_ok = n < a.N;
        const float swn = (EPI != EPI_PARTIAL && n_ok) ? a.sw[n] : 0.f;
#pragma unroll 1
        for (int c = 0; c < TOK / 16; ++c) {
            uint32_t v[16];
            tmem_ld16(tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(c * 16), v);
            tmem_ld_wait();
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const int m = m0 + c * 16 + j;
                if (m >= a.M) break;  // warp-uniform
                const float acc = __uint_as_float(v[j]);
                if (EPI == EPI_PARTIAL) {
                    if (n_ok) a.partial[((size_t)blockIdx.z * a.M + m) * a.N + n] = acc;
                } else {
                    const float y = mul_rn(mul_rn(acc, a.sx[m]), swn);
                    if (EPI == EPI_STORE) {
                        if (n_ok) a.out[(size_t)m * a.ldo + n] = y;
                    } else if (EPI == EPI_RESID) {
                        if (n_ok) { float* p = a.out + (size_t)m * a.ldo + n; *p = add_rn(*p, y); }
                    } else {  // EPI_ARGMAX
                        if (n_ok && a.out) a.out[(size_t)m * a.ldo + n] = y;
                        unsigned long long key = n_ok ? (((unsigned long long)ordered_bits(y) << 32) | (0xFFFFFFFFu - (uint32_t)n)) : 0ull;
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) {
                            const unsigned long long other = __shfl_xor_sync(0xffffffffu, key, o);
                            key = other > key ? other : key;
                        }
                        if (lane == 0) atomicMax(a.argmax_keys + m, key);
                    }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc<S::TMEM_COLS>(tmem_base);
}

// split-K finish: y = (sum_s partial[s]) * s_x * s_w (+ residual), splits summed in index order
__global__ void __launch_bounds__(256) splitk_finish_kernel(const float* __restrict__ partial, int splits, int M, int N,
                                                            const float* __restrict__ sx, const float* __restrict__ sw,
                                                            float* out, int ldo, int add_resid) {
    const size_t total = (size_t)M * N;
    for (size_t i = blockIdx.x * (size_t)256 + threadIdx.x; i < total; i += (size_t)gridDim.x * 256) {
        const int m = (int)(i / N), n = (int)(i % N);
        float acc = partial[i];
        for (int s = 1; s < splits; ++s) acc = add_rn(acc, partial[(size_t)s * total + i]);
        const float y = mul_rn(mul_rn(acc, sx[m]), sw[n]);
        float* p = out + (size_t)m * ldo + n;
        *p = add_resid ? add_rn(*p, y) : y;
    }
}

// debug / bring-up reference: same contraction on CUDA cores (exact products, fp32 accumulation).
// Used only by ev_op_linear(..., impl=naive) in tests to bisect tensor-core issues.
__global__ void __launch_bounds__(128) gemm_e4m3_naive_kernel(const uint8_t* __restrict__ X, const uint8_t* __restrict__ W,
                                                              int M, int N, int K, const float* sx, const float* sw,
                                                              float* out, int ldo, int add_resid) {
    const int n = blockIdx.x * 128 + threadIdx.x, m = blockIdx.y;
    if (n >= N) return;
    float acc = 0.f;
    for (int k = 0; k < K; ++k) {
        const __half_raw hx = __nv_cvt_fp8_to_halfraw(X[(size_t)m * K + k], __NV_E4M3);
        const __half_raw hw = __nv_cvt_fp8_to_halfraw(W[(size_t)n * K + k], __NV_E4M3);
        acc = fmaf(__half2float(__half(hx)), __half2float(__half(hw)), acc);
    }
    const float y = mul_rn(mul_rn(acc, sx[m]), sw[n]);
    float* p = out + (size_t)m * ldo + n;
    *p = add_resid ? add_rn(*p, y) : y;
}

}  // namespace ev
