// K5: tree-masked GQA attention over the paged bf16 KV cache ("tree attention";
// BASELINE.json:north_star (2)), split over the key axis, + K7: merge of the splits fused with the
// per-token absmax / E4M3 quantization that feeds the O projection.
//
// One CTA = (sequence b, kv head, group of 8 row tiles, key split).  The query rows of one kv head
// are the T nodes x G query heads that share it (row = node*G + g), 16 rows per warp.  Keys are the
// L committed context slots followed by the T tree slots L..L+T-1 (written by the RoPE/KV-write
// kernel just before); a tree key j is visible to node i iff j is an ancestor-or-self of i (bit j
// of anc[i]).  Pages are gathered with 16-byte cp.async into XOR-swizzled shared memory (each
// (page, K|V, head) block is page_size*D*2 contiguous bytes), double buffered; Q.K^T and P.V run on
// the tensor cores (mma.sync m16n8k16 bf16, fp32 accumulate) with Q and P each split into
// hi + mid + lo bf16 parts: 3 x 8 significand bits represent an fp32 value exactly, K and V are bf16
// already, so every product is exact and only the fp32 accumulation rounds (DESIGN.md section 6
// "attention precision": a 2-way split left 2^-17 errors that flip E4M3 codes downstream);
// the online softmax is done in fp32 registers with warp shuffles across the 4 lanes of a row.
#pragma once
#include "ev_common.cuh"
#include "ev_elementwise.cuh"

namespace ev {

constexpr int ATT_THREADS = 256;
constexpr int ATT_WARPS = 8;
constexpr int ATT_CH = 64;  // keys per pipeline chunk

struct AttnArgs {
    const float* q;       // qkv buffer after RoPE; q head h of row m at q[m*q_ld + h*D]
    int q_ld, T, G, Hq, Hkv;
    const __nv_bfloat16* pool;  // this layer: [page][2][Hkv][page_size][D]
    const int32_t* page_table;  // [max_seqs][max_pages]
    int max_pages, page_size;
    const int32_t* seq_slots;   // [B]
    const int32_t* Lsnap;       // [B]
    const int32_t* nn_eff;      // [B]
    const int32_t* order;       // [B] grid z -> sequence (longest context first); null = identity
    const unsigned long long* anc;  // [B][T]
    int split_len;              // keys per split, multiple of ATT_CH
    int n_splits;               // grid.x
    float scale;                // 1/sqrt(D)
    float* o_part;              // [M][Hq][n_splits][D]
    float* ml_part;             // [M][Hq][n_splits][2]  (running max, running sum)
    unsigned long long* ts;     // bring-up: phase timestamps of CTA (0,0,0), or null
};

__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_trans(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
// D(16x8, fp32) += A(16x16 bf16, row) * B(16x8 bf16, col)
__device__ __forceinline__ void mma_bf16(float* d, const uint32_t* a, uint32_t b0, uint32_t b1) {
    asm(
        "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// x = hi + mid + lo exactly (8 + 8 + 8 significand bits)
__device__ __forceinline__ void split3(float x0, float x1, uint32_t& hi, uint32_t& mid, uint32_t& lo) {
    const __nv_bfloat16 h0 = __float2bfloat16_rn(x0), h1 = __float2bfloat16_rn(x1);
    const float r0 = x0 - __bfloat162float(h0), r1 = x1 - __bfloat162float(h1);
    const __nv_bfloat16 m0 = __float2bfloat16_rn(r0), m1 = __float2bfloat16_rn(r1);
    const __nv_bfloat16 l0 = __float2bfloat16_rn(r0 - __bfloat162float(m0));
    const __nv_bfloat16 l1 = __float2bfloat16_rn(r1 - __bfloat162float(m1));
    hi = (uint32_t)__bfloat16_as_ushort(h0) | ((uint32_t)__bfloat16_as_ushort(h1) << 16);
    mid = (uint32_t)__bfloat16_as_ushort(m0) | ((uint32_t)__bfloat16_as_ushort(m1) << 16);
    lo = (uint32_t)__bfloat16_as_ushort(l0) | ((uint32_t)__bfloat16_as_ushort(l1) << 16);
}
__device__ __forceinline__ void cp_async16_zfill(void* smem_dst, const void* gsrc, bool valid) {
    const int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_u32(smem_dst)), "l"(gsrc), "r"(sz) : "memory");
}

#define ATS(i) do { if (a.ts && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && threadIdx.x == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t_)); a.ts[i] = t_; } } while (0)
template <int D>
__global__ void __launch_bounds__(ATT_THREADS, 1) tree_attn_partial_kernel(AttnArgs a) {
    pdl_launch_dependents();
    pdl_wait();
    ATS(0);
    constexpr int ROWB = D * 2;           // bytes per key row
    constexpr int CPR = ROWB / 16;        // 16-byte chunks per row
    constexpr int TILE = ATT_CH * ROWB;   // bytes per K (or V) tile
    constexpr int KT = D / 16;            // k-tiles of the Q.K^T contraction
    constexpr int QTILE = 16 * ROWB;      // one warp's 16 query rows, one bf16 part
    extern __shared__ __align__(128) uint8_t att_smem[];  // [2 stages][K tile | V tile] [warp][hi|mid|lo][16 rows]

    const int split = blockIdx.x;
    const int kvh = blockIdx.y % a.Hkv, rg = blockIdx.y / a.Hkv;
    const int b = blockIdx.z;
    const int nn = a.nn_eff[b];     // the three scalars are loaded together, before the first branch
    const int L = a.Lsnap[b];
    const int seq_slot = a.seq_slots[b];
    if (nn == 0) return;
    const int n_keys = L + nn;
    const int k_begin = split * a.split_len;
    if (k_begin >= n_keys) return;
    const int k_end = min(k_begin + a.split_len, n_keys);
    const int n_chunks = (k_end - k_begin + ATT_CH - 1) / ATT_CH;
    const int32_t* pt = a.page_table + (size_t)seq_slot * a.max_pages;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int R = a.T * a.G;
    const int rt = rg * ATT_WARPS + warp;
    const bool active = rt * 16 < R;
    const int row0 = rt * 16 + (lane >> 2), row1 = row0 + 8;
    const int node0 = row0 / a.G, g0 = row0 % a.G, node1 = row1 / a.G, g1 = row1 % a.G;
    const bool v0 = active && row0 < R && node0 < nn, v1 = active && row1 < R && node1 < nn;
    const unsigned long long anc0 = v0 ? a.anc[b * a.T + node0] : 0ull, anc1 = v1 ? a.anc[b * a.T + node1] : 0ull;

    // ---- Q rows -> this warp's shared-memory tiles, split hi/mid/lo (A operand, read by ldmatrix) ----
    const uint32_t qs = smem_u32(att_smem + 4 * TILE + warp * 3 * QTILE);
    {
        uint8_t* qsp = att_smem + 4 * TILE + warp * 3 * QTILE;
        const float* q0 = a.q + (size_t)(b * a.T + (v0 ? node0 : 0)) * a.q_ld + (size_t)(kvh * a.G + (v0 ? g0 : 0)) * D;
        const float* q1 = a.q + (size_t)(b * a.T + (v1 ? node1 : 0)) * a.q_ld + (size_t)(kvh * a.G + (v1 ? g1 : 0)) * D;
        const int r0 = lane >> 2, r1 = r0 + 8;
#pragma unroll
        for (int c8 = 0; c8 < D / 8; ++c8) {
            const int c = c8 * 8 + (lane & 3) * 2;
            const float2 x0 = v0 ? *reinterpret_cast<const float2*>(q0 + c) : make_float2(0.f, 0.f);
            const float2 x1 = v1 ? *reinterpret_cast<const float2*>(q1 + c) : make_float2(0.f, 0.f);
            uint32_t h, md, l;
            split3(x0.x, x0.y, h, md, l);
            const int o0 = r0 * ROWB + ((c8 ^ (r0 & 7)) * 16) + (lane & 3) * 4;
            *reinterpret_cast<uint32_t*>(qsp + o0) = h;
            *reinterpret_cast<uint32_t*>(qsp + QTILE + o0) = md;
            *reinterpret_cast<uint32_t*>(qsp + 2 * QTILE + o0) = l;
            split3(x1.x, x1.y, h, md, l);
            const int o1 = r1 * ROWB + ((c8 ^ (r1 & 7)) * 16) + (lane & 3) * 4;
            *reinterpret_cast<uint32_t*>(qsp + o1) = h;
            *reinterpret_cast<uint32_t*>(qsp + QTILE + o1) = md;
            *reinterpret_cast<uint32_t*>(qsp + 2 * QTILE + o1) = l;
        }
        __syncwarp();
    }
    ATS(1);

    // ---- page gather: chunk ch -> stage ----
    auto load_chunk = [&](int stage, int ch) {
        uint8_t* kt_s = att_smem + stage * 2 * TILE;
        uint8_t* vt_s = kt_s + TILE;
        const int kbase = k_begin + ch * ATT_CH;
        for (int i = threadIdx.x; i < ATT_CH * CPR; i += ATT_THREADS) {
            const int r = i / CPR, c = i % CPR;
            const int kidx = kbase + r;
            const bool ok = kidx < k_end;
            const int kk = ok ? kidx : k_begin;
            const size_t base = (size_t)pt[kk / a.page_size] * 2 * a.Hkv * a.page_size * D +
                                (size_t)kvh * a.page_size * D + (size_t)(kk % a.page_size) * D + (size_t)c * 8;
            const int so = r * ROWB + ((c ^ (r & 7)) * 16);
            cp_async16_zfill(kt_s + so, a.pool + base, ok);
            cp_async16_zfill(vt_s + so, a.pool + base + (size_t)a.Hkv * a.page_size * D, ok);
        }
    };

    float o[D / 8][4];
#pragma unroll
    for (int i = 0; i < D / 8; ++i) { o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f; }
    float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;

    load_chunk(0, 0);
    cp_async_commit();
    for (int ch = 0; ch < n_chunks; ++ch) {
        if (ch + 1 < n_chunks) {
            load_chunk((ch + 1) & 1, ch + 1);
            cp_async_commit();
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        __syncthreads();
        if (ch < 4) ATS(2 + 2 * ch);
        if (active) {
            const uint32_t ks = smem_u32(att_smem + (ch & 1) * 2 * TILE);
            const uint32_t vs = ks + TILE;
            const int kbase = k_begin + ch * ATT_CH;
            // ---- S = Q K^T (16 rows x 64 keys per warp) ----
            float s[ATT_CH / 8][4];
#pragma unroll
            for (int nt = 0; nt < ATT_CH / 8; ++nt) s[nt][0] = s[nt][1] = s[nt][2] = s[nt][3] = 0.f;
#pragma unroll
            for (int kp = 0; kp < KT / 2; ++kp) {
                uint32_t qa[2][3][4];  // [k-tile of the pair][hi|mid|lo][A fragment]
                {
                    const int r = ((lane >> 3) & 1) * 8 + (lane & 7);
#pragma unroll
                    for (int t = 0; t < 2; ++t) {
                        const int c = (2 * kp + t) * 2 + (lane >> 4);
                        const uint32_t ad = qs + r * ROWB + ((c ^ (r & 7)) * 16);
#pragma unroll
                        for (int part = 0; part < 3; ++part)
                            ldsm_x4(ad + part * QTILE, qa[t][part][0], qa[t][part][1], qa[t][part][2], qa[t][part][3]);
                    }
                }
#pragma unroll
                for (int nt4 = 0; nt4 < ATT_CH / 32; ++nt4) {  // four n-tiles at a time: four independent accumulator chains
                    uint32_t bk[4][4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int r = (nt4 * 4 + u) * 8 + (lane & 7);
                        const int c = kp * 4 + (lane >> 3);
                        ldsm_x4(ks + r * ROWB + ((c ^ (r & 7)) * 16), bk[u][0], bk[u][1], bk[u][2], bk[u][3]);
                    }
#pragma unroll
                    for (int part = 2; part >= 0; --part) {  // smallest parts first
#pragma unroll
                        for (int u = 0; u < 4; ++u) mma_bf16(s[nt4 * 4 + u], qa[0][part], bk[u][0], bk[u][1]);
#pragma unroll
                        for (int u = 0; u < 4; ++u) mma_bf16(s[nt4 * 4 + u], qa[1][part], bk[u][2], bk[u][3]);
                    }
                }
            }
            // ---- scale, mask, row max ----
            const bool need_mask = kbase + ATT_CH > L;  // chunk touches tree keys or the split end
            float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
            for (int nt = 0; nt < ATT_CH / 8; ++nt) {
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    float v = mul_rn(s[nt][e], a.scale);
                    if (need_mask) {
                        const int kidx = kbase + nt * 8 + (lane & 3) * 2 + (e & 1);
                        const unsigned long long am = (e < 2) ? anc0 : anc1;
                        const bool ok = kidx < k_end && (kidx < L || ((am >> (kidx - L)) & 1ull));
                        if (!ok) v = -INFINITY;
                    }
                    s[nt][e] = v;
                    if (e < 2) mx0 = fmaxf(mx0, v); else mx1 = fmaxf(mx1, v);
                }
            }
            mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1));
            mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
            mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1));
            mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
            const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);
            const float mu0 = (mn0 == -INFINITY) ? 0.f : mn0, mu1 = (mn1 == -INFINITY) ? 0.f : mn1;
            const float c0 = expf(m0 - mu0), c1 = expf(m1 - mu1);  // exp(-inf) = 0 on the first chunk
            m0 = mn0; m1 = mn1;
            l0 *= c0; l1 *= c1;
#pragma unroll
            for (int nt = 0; nt < ATT_CH / 8; ++nt) {
                s[nt][0] = expf(s[nt][0] - mu0); s[nt][1] = expf(s[nt][1] - mu0);
                s[nt][2] = expf(s[nt][2] - mu1); s[nt][3] = expf(s[nt][3] - mu1);
                l0 += s[nt][0] + s[nt][1];
                l1 += s[nt][2] + s[nt][3];
            }
            // ---- O += P V: the chunk's product is accumulated from zero inside the tensor core and added to
            // the running output with ONE rounded fp32 add per chunk (long chains of tensor-core accumulation
            // truncate: 16k keys in one chain cost ~2e-5 relative) ----
            float oc[D / 8][4];
#pragma unroll
            for (int i = 0; i < D / 8; ++i) { oc[i][0] = oc[i][1] = oc[i][2] = oc[i][3] = 0.f; }
#pragma unroll
            for (int kt2 = 0; kt2 < ATT_CH / 16; ++kt2) {
                uint32_t pp[3][4];  // hi | mid | lo
                split3(s[2 * kt2][0], s[2 * kt2][1], pp[0][0], pp[1][0], pp[2][0]);
                split3(s[2 * kt2][2], s[2 * kt2][3], pp[0][1], pp[1][1], pp[2][1]);
                split3(s[2 * kt2 + 1][0], s[2 * kt2 + 1][1], pp[0][2], pp[1][2], pp[2][2]);
                split3(s[2 * kt2 + 1][2], s[2 * kt2 + 1][3], pp[0][3], pp[1][3], pp[2][3]);
                const int r = kt2 * 16 + ((lane >> 3) & 1) * 8 + (lane & 7);
#pragma unroll
                for (int np2 = 0; np2 < D / 32; ++np2) {  // four n-tiles (32 dims) at a time: four independent chains
                    uint32_t bv[2][4];
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
                        const int c = (np2 * 2 + u) * 2 + (lane >> 4);
                        ldsm_x4_trans(vs + r * ROWB + ((c ^ (r & 7)) * 16), bv[u][0], bv[u][1], bv[u][2], bv[u][3]);
                    }
#pragma unroll
                    for (int part = 2; part >= 0; --part) {
#pragma unroll
                        for (int u = 0; u < 2; ++u) {
                            mma_bf16(oc[(np2 * 2 + u) * 2], pp[part], bv[u][0], bv[u][1]);
                            mma_bf16(oc[(np2 * 2 + u) * 2 + 1], pp[part], bv[u][2], bv[u][3]);
                        }
                    }
                }
            }
#pragma unroll
            for (int i = 0; i < D / 8; ++i) {
                o[i][0] = fmaf(o[i][0], c0, oc[i][0]); o[i][1] = fmaf(o[i][1], c0, oc[i][1]);
                o[i][2] = fmaf(o[i][2], c1, oc[i][2]); o[i][3] = fmaf(o[i][3], c1, oc[i][3]);
            }
        }
        if (ch < 4) ATS(3 + 2 * ch);
        __syncthreads();
    }
    if (!active) return;
    l0 += __shfl_xor_sync(0xffffffffu, l0, 1);
    l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
    l1 += __shfl_xor_sync(0xffffffffu, l1, 1);
    l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
    if (row0 < R) {
        const size_t pi = ((size_t)(b * a.T + node0) * a.Hq + kvh * a.G + g0) * a.n_splits + split;
        float* op = a.o_part + pi * D + (lane & 3) * 2;
#pragma unroll
        for (int i = 0; i < D / 8; ++i) *reinterpret_cast<float2*>(op + i * 8) = make_float2(o[i][0], o[i][1]);
        if ((lane & 3) == 0) *reinterpret_cast<float2*>(a.ml_part + pi * 2) = make_float2(m0, l0);
    }
    if (row1 < R) {
        const size_t pi = ((size_t)(b * a.T + node1) * a.Hq + kvh * a.G + g1) * a.n_splits + split;
        float* op = a.o_part + pi * D + (lane & 3) * 2;
#pragma unroll
        for (int i = 0; i < D / 8; ++i) *reinterpret_cast<float2*>(op + i * 8) = make_float2(o[i][2], o[i][3]);
        if ((lane & 3) == 0) *reinterpret_cast<float2*>(a.ml_part + pi * 2) = make_float2(m1, l1);
    }
    ATS(10);
}

// ---- merge of the key splits (fixed order 0..ns-1) + per-token absmax + E4M3 quantize -----------
// One CTA of 512 threads per token.  Phase 1 stages the (max, sum) pairs of all heads x splits in shared
// memory, phase 2 turns them into softmax weights w[h][s] = exp(m_s - max) and the denominator per head,
// phase 3 forms out = (sum_s w_s O_s) / den with all S partial loads of a thread in flight at once; the
// merged row stays in registers for the quantizer.
struct MergeArgs {
    int T, Hq, D, n_splits, split_len;
    const int32_t* Lsnap;
    const int32_t* nn_eff;
    const float* o_part;
    const float* ml_part;
    float* attn;   // optional [M][Hq*D] fp32 merged output (debug tap) or null
    QuantOut q;
    L2Prefetch pf;
};
constexpr int MERGE_THREADS = 256;   // = ROW_THREADS (ev_elementwise.cuh): Hq * D <= 4 * 256 * NV4 * cluster size
template <int MERGE_NV4>
__global__ void __launch_bounds__(MERGE_THREADS) attn_merge_quant_kernel(MergeArgs a) {
    pdl_launch_dependents();  // the O-projection GEMM may start prefetching its weights now
    l2_prefetch_issue(a.pf);
    pdl_wait();
    trace_past_wait(a.pf);
    extern __shared__ float msm[];             // w[Hq][S] | l[Hq][S] | den[Hq]
    __shared__ float red[MERGE_THREADS / 32];
    __shared__ float xch_f[CLUSTER_MAX];
    const int m = blockIdx.x / cluster_nctarank();   // one token row per cluster
    const int b = m / a.T, node = m % a.T;
    const int nn = a.nn_eff[b];
    const int K = a.Hq * a.D, S = a.n_splits;
    const bool valid = node < nn;
    const int ns = valid ? (a.Lsnap[b] + nn + a.split_len - 1) / a.split_len : 0;
    float* w = msm;
    float* ls = msm + a.Hq * S;
    float* den = ls + a.Hq * S;
    // The partial outputs of the first NB splits are requested BEFORE the split weights are computed (they only need
    // ns): the (max, sum) round trip, the two CTA barriers and the exps then run under the loads instead of in front
    // of them.  One float4 per thread (few tokens, rows spread over a cluster): 12 splits in flight; else 4.
    constexpr int NB = MERGE_NV4 == 1 ? 12 : 4;
    float4 v[MERGE_NV4];
    int c0, c1;
    cluster_cols(K / 4, c0, c1);
    float4 t0[NB];
    {
        const int i4 = c0 + threadIdx.x;
        const int i = i4 * 4;
        if (i4 < c1 && valid) {
            const float* op = a.o_part + ((size_t)m * a.Hq + i / a.D) * S * a.D + i % a.D;
#pragma unroll
            for (int u = 0; u < NB; ++u)
                if (u < ns) t0[u] = __ldcg(reinterpret_cast<const float4*>(op + (size_t)u * a.D));
        }
    }
    for (int i = threadIdx.x; i < a.Hq * S; i += MERGE_THREADS) {
        const int h = i / S, sp = i % S;
        float2 ml = make_float2(-INFINITY, 0.f);
        if (sp < ns) ml = __ldcg(reinterpret_cast<const float2*>(a.ml_part + (((size_t)m * a.Hq + h) * S + sp) * 2));
        w[i] = ml.x;
        ls[i] = ml.y;
    }
    __syncthreads();
    if ((int)threadIdx.x < a.Hq) {
        const int h = threadIdx.x;
        float mx = -INFINITY;
        for (int sp = 0; sp < ns; ++sp) mx = fmaxf(mx, w[h * S + sp]);
        float d = 0.f;
        for (int sp = 0; sp < ns; ++sp) {
            const float ms = w[h * S + sp];
            const float wt = (ms == -INFINITY) ? 0.f : expf(ms - mx);
            w[h * S + sp] = wt;
            d += wt * ls[h * S + sp];
        }
        den[h] = d;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < MERGE_NV4; ++k) {
        const int i4 = c0 + threadIdx.x + k * MERGE_THREADS;
        const int i = i4 * 4;
        v[k] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (i4 < c1 && valid) {
            const int h = i / a.D, d = i % a.D;
            const float* op = a.o_part + ((size_t)m * a.Hq + h) * S * a.D + d;
            float4 num = make_float4(0.f, 0.f, 0.f, 0.f);
            int s_done = 0;
            if (k == 0) {   // the splits requested up front
#pragma unroll
                for (int u = 0; u < NB; ++u)
                    if (u < ns) {
                        const float wt = w[h * S + u];
                        num.x += wt * t0[u].x; num.y += wt * t0[u].y; num.z += wt * t0[u].z; num.w += wt * t0[u].w;
                    }
                s_done = NB;
            }
            for (int s0 = s_done; s0 < ns; s0 += 4) {   // splits are added in index order, whatever the batching
                float4 t[4];
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (s0 + u < ns) t[u] = __ldcg(reinterpret_cast<const float4*>(op + (size_t)(s0 + u) * a.D));
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (s0 + u < ns) {
                        const float wt = w[h * S + s0 + u];
                        num.x += wt * t[u].x; num.y += wt * t[u].y; num.z += wt * t[u].z; num.w += wt * t[u].w;
                    }
            }
            const float dn = den[h];
            v[k] = make_float4(div_rn(num.x, dn), div_rn(num.y, dn), div_rn(num.z, dn), div_rn(num.w, dn));
        }
        if (i4 < c1 && a.attn) *reinterpret_cast<float4*>(a.attn + (size_t)m * K + i) = v[k];
    }
    quantize_regs<MERGE_NV4>(v, m, K, c0, c1, a.q, red, xch_f);
    trace_exit(a.pf);
}

}  // namespace ev
