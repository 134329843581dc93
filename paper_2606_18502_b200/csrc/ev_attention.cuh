// K5: tree-masked GQA attention over the paged bf16 KV cache ("tree attention";
// BASELINE.json:north_star (2)), + K7: merge fused with the per-token absmax / E4M3 quantization that feeds
// the O projection.
//
// Batch-invariant reduction order (speculative verification must emit exactly what plain decoding
// emits, so a node's attention output may not depend on the tree or batch it is verified in).  A node at position
// p = L + depth attends to positions [0, p].  The key set is cut the same way wherever the node appears:
//   BULK  = positions [0, p - ATT_TAIL_R), in CHUNKS of `chunk` keys aligned to absolute positions (chunk j = keys
//           [j chunk, (j+1) chunk)); each chunk is an online softmax over 64-key tiles from a fresh state, on the tensor
//           cores (tree_attn_tc_kernel, or tree_attn_partial_kernel below for page sizes other than 16);
//   TAIL  = the last ATT_TAIL_R + 1 positions (youngest cached tokens, then the node's nearest ancestors in depth
//           order, itself last), scored key by key in fp32 by the merge kernel;
//   MERGE = out = (sum_j w_j O_j + sum_t e_t v_t) / (sum_j w_j l_j + sum_t e_t), chunks in index order, then the tail
//           keys in position order, w_j = exp(m_j - M), e_t = exp(s_t - M) (ex2.approx), M = the overall maximum; the division is a
//           correctly rounded reciprocal and a multiply.
// For trees no deeper than ATT_TAIL_R the bulk lies inside the committed context: which tree slots the ancestors sit
// in, how many nodes and sequences share the launch and how many CTAs there are no longer enter the arithmetic.
// Deeper trees (prefill chains) put the older ancestors into the bulk by slot (anc_bulk); chains stay invariant
// because a chain's slots are its positions.
//
// tree_attn_partial_kernel: one CTA = (sequence b, kv head, group of 8 row tiles, chunk).  The query rows of one kv
// head are the T nodes x G query heads that share it (row = node*G + g), 16 rows per warp.  Pages are gathered with
// 16-byte cp.async into XOR-swizzled shared memory (each (page, K|V, head) block is page_size*D*2 contiguous bytes),
// double buffered; Q.K^T and P.V run on the tensor cores (mma.sync m16n8k16 bf16, fp32 accumulate) with Q and P each
// split into hi + mid + lo bf16 parts: 3 x 8 significand bits represent an fp32 value exactly, K and V are bf16
// already, so every product is exact and only the fp32 accumulation rounds; the online softmax is done in fp32
// registers with warp shuffles across the 4 lanes of a row.
#pragma once
#include <cuda_fp16.h>
#include "ev_common.cuh"
#include "ev_elementwise.cuh"

namespace ev {

constexpr int ATT_THREADS = 256;
constexpr int ATT_WARPS = 8;
constexpr int ATT_CH = 64;  // keys per pipeline tile

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
    const unsigned long long* anc_bulk;  // [B][T] tree slots among the row's bulk keys (tree_prep_kernel)
    const int32_t* erow;        // [B][T] cached positions below erow[row] are bulk keys of the row
    const int32_t* kend_seq;    // [B] one past the last bulk key slot of the sequence
    int chunk;                  // keys per chunk, multiple of ATT_CH: a constant of the model, NOT a function of the batch
    int n_chunks;               // chunks the grid covers; stride of the partial arrays
    int cpg;                    // consecutive chunks one CTA walks (grid.x = ceil(n_chunks / cpg)); a scheduling choice, no effect on results
    float scale;                // 1/sqrt(D)
    float* o_part;              // [M][Hq][n_chunks][D]
    float* ml_part;             // [M][Hq][n_chunks][2]  (running max, running sum)
};
// bulk membership of key slot kidx for a row (erow e, tree bits ab) of a sequence with L cached tokens
__device__ __forceinline__ bool bulk_key(int kidx, int L, int e, unsigned long long ab) {
    return kidx < L ? kidx < e : (kidx - L < 64 && ((ab >> (kidx - L)) & 1ull));
}

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

template <int D>
__global__ void __launch_bounds__(ATT_THREADS, 1) tree_attn_partial_kernel(AttnArgs a) {
    pdl_launch_dependents();
    pdl_wait();
    constexpr int ROWB = D * 2;           // bytes per key row
    constexpr int CPR = ROWB / 16;        // 16-byte chunks per row
    constexpr int TILE = ATT_CH * ROWB;   // bytes per K (or V) tile
    constexpr int KT = D / 16;            // k-tiles of the Q.K^T contraction
    constexpr int QTILE = 16 * ROWB;      // one warp's 16 query rows, one bf16 part
    extern __shared__ __align__(128) uint8_t att_smem[];  // [2 stages][K tile | V tile] [warp][hi|mid|lo][16 rows]

    const int split = blockIdx.x;
    const int kvh = blockIdx.y % a.Hkv, rg = blockIdx.y / a.Hkv;
    const int b = blockIdx.z;
    const int nn = a.nn_eff[b];     // the scalars are loaded together, before the first branch
    const int L = a.Lsnap[b];
    const int seq_slot = a.seq_slots[b];
    const int n_keys = a.kend_seq[b];
    if (nn == 0) return;
    const int k_begin = split * a.chunk;   // this kernel: one chunk per CTA (cpg == 1)
    if (k_begin >= n_keys) return;
    const int k_end = min(k_begin + a.chunk, n_keys);
    const int n_chunks = (k_end - k_begin + ATT_CH - 1) / ATT_CH;
    const int32_t* pt = a.page_table + (size_t)seq_slot * a.max_pages;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int R = a.T * a.G;
    const int rt = rg * ATT_WARPS + warp;
    const bool active = rt * 16 < R;
    const int row0 = rt * 16 + (lane >> 2), row1 = row0 + 8;
    const int node0 = row0 / a.G, g0 = row0 % a.G, node1 = row1 / a.G, g1 = row1 % a.G;
    const bool v0 = active && row0 < R && node0 < nn, v1 = active && row1 < R && node1 < nn;
    const unsigned long long anc0 = v0 ? a.anc_bulk[b * a.T + node0] : 0ull, anc1 = v1 ? a.anc_bulk[b * a.T + node1] : 0ull;
    const int e0 = v0 ? a.erow[b * a.T + node0] : 0, e1 = v1 ? a.erow[b * a.T + node1] : 0;

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
            const bool need_mask = kbase + ATT_CH > L - ATT_TAIL_R;  // tile reaches the end of some row's bulk
            float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
            for (int nt = 0; nt < ATT_CH / 8; ++nt) {
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    float v = mul_rn(s[nt][e], a.scale);
                    if (need_mask) {
                        const int kidx = kbase + nt * 8 + (lane & 3) * 2 + (e & 1);
                        const bool ok = kidx < k_end && bulk_key(kidx, L, (e < 2) ? e0 : e1, (e < 2) ? anc0 : anc1);
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
        __syncthreads();
    }
    if (!active) return;
    l0 += __shfl_xor_sync(0xffffffffu, l0, 1);
    l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
    l1 += __shfl_xor_sync(0xffffffffu, l1, 1);
    l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
    if (row0 < R) {
        const size_t pi = ((size_t)(b * a.T + node0) * a.Hq + kvh * a.G + g0) * a.n_chunks + split;
        float* op = a.o_part + pi * D + (lane & 3) * 2;
#pragma unroll
        for (int i = 0; i < D / 8; ++i) *reinterpret_cast<float2*>(op + i * 8) = make_float2(o[i][0], o[i][1]);
        if ((lane & 3) == 0) *reinterpret_cast<float2*>(a.ml_part + pi * 2) = make_float2(m0, l0);
    }
    if (row1 < R) {
        const size_t pi = ((size_t)(b * a.T + node1) * a.Hq + kvh * a.G + g1) * a.n_chunks + split;
        float* op = a.o_part + pi * D + (lane & 3) * 2;
#pragma unroll
        for (int i = 0; i < D / 8; ++i) *reinterpret_cast<float2*>(op + i * 8) = make_float2(o[i][2], o[i][3]);
        if ((lane & 3) == 0) *reinterpret_cast<float2*>(a.ml_part + pi * 2) = make_float2(m1, l1);
    }
}

// ---- tail keys + merge of the chunks (fixed order) + per-token absmax + E4M3 quantize ---------------
// One cluster of MERGE_THREADS-thread CTAs per token row; a thread owns float4s of the row, i.e. 4 output dims of one
// query head, and the D/4 consecutive lanes that share a head form one reduction group (aligned: the CTA's first
// float4 is a multiple of 32).  Per head: (1) the tail keys - cached slots [erow, L) then the row's own ancestors in
// the tail, in position order - are scored in fp32: partial dot of 4 dims per lane (one fixed FMA chain), xor-butterfly
// over the group (every lane ends with the same bits), times 1/sqrt(d); (2) the chunk partials (max, sum, O) of the
// bulk are read in chunk order; (3) out = (sum_j w_j O_j + sum_t e_t v_t) / (sum_j w_j l_j + sum_t e_t).  The merged
// row stays in registers for the quantizer.  Nothing here depends on the cluster size or on how many rows there are.
constexpr int ATT_TAIL_MAX = ATT_TAIL_R + 1;
struct MergeArgs {
    int T, Hq, Hkv, D, n_chunks, chunk;
    const int32_t* Lsnap;
    const int32_t* nn_eff;
    const int32_t* seq_slots;
    const int32_t* erow;
    const int32_t* kend_row;
    const unsigned long long* anc;
    const unsigned long long* anc_bulk;
    const float* o_part;
    const float* ml_part;
    const float* qkv;      // rotated q (fp32): head h of row m at qkv[m * q_ld + h * D]
    int q_ld;
    const __nv_bfloat16* pool;   // this layer
    const int32_t* page_table;
    int max_pages, page_size, kv_f16;
    const uint8_t* pool8;   // FP8 KV cache: this layer's pool as E4M3 codes (kv_dtype 1), or null
    float k_scale, v_scale; // its static scales: value = fp32(decode(code) * s)
    float scale;
    float* attn;   // optional [M][Hq*D] fp32 merged output (debug tap) or null
    QuantOut q;
    L2Prefetch pf;
};
constexpr int MERGE_THREADS = 256;   // = ROW_THREADS (ev_elementwise.cuh): Hq * D <= 4 * 256 * NV4 * cluster size
__device__ __forceinline__ float4 kv_cvt4_e4m3(uint32_t w, float s) {   // 4 E4M3 codes -> fp32(decode(code) * s)
    const __half2_raw lo = __nv_cvt_fp8x2_to_halfraw2((__nv_fp8x2_storage_t)(w & 0xFFFFu), __NV_E4M3);
    const __half2_raw hi = __nv_cvt_fp8x2_to_halfraw2((__nv_fp8x2_storage_t)(w >> 16), __NV_E4M3);
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&lo)), b = __half22float2(*reinterpret_cast<const __half2*>(&hi));
    return make_float4(mul_rn(a.x, s), mul_rn(a.y, s), mul_rn(b.x, s), mul_rn(b.y, s));
}
__device__ __forceinline__ float4 kv_cvt4(uint2 w, int kv_f16) {   // 4 consecutive K or V elements (raw pool bits) as fp32
    if (kv_f16) {
        const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&w.x)), b = __half22float2(*reinterpret_cast<const __half2*>(&w.y));
        return make_float4(a.x, a.y, b.x, b.y);
    }
    return make_float4(__uint_as_float(w.x << 16), __uint_as_float(w.x & 0xFFFF0000u), __uint_as_float(w.y << 16), __uint_as_float(w.y & 0xFFFF0000u));
}
template <int MERGE_NV4>
__global__ void __launch_bounds__(MERGE_THREADS, 2) attn_merge_quant_kernel(MergeArgs a) {
    pdl_launch_dependents();  // the O-projection GEMM may start prefetching its weights now
    l2_prefetch_issue(a.pf);
    // The row's key plan (tree_prep_kernel's output, complete before any kernel of the step starts: ev_api.cu
    // serial_next_launch) and the page lookups of its tail keys come BEFORE griddepcontrol.wait: three dependent L2 round
    // trips that used to sit between the wait and the first K/V load.  __ldcg: no stale L1 line of the previous step.
    __shared__ float red[MERGE_THREADS / 32];
    __shared__ float xch_f[CLUSTER_MAX];
    __shared__ long long tbase[ATT_TAIL_MAX];   // element offset of the tail key's K row (kv head 0, dim 0) in this layer's pool
    const int m = blockIdx.x / cluster_nctarank();   // one token row per cluster
    const int b = m / a.T, node = m % a.T;
    const int nn = __ldcg(a.nn_eff + b);
    const int K = a.Hq * a.D, S = a.n_chunks, D = a.D;
    const bool valid = node < nn;
    const int L = __ldcg(a.Lsnap + b);
    const int e = valid ? __ldcg(a.erow + m) : 0;
    const int ns = valid ? (__ldcg(a.kend_row + m) + a.chunk - 1) / a.chunk : 0;
    // tail keys, in position order: n_ctx cached slots e .. L-1, then the ancestors of the tail (lowest node index = lowest depth first)
    const int n_ctx = valid ? min(max(0, L - e), ATT_TAIL_MAX) : 0;
    const unsigned long long anc_tail = valid ? (__ldcg(a.anc + m) & ~__ldcg(a.anc_bulk + m)) : 0ull;
    const int nt = min(n_ctx + __popcll(anc_tail), ATT_TAIL_MAX);
    const size_t kv_stride = (size_t)a.Hkv * a.page_size * D;   // K block -> V block of a page
    if ((int)threadIdx.x < nt) {
        const int u = threadIdx.x;
        int sl = e + u;
        if (u >= n_ctx) {   // the (u - n_ctx)-th set bit of anc_tail
            unsigned long long at = anc_tail;
            for (int i = n_ctx; i < u; ++i) at &= at - 1;
            sl = L + __ffsll((long long)at) - 1;
        }
        const int32_t* pt = a.page_table + (size_t)__ldcg(a.seq_slots + b) * a.max_pages;
        tbase[u] = (long long)((size_t)pt[sl / a.page_size] * 2 * kv_stride + (size_t)(sl % a.page_size) * D);
    }
    __syncthreads();
    pdl_wait();
    trace_past_wait(a.pf);
    const int G = a.Hq / a.Hkv;
    const int gl = D / 4;   // lanes per head group (32 or 16)
    float4 v[MERGE_NV4];
    int c0, c1;
    cluster_cols(K / 4, c0, c1);
#pragma unroll
    for (int k = 0; k < MERGE_NV4; ++k) {
        const int i4 = c0 + threadIdx.x + k * MERGE_THREADS;
        const int i = i4 * 4;
        v[k] = make_float4(0.f, 0.f, 0.f, 0.f);
        const bool on = i4 < c1 && valid;      // uniform over a head group (D / 4 lanes, aligned)
        const int h = on ? i / D : 0, d = on ? i % D : 0;
        const float* op = a.o_part + ((size_t)m * a.Hq + h) * S * D + d;
        const float* mlp = a.ml_part + ((size_t)m * a.Hq + h) * S * 2;
        // every load of this float4 is requested before the first use: chunk partials, q, the tail keys' K and V
        constexpr int NB = 4;
        float4 t0[NB];
        float2 ml0[NB];
        uint2 kr[ATT_TAIL_MAX], vr[ATT_TAIL_MAX];
        float4 q4 = make_float4(0.f, 0.f, 0.f, 0.f);
        const size_t hoff = (size_t)(h / G) * a.page_size * D + d;
#pragma unroll
        for (int u = 0; u < ATT_TAIL_MAX; ++u) {
            kr[u] = make_uint2(0u, 0u); vr[u] = make_uint2(0u, 0u);
            if (on && u < nt) {
                if (a.pool8) {   // one byte per element: 4 codes in the low word
                    const uint8_t* kp = a.pool8 + tbase[u] + hoff;
                    kr[u].x = *reinterpret_cast<const uint32_t*>(kp);
                    vr[u].x = *reinterpret_cast<const uint32_t*>(kp + kv_stride);
                } else {
                    const __nv_bfloat16* kp = a.pool + tbase[u] + hoff;
                    kr[u] = *reinterpret_cast<const uint2*>(kp);              // L1-cached: the G query heads of a kv head read the same rows
                    vr[u] = *reinterpret_cast<const uint2*>(kp + kv_stride);
                }
            }
        }
        if (on) q4 = *reinterpret_cast<const float4*>(a.qkv + (size_t)m * a.q_ld + i);
#pragma unroll
        for (int u = 0; u < NB; ++u)
            if (on && u < ns) { t0[u] = __ldcg(reinterpret_cast<const float4*>(op + (size_t)u * D)); ml0[u] = __ldcg(reinterpret_cast<const float2*>(mlp + 2 * u)); }
        // (1) tail scores: fixed FMA chain over the lane's 4 dims, xor butterfly over the head group, times 1/sqrt(d)
        float ts[ATT_TAIL_MAX];
#pragma unroll
        for (int u = 0; u < ATT_TAIL_MAX; ++u) {
            const float4 k4 = a.pool8 ? kv_cvt4_e4m3(kr[u].x, a.k_scale) : kv_cvt4(kr[u], a.kv_f16);
            float part = fmaf(q4.w, k4.w, fmaf(q4.z, k4.z, fmaf(q4.y, k4.y, __fmul_rn(q4.x, k4.x))));
            for (int o = gl >> 1; o > 0; o >>= 1) part = __fadd_rn(part, __shfl_xor_sync(0xffffffffu, part, o));
            ts[u] = mul_rn(part, a.scale);
        }
        if (on) {
            // (2) overall maximum: chunk maxima, then tail scores
            float mx = -INFINITY;
#pragma unroll
            for (int u = 0; u < NB; ++u)
                if (u < ns) mx = fmaxf(mx, ml0[u].x);
            for (int j = NB; j < ns; ++j) mx = fmaxf(mx, __ldcg(mlp + 2 * j));
#pragma unroll
            for (int u = 0; u < ATT_TAIL_MAX; ++u)
                if (u < nt) mx = fmaxf(mx, ts[u]);
            // (3) weighted sums, chunks in index order then the tail in position order
            float den = 0.f;
            float4 num = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
            for (int u = 0; u < NB; ++u)
                if (u < ns) {
                    const float wt = (ml0[u].x == -INFINITY) ? 0.f : exp_fast(ml0[u].x - mx);
                    den = fmaf(wt, ml0[u].y, den);
                    num.x = fmaf(wt, t0[u].x, num.x); num.y = fmaf(wt, t0[u].y, num.y); num.z = fmaf(wt, t0[u].z, num.z); num.w = fmaf(wt, t0[u].w, num.w);
                }
            for (int s0 = NB; s0 < ns; s0 += 4) {
                float4 t[4];
                float2 ml[4];
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (s0 + u < ns) { t[u] = __ldcg(reinterpret_cast<const float4*>(op + (size_t)(s0 + u) * D)); ml[u] = __ldcg(reinterpret_cast<const float2*>(mlp + 2 * (s0 + u))); }
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (s0 + u < ns) {
                        const float wt = (ml[u].x == -INFINITY) ? 0.f : exp_fast(ml[u].x - mx);
                        den = fmaf(wt, ml[u].y, den);
                        num.x = fmaf(wt, t[u].x, num.x); num.y = fmaf(wt, t[u].y, num.y); num.z = fmaf(wt, t[u].z, num.z); num.w = fmaf(wt, t[u].w, num.w);
                    }
            }
#pragma unroll
            for (int u = 0; u < ATT_TAIL_MAX; ++u)
                if (u < nt) {
                    const float et = exp_fast(ts[u] - mx);
                    const float4 v4 = a.pool8 ? kv_cvt4_e4m3(vr[u].x, a.v_scale) : kv_cvt4(vr[u], a.kv_f16);
                    den = __fadd_rn(den, et);
                    num.x = fmaf(et, v4.x, num.x); num.y = fmaf(et, v4.y, num.y); num.z = fmaf(et, v4.z, num.z); num.w = fmaf(et, v4.w, num.w);
                }
            const float inv = __frcp_rn(den);   // one correctly rounded reciprocal, four rounded multiplies
            v[k] = make_float4(mul_rn(num.x, inv), mul_rn(num.y, inv), mul_rn(num.z, inv), mul_rn(num.w, inv));
            if (a.attn) *reinterpret_cast<float4*>(a.attn + (size_t)m * K + i) = v[k];
        }
    }
    quantize_regs<MERGE_NV4>(v, m, K, c0, c1, a.q, red, xch_f);
    trace_exit(a.pf);
}

// ---- the same computation for many rows (D = 128, one CTA per row, no cluster): warp = one kv head, lane = 4 output dims.
// The tail keys' K and V are loaded ONCE per kv head and shared by its G query heads (the generic kernel above loads them
// per query head), every load of the warp's G heads is issued before the first use, and a thread ends up holding G float4s
// of the row for the quantizer.  Same arithmetic, same order per (row, head): results are bit-identical to the generic
// kernel (tests/test_gpu_verify_tiny.py runs D = 64 through the generic one, the 8B tests run both). ----
template <int G>
__global__ void __launch_bounds__(256, 2) attn_merge_rowkv_kernel(MergeArgs a) {
    pdl_launch_dependents();
    l2_prefetch_issue(a.pf);
    constexpr int D = 128;
    __shared__ float red[8];
    __shared__ long long tbase[ATT_TAIL_MAX];
    // key plan and page lookups before griddepcontrol.wait (see attn_merge_quant_kernel)
    const int m = blockIdx.x;
    const int b = m / a.T, node = m % a.T;
    const int nn = __ldcg(a.nn_eff + b);
    const int K = a.Hq * D, S = a.n_chunks;
    const bool valid = node < nn;
    const int L = __ldcg(a.Lsnap + b);
    const int e = valid ? __ldcg(a.erow + m) : 0;
    const int ns = valid ? (__ldcg(a.kend_row + m) + a.chunk - 1) / a.chunk : 0;
    const int n_ctx = valid ? min(max(0, L - e), ATT_TAIL_MAX) : 0;
    const unsigned long long anc_tail = valid ? (__ldcg(a.anc + m) & ~__ldcg(a.anc_bulk + m)) : 0ull;
    const int nt = min(n_ctx + __popcll(anc_tail), ATT_TAIL_MAX);
    const size_t kv_stride = (size_t)a.Hkv * a.page_size * D;
    if ((int)threadIdx.x < nt) {
        const int u = threadIdx.x;
        int sl = e + u;
        if (u >= n_ctx) {
            unsigned long long at = anc_tail;
            for (int i = n_ctx; i < u; ++i) at &= at - 1;
            sl = L + __ffsll((long long)at) - 1;
        }
        const int32_t* pt = a.page_table + (size_t)__ldcg(a.seq_slots + b) * a.max_pages;
        tbase[u] = (long long)((size_t)pt[sl / a.page_size] * 2 * kv_stride + (size_t)(sl % a.page_size) * D);
    }
    __syncthreads();
    pdl_wait();
    trace_past_wait(a.pf);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int kvh = warp;                 // blockDim = 32 * Hkv
    const int d = lane * 4;
    float4 v[G];
    float amax = 0.f;
    {
        // every load of this warp, up front
        uint2 kr[ATT_TAIL_MAX], vr[ATT_TAIL_MAX];
        const size_t hoff = (size_t)kvh * a.page_size * D + d;
#pragma unroll
        for (int u = 0; u < ATT_TAIL_MAX; ++u) {
            kr[u] = make_uint2(0u, 0u); vr[u] = make_uint2(0u, 0u);
            if (valid && u < nt) {
                if (a.pool8) {
                    const uint8_t* kp = a.pool8 + tbase[u] + hoff;
                    kr[u].x = *reinterpret_cast<const uint32_t*>(kp);
                    vr[u].x = *reinterpret_cast<const uint32_t*>(kp + kv_stride);
                } else {
                    const __nv_bfloat16* kp = a.pool + tbase[u] + hoff;
                    kr[u] = *reinterpret_cast<const uint2*>(kp);
                    vr[u] = *reinterpret_cast<const uint2*>(kp + kv_stride);
                }
            }
        }
        constexpr int NB = 2;
        float4 q4[G], t0[G][NB];
        float2 ml0[G][NB];
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const int h = kvh * G + g;
            q4[g] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (valid) q4[g] = *reinterpret_cast<const float4*>(a.qkv + (size_t)m * a.q_ld + h * D + d);
#pragma unroll
            for (int u = 0; u < NB; ++u)
                if (valid && u < ns) {
                    t0[g][u] = __ldcg(reinterpret_cast<const float4*>(a.o_part + (((size_t)m * a.Hq + h) * S + u) * D + d));
                    ml0[g][u] = __ldcg(reinterpret_cast<const float2*>(a.ml_part + (((size_t)m * a.Hq + h) * S + u) * 2));
                }
        }
        float4 kf[ATT_TAIL_MAX];
#pragma unroll
        for (int u = 0; u < ATT_TAIL_MAX; ++u) kf[u] = a.pool8 ? kv_cvt4_e4m3(kr[u].x, a.k_scale) : kv_cvt4(kr[u], a.kv_f16);
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const int h = kvh * G + g;
            const float* op = a.o_part + ((size_t)m * a.Hq + h) * S * D + d;
            const float* mlp = a.ml_part + ((size_t)m * a.Hq + h) * S * 2;
            float ts[ATT_TAIL_MAX];
#pragma unroll
            for (int u = 0; u < ATT_TAIL_MAX; ++u) {
                float part = fmaf(q4[g].w, kf[u].w, fmaf(q4[g].z, kf[u].z, fmaf(q4[g].y, kf[u].y, __fmul_rn(q4[g].x, kf[u].x))));
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) part = __fadd_rn(part, __shfl_xor_sync(0xffffffffu, part, o));
                ts[u] = mul_rn(part, a.scale);
            }
            v[g] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (valid) {
                float mx = -INFINITY;
#pragma unroll
                for (int u = 0; u < NB; ++u)
                    if (u < ns) mx = fmaxf(mx, ml0[g][u].x);
                for (int j = NB; j < ns; ++j) mx = fmaxf(mx, __ldcg(mlp + 2 * j));
#pragma unroll
                for (int u = 0; u < ATT_TAIL_MAX; ++u)
                    if (u < nt) mx = fmaxf(mx, ts[u]);
                float den = 0.f;
                float4 num = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                for (int u = 0; u < NB; ++u)
                    if (u < ns) {
                        const float wt = (ml0[g][u].x == -INFINITY) ? 0.f : exp_fast(ml0[g][u].x - mx);
                        den = fmaf(wt, ml0[g][u].y, den);
                        num.x = fmaf(wt, t0[g][u].x, num.x); num.y = fmaf(wt, t0[g][u].y, num.y); num.z = fmaf(wt, t0[g][u].z, num.z); num.w = fmaf(wt, t0[g][u].w, num.w);
                    }
                for (int s0 = NB; s0 < ns; s0 += 4) {
                    float4 t[4];
                    float2 ml[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u)
                        if (s0 + u < ns) { t[u] = __ldcg(reinterpret_cast<const float4*>(op + (size_t)(s0 + u) * D)); ml[u] = __ldcg(reinterpret_cast<const float2*>(mlp + 2 * (s0 + u))); }
#pragma unroll
                    for (int u = 0; u < 4; ++u)
                        if (s0 + u < ns) {
                            const float wt = (ml[u].x == -INFINITY) ? 0.f : exp_fast(ml[u].x - mx);
                            den = fmaf(wt, ml[u].y, den);
                            num.x = fmaf(wt, t[u].x, num.x); num.y = fmaf(wt, t[u].y, num.y); num.z = fmaf(wt, t[u].z, num.z); num.w = fmaf(wt, t[u].w, num.w);
                        }
                }
#pragma unroll
                for (int u = 0; u < ATT_TAIL_MAX; ++u)
                    if (u < nt) {
                        const float et = exp_fast(ts[u] - mx);
                        const float4 v4 = a.pool8 ? kv_cvt4_e4m3(vr[u].x, a.v_scale) : kv_cvt4(vr[u], a.kv_f16);
                        den = __fadd_rn(den, et);
                        num.x = fmaf(et, v4.x, num.x); num.y = fmaf(et, v4.y, num.y); num.z = fmaf(et, v4.z, num.z); num.w = fmaf(et, v4.w, num.w);
                    }
                const float inv = __frcp_rn(den);
                v[g] = make_float4(mul_rn(num.x, inv), mul_rn(num.y, inv), mul_rn(num.z, inv), mul_rn(num.w, inv));
                if (a.attn) *reinterpret_cast<float4*>(a.attn + (size_t)m * K + h * D + d) = v[g];
            }
            amax = fmaxf(amax, fmaxf(fmaxf(fabsf(v[g].x), fabsf(v[g].y)), fmaxf(fabsf(v[g].z), fabsf(v[g].w))));
        }
    }
    // per-token quantization of the row (the tail of quantize_regs for this thread layout)
    amax = block_max(amax, red);
    const QuantOut& q = a.q;
    float s;
    if (q.static_scale) s = *q.static_scale;
    else s = (amax == 0.f) ? 1.0f : div_rn(amax, 448.0f);
    if (threadIdx.x == 0) {
        q.sx[m] = s;
        if (q.site_amax) atomicMax(reinterpret_cast<int*>(q.site_amax), __float_as_int(amax));
    }
    uint32_t* dst = reinterpret_cast<uint32_t*>(q.codes + (size_t)m * K);
    const float thr = mul_rn(448.0f, s);
    unsigned clipped = 0;
#pragma unroll
    for (int g = 0; g < G; ++g) {
        dst[(kvh * G + g) * (D / 4) + lane] = e4m3x4(div_rn(v[g].x, s), div_rn(v[g].y, s), div_rn(v[g].z, s), div_rn(v[g].w, s));
        if (q.clip_count) clipped += clip4(v[g].x, v[g].y, v[g].z, v[g].w, thr);
    }
    clip_add(q, clipped);
    trace_exit(a.pf);
}

}  // namespace ev
