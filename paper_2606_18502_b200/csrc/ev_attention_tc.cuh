// K5 (tcgen05 version): tree-masked GQA attention over the paged bf16 KV cache on the 5th-gen tensor
// cores ("tree attention"; BASELINE.json:north_star (2)).  Same decomposition and outputs
// as tree_attn_partial_kernel (ev_attention.cuh): one CTA = (sequence, kv head, 128-row tile, key split);
// rows = tree nodes x GQA group; partial (O, max, sum) per split, merged by attn_merge_quant_kernel.
//
// Data flow per 64-key tile j (a CTA walks its key range tile by tile):
//   TMA warp      : 4 pages x {K,V} x {d-halves} boxes of 16 tokens x 64 dims -> 128-byte-swizzled smem
//                   (the pool's 4 KiB (page, K|V, head) blocks are read in place through one 2-D tensor map)
//   MMA thread    : S[j&1]  = Q . K_j^T   (tcgen05.mma kind::f16, A = Q from smem, B = K tile, D in TMEM)
//                   Oc      = P[j&1] . V_j (A = P from TMEM, B = V tile MN-major, D in TMEM, from zero)
//   8 softmax warps (thread = one query row x half of the tile's keys / half of d):
//                   S -> registers (tcgen05.ld), scale, tree mask, online max (halves meet in smem),
//                   p = 2^((s-m) log2 e), P -> TMEM (tcgen05.st); then Oc -> registers and
//                   O = O * exp(m_old - m_new) + Oc with ONE rounded fp32 operation per tile.
// Precision (DESIGN.md section 6 "attention precision"): Q and P are fp32 values split into hi+mid+lo bf16
// parts (3 x 8 significand bits: exact), K and V are bf16, so every product is exact; the tensor core only
// accumulates (smallest parts first).  The running output lives in registers, not in TMEM, because long
// tensor-core accumulation chains truncate.
#pragma once
#include "ev_common.cuh"
#include "ev_attention.cuh"

namespace ev {

constexpr int TCA_THREADS = 320;  // warp 0 TMA producer, warp 1 MMA issuer, warps 2..9 softmax / correction
constexpr int TCA_BN = 64;        // keys per tile (= ATT_CH: the split plan is shared with the legacy kernel)
constexpr int TCA_STAGES = 3;
constexpr int TCA_PAGE = 16;      // tokens per page this kernel is built for

template <int D>
struct TcaCfg {
    static constexpr int NH = D / 64;                    // 128-byte (64-element) halves of a head row
    static constexpr int Q_PART = NH * 128 * 128;        // bytes of one bf16 part of the 128 x D query tile
    static constexpr int Q_BYTES = 3 * Q_PART;
    static constexpr int KV_HALF = TCA_BN * 128;         // 8 KiB: 64 keys x 128 B
    static constexpr int K_BYTES = NH * KV_HALF;
    static constexpr int STAGE = 2 * K_BYTES;            // K tile | V tile
    static constexpr int BAR_BYTES = 256;
    static constexpr int XCH_BYTES = (2 * 2 * 128 + 2 * 128) * 4;  // max exchange (double buffered) + sum exchange
    static constexpr int SMEM = 1024 + Q_BYTES + TCA_STAGES * STAGE + BAR_BYTES + XCH_BYTES;
    // TMEM columns
    static constexpr int TS = 0;            // S[2]: 2 x 64 fp32 columns
    static constexpr int TP = 128;          // P[2][3 parts]: 32 columns each (64 bf16 pairs)
    static constexpr int TO = 320;          // O chunk: D fp32 columns
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
// instruction descriptor, kind::f16: D fp32, A = B = bf16, A K-major, B K-major (0) or MN-major (1)
__host__ __device__ constexpr uint32_t umma_idesc_bf16(int M, int N, int b_mn_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)b_mn_major << 16) | ((uint32_t)(N >> 3) << 17) |
           ((uint32_t)(M >> 4) << 24);
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
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void softmax_bar_sync() { asm volatile("bar.sync 1, 256;" ::: "memory"); }
__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// (x0, x1) -> packed bf16 pairs hi, mid, lo with x = hi + mid + lo exactly (x0 in the low half)
__device__ __forceinline__ void split3_pack(float x0, float x1, uint32_t& hi, uint32_t& mid, uint32_t& lo) {
    uint32_t h, m, l;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(h) : "f"(x1), "f"(x0));
    const float r0 = x0 - __uint_as_float(h << 16), r1 = x1 - __uint_as_float(h & 0xFFFF0000u);
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(m) : "f"(r1), "f"(r0));
    const float t0 = r0 - __uint_as_float(m << 16), t1 = r1 - __uint_as_float(m & 0xFFFF0000u);
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(l) : "f"(t1), "f"(t0));
    hi = h; mid = m; lo = l;
}

struct TcAttnArgs {
    AttnArgs a;       // same fields as the legacy kernel (pool pointer unused here)
    int row0;         // first row of this layer in the pool tensor map: layer * n_pages * 2 * Hkv * 16
    L2Prefetch pf;
};

template <int D>
__global__ void __launch_bounds__(TCA_THREADS, 1) tree_attn_tc_kernel(const __grid_constant__ CUtensorMap tmKV, TcAttnArgs ta) {
    using C = TcaCfg<D>;
    const AttnArgs& a = ta.a;
    extern __shared__ uint8_t tca_smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(tca_smem_raw) + 1023) & ~(uintptr_t)1023);
    uint8_t* q_s = smem;                                  // [3 parts][NH][128 rows][128 B]
    uint8_t* kv_s = smem + C::Q_BYTES;                    // [STAGES][K: NH x 8 KiB | V: NH x 8 KiB]
    uint64_t* bars = reinterpret_cast<uint64_t*>(kv_s + TCA_STAGES * C::STAGE);
    uint64_t* kv_full = bars;                             // [STAGES]
    uint64_t* kv_empty = bars + TCA_STAGES;               // [STAGES]
    uint64_t* s_full = bars + 2 * TCA_STAGES;             // [2]
    uint64_t* p_full = s_full + 2;                        // [2]
    uint64_t* o_full = p_full + 2;                        // [1]
    uint64_t* o_empty = o_full + 1;                       // [1]
    uint32_t* tmem_base_smem = reinterpret_cast<uint32_t*>(o_empty + 1);
    float* xmax = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(bars) + C::BAR_BYTES);  // [2 buf][2 wg][128]
    float* xsum = xmax + 2 * 2 * 128;                     // [2 wg][128]

    const int split = blockIdx.x;
    const int kvh = blockIdx.y % a.Hkv, rg = blockIdx.y / a.Hkv;
    const int b = blockIdx.z;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int R = a.T * a.G;

    // ---- prologue that does not depend on the previous kernel (overlaps it under PDL): barriers, TMEM ----
    pdl_launch_dependents();
    l2_prefetch_issue(ta.pf);
    if (threadIdx.x == 0) {
        for (int s = 0; s < TCA_STAGES; ++s) { mbar_init(&kv_full[s], 1); mbar_init(&kv_empty[s], 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(&s_full[i], 1); mbar_init(&p_full[i], 8); }
        mbar_init(o_full, 1);
        mbar_init(o_empty, 8);
        fence_barrier_init();
        tma_prefetch_desc(&tmKV);
    }
    if (warp == 1) tmem_alloc<512>(tmem_base_smem);
    pdl_wait();
    trace_past_wait(ta.pf);
    const int nn = a.nn_eff[b];
    const int L = a.Lsnap[b];
    const int seq_slot = a.seq_slots[b];
    const int n_keys = L + nn;
    const int k_begin = split * a.split_len;
    const bool active = nn != 0 && k_begin < n_keys;   // uniform over the CTA
    const int k_end = min(k_begin + a.split_len, n_keys);
    const int n_tiles = active ? (k_end - k_begin + TCA_BN - 1) / TCA_BN : 0;
    // ---- Q tile (fp32 -> hi | mid | lo bf16, 128-byte swizzled K-major) ----
    if (active)
    {
        constexpr int CPR = D / 8;  // 16-byte chunks (8 elements) per row
        for (int it = threadIdx.x; it < 128 * CPR; it += TCA_THREADS) {
            const int r = it / CPR, c = it % CPR;
            const int row = rg * 128 + r;
            const int node = row / a.G, gi = row % a.G;
            float x[8];
            if (row < R && node < nn) {
                const float* qp = a.q + (size_t)(b * a.T + node) * a.q_ld + (size_t)(kvh * a.G + gi) * D + c * 8;
                const float4 u0 = *reinterpret_cast<const float4*>(qp), u1 = *reinterpret_cast<const float4*>(qp + 4);
                x[0] = u0.x; x[1] = u0.y; x[2] = u0.z; x[3] = u0.w; x[4] = u1.x; x[5] = u1.y; x[6] = u1.z; x[7] = u1.w;
            } else {
#pragma unroll
                for (int i = 0; i < 8; ++i) x[i] = 0.f;
            }
            uint32_t h[4], m[4], l[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) split3_pack(x[2 * i], x[2 * i + 1], h[i], m[i], l[i]);
            const int half = c >> 3, cc = c & 7;
            const int off = half * (128 * 128) + r * 128 + ((cc ^ (r & 7)) << 4);
            *reinterpret_cast<uint4*>(q_s + off) = make_uint4(h[0], h[1], h[2], h[3]);
            *reinterpret_cast<uint4*>(q_s + C::Q_PART + off) = make_uint4(m[0], m[1], m[2], m[3]);
            *reinterpret_cast<uint4*>(q_s + 2 * C::Q_PART + off) = make_uint4(l[0], l[1], l[2], l[3]);
        }
    }
    fence_proxy_async();   // generic-proxy smem writes (Q) -> visible to the tensor core's async proxy
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_base_smem;

    if (!active) {
        // nothing to do for this (sequence, split): fall through to the TMEM release
    } else if (warp == 0) {
        // ===== TMA producer: lane i issues box i of the tile (K|V, page, half) =====
        constexpr int OPS = 2 * 4 * C::NH;
        const int32_t* pt = a.page_table + (size_t)seq_slot * a.max_pages;
        const int kv = lane / (4 * C::NH), pg = (lane / C::NH) & 3, half = lane % C::NH;
        for (int j = 0; j < n_tiles; ++j) {
            const int s = j % TCA_STAGES;
            int pid = 0;
            if (lane < OPS) pid = pt[min((k_begin + j * TCA_BN) / TCA_PAGE + pg, a.max_pages - 1)];
            mbar_wait(&kv_empty[s], ((j / TCA_STAGES) & 1) ^ 1);
            if (lane == 0) mbar_arrive_expect_tx(&kv_full[s], C::STAGE);
            __syncwarp();
            if (lane < OPS) {
                uint8_t* dst = kv_s + s * C::STAGE + kv * C::K_BYTES + half * C::KV_HALF + pg * (TCA_PAGE * 128);
                tma_load_2d(dst, &tmKV, &kv_full[s], half * 64, ta.row0 + ((pid * 2 + kv) * a.Hkv + kvh) * TCA_PAGE);
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            // ===== MMA issuer =====
            constexpr uint32_t idesc_qk = umma_idesc_bf16(128, TCA_BN, 0);
            constexpr uint32_t idesc_pv = umma_idesc_bf16(128, D, 1);
            const uint32_t q_addr = smem_u32(q_s);
            auto issue_pv = [&](int i) {
                const int s = i % TCA_STAGES;
                mbar_wait(&p_full[i & 1], (i >> 1) & 1);
                if (i >= 1) mbar_wait(o_empty, (i - 1) & 1);
                tc_fence_after();
                const uint32_t v_addr = smem_u32(kv_s + s * C::STAGE + C::K_BYTES);
                const uint64_t vdesc = umma_desc_mn128(v_addr, C::KV_HALF, 1024);
                bool first = true;
#pragma unroll
                for (int part = 2; part >= 0; --part) {
#pragma unroll
                    for (int t = 0; t < TCA_BN / 16; ++t) {
                        umma_bf16_ts(tmem_base + C::TO, tmem_base + C::TP + (i & 1) * 96 + part * 32 + t * 8,
                                     vdesc + (uint64_t)(t * (16 * 128 >> 4)), idesc_pv, first ? 0u : 1u);
                        first = false;
                    }
                }
                umma_commit(&kv_empty[s]);
                umma_commit(o_full);
            };
            for (int j = 0; j < n_tiles; ++j) {
                const int s = j % TCA_STAGES;
                mbar_wait(&kv_full[s], (j / TCA_STAGES) & 1);
                tc_fence_after();
                const uint32_t k_addr = smem_u32(kv_s + s * C::STAGE);
                bool first = true;
#pragma unroll
                for (int part = 2; part >= 0; --part) {
#pragma unroll
                    for (int h = 0; h < C::NH; ++h) {
                        const uint64_t adesc = umma_desc_k128(q_addr + part * C::Q_PART + h * (128 * 128));
                        const uint64_t bdesc = umma_desc_k128(k_addr + h * C::KV_HALF);
#pragma unroll
                        for (int ks = 0; ks < 4; ++ks) {  // UMMA K = 16 bf16 = 32 B
                            umma_bf16_ss(tmem_base + C::TS + (j & 1) * TCA_BN, adesc + 2 * ks, bdesc + 2 * ks, idesc_qk, first ? 0u : 1u);
                            first = false;
                        }
                    }
                }
                umma_commit(&s_full[j & 1]);
                if (j >= 1) issue_pv(j - 1);
            }
            issue_pv(n_tiles - 1);
        }
    } else {
        // ===== softmax / correction: thread = (row, warpgroup); wg handles keys [32 wg, +32) of a tile and
        // output columns [DH wg, +DH).  Warp w may touch TMEM lanes 32 (w % 4) .. +31. =====
        const int wg = (warp - 2) >> 2;
        const int r = (warp & 3) * 32 + lane;
        const int row = rg * 128 + r;
        const int node = row / a.G, gi = row % a.G;
        const bool valid = row < R && node < nn;
        const unsigned long long anc = valid ? a.anc[b * a.T + node] : 1ull;
        const uint32_t lane_addr = tmem_base + ((uint32_t)((warp & 3) * 32) << 16);
        constexpr float LOG2E = 1.4426950408889634f;
        float o[C::DH];
#pragma unroll
        for (int i = 0; i < C::DH; ++i) o[i] = 0.f;
        float m_run = -INFINITY, l_run = 0.f, c_prev = 0.f;

        auto correct = [&](int i) {  // O = O * c_prev + Oc(i)
            mbar_wait(o_full, i & 1);
            tc_fence_after();
#pragma unroll
            for (int cb = 0; cb < C::DH / 32; ++cb) {
                uint32_t ov[32];
                tmem_ld32(lane_addr + C::TO + wg * C::DH + cb * 32, ov);
                tmem_ld_wait();
                if (cb == C::DH / 32 - 1) {
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(o_empty);
                }
#pragma unroll
                for (int e = 0; e < 32; ++e) o[cb * 32 + e] = fmaf(o[cb * 32 + e], c_prev, __uint_as_float(ov[e]));
            }
        };

        for (int j = 0; j < n_tiles; ++j) {
            mbar_wait(&s_full[j & 1], (j >> 1) & 1);
            tc_fence_after();
            uint32_t sv[32];
            tmem_ld32(lane_addr + C::TS + (j & 1) * TCA_BN + wg * 32, sv);
            tmem_ld_wait();
            const int kb = k_begin + j * TCA_BN + wg * 32;
            const bool need_mask = kb + 32 > L;   // tile half touches tree keys or the end of the key range
            float mx = -INFINITY;
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                float v = mul_rn(__uint_as_float(sv[e]), a.scale);
                if (need_mask) {
                    const int kidx = kb + e;
                    const bool ok = kidx < k_end && (kidx < L || ((anc >> (kidx - L)) & 1ull));
                    if (!ok) v = -INFINITY;
                }
                sv[e] = __float_as_uint(v);
                mx = fmaxf(mx, v);
            }
            xmax[((j & 1) * 2 + wg) * 128 + r] = mx;
            softmax_bar_sync();
            mx = fmaxf(mx, xmax[((j & 1) * 2 + (wg ^ 1)) * 128 + r]);
            const float mn = fmaxf(m_run, mx);
            const float mu = (mn == -INFINITY) ? 0.f : mn;
            const float c = ex2_approx((m_run - mu) * LOG2E);  // 2^-inf = 0 on the first tile
            m_run = mn;
            float ls = 0.f;
            uint32_t ph[16], pm[16], pl[16];
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                const float p0 = ex2_approx((__uint_as_float(sv[2 * e]) - mu) * LOG2E);
                const float p1 = ex2_approx((__uint_as_float(sv[2 * e + 1]) - mu) * LOG2E);
                ls += p0 + p1;
                split3_pack(p0, p1, ph[e], pm[e], pl[e]);
            }
            l_run = fmaf(l_run, c, ls);
            const uint32_t p_addr = lane_addr + C::TP + (j & 1) * 96 + wg * 16;
            tmem_st16(p_addr, ph);
            tmem_st16(p_addr + 32, pm);
            tmem_st16(p_addr + 64, pl);
            tmem_st_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(&p_full[j & 1]);
            if (j >= 1) correct(j - 1);
            c_prev = c;
        }
        correct(n_tiles - 1);
        // ---- partial result of this split: O (unnormalised), running max, running sum ----
        xsum[wg * 128 + r] = l_run;
        softmax_bar_sync();
        if (valid) {
            const size_t pi = ((size_t)(b * a.T + node) * a.Hq + kvh * a.G + gi) * a.n_splits + split;
            float* op = a.o_part + pi * D + wg * C::DH;
#pragma unroll
            for (int i = 0; i < C::DH; i += 4) *reinterpret_cast<float4*>(op + i) = make_float4(o[i], o[i + 1], o[i + 2], o[i + 3]);
            if (wg == 0) *reinterpret_cast<float2*>(a.ml_part + pi * 2) = make_float2(m_run, l_run + xsum[128 + r]);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc<512>(tmem_base);
    trace_exit(ta.pf);
}

}  // namespace ev
