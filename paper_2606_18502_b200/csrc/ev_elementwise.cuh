// HBM-/latency-bound kernels of the verify step: weight quantizer (K1), embedding gather (K11),
// RMSNorm + per-token absmax + E4M3 quantize (K3), RoPE + paged KV write (K4), SwiGLU + quantize
// (K6), tree bookkeeping, argmax finalize (K8), greedy acceptance walk (K9), KV compaction (K10).
// All element-wise arithmetic uses explicitly rounded fp32 operations (ev::mul_rn ...) so each
// value is bit-identical to the method's definition given the same inputs.
#pragma once
#include "ev_common.cuh"

namespace ev {

constexpr int EW_THREADS = 256;

// red: >= blockDim.x / 32 floats of shared memory
__device__ __forceinline__ float block_max(float v, float* red) {
    v = warp_max(v);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = blockDim.x >> 5;
    __syncthreads();
    if (l == 0) red[w] = v;
    __syncthreads();
    float r = red[0];
    for (int i = 1; i < nw; ++i) r = fmaxf(r, red[i]);
    return r;
}

// absmax of a bf16 matrix (per-tensor weight scales): atomicMax on the bits of a non-negative float; *out zeroed before
__global__ void __launch_bounds__(256) tensor_absmax_bf16_kernel(const __nv_bfloat16* __restrict__ w, long n8, float* __restrict__ out) {
    __shared__ float red[8];
    const uint4* src = reinterpret_cast<const uint4*>(w);
    float amax = 0.f;
    for (long i = blockIdx.x * 256L + threadIdx.x; i < n8; i += (long)gridDim.x * 256) {
        const uint4 v = __ldg(src + i);
        const uint32_t u[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            amax = fmaxf(amax, fabsf(__uint_as_float(u[j] << 16)));
            amax = fmaxf(amax, fabsf(__uint_as_float(u[j] & 0xFFFF0000u)));
        }
    }
    amax = block_max(amax, red);
    if (threadIdx.x == 0) atomicMax(reinterpret_cast<int*>(out), __float_as_int(amax));
}

// ---- K1: per-output-channel absmax -> scale, E4M3 codes --------------------------------------
// one CTA per output channel (row); cols % 8 == 0.  Codes are written straight into the GEMM's HBM
// layout: [n/128][k/128] tiles of 128 rows x 128 bytes, 16 KiB contiguous, 128-byte swizzled
// (ev_gemm.cuh); row_off = first row of this matrix inside fused storage (QKV, gate|up).
__global__ void __launch_bounds__(EW_THREADS) quantize_weight_rows_kernel(const __nv_bfloat16* __restrict__ w, long cols,
                                                                          uint8_t* __restrict__ codes_tiled, int total_kb,
                                                                          long row_off, float* __restrict__ scales,
                                                                          const float* __restrict__ tensor_amax) {
    __shared__ float red[EW_THREADS / 32];
    const long row = blockIdx.x;
    const uint4* src = reinterpret_cast<const uint4*>(w + row * cols);
    const int nvec = (int)(cols / 8);
    float amax = 0.f;
    for (int i = threadIdx.x; i < nvec; i += EW_THREADS) {
        uint4 v = __ldg(src + i);
        const uint32_t u[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            amax = fmaxf(amax, fabsf(__uint_as_float(u[j] << 16)));
            amax = fmaxf(amax, fabsf(__uint_as_float(u[j] & 0xFFFF0000u)));
        }
    }
    amax = block_max(amax, red);
    if (tensor_amax) amax = *tensor_amax;   // per-tensor mode: the whole matrix's absmax (tensor_absmax_bf16_kernel)
    const float s = (amax == 0.f) ? 1.0f : div_rn(amax, 448.0f);
    const long n = row_off + row;
    if (threadIdx.x == 0) scales[n] = s;
    const int r = (int)(n & 127);
    uint8_t* trow = codes_tiled + (size_t)(n >> 7) * total_kb * 16384;
    for (int i = threadIdx.x; i < nvec; i += EW_THREADS) {
        uint4 v = __ldg(src + i);
        const uint32_t u[4] = {v.x, v.y, v.z, v.w};
        float f[8];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            f[2 * j] = div_rn(__uint_as_float(u[j] << 16), s);
            f[2 * j + 1] = div_rn(__uint_as_float(u[j] & 0xFFFF0000u), s);
        }
        uint2 o;
        o.x = e4m3x4(f[0], f[1], f[2], f[3]);
        o.y = e4m3x4(f[4], f[5], f[6], f[7]);
        const int k = i * 8, c = k & 127;
        const int off = r * 128 + ((((c >> 4) ^ (r & 7)) << 4) | (c & 15));
        *reinterpret_cast<uint2*>(trow + (size_t)(k >> 7) * 16384 + off) = o;
    }
}

// ---- tree bookkeeping: one thread per sequence -----------------------------------------------
// Besides depths, positions and ancestor masks this kernel fixes how every node's key set is cut for attention
// (ev_attention_tc.cuh, "batch-invariant reduction order"): a node at position p = L + depth attends to positions
// [0, p].  The BULK [0, p - ATT_TAIL_R) goes through the tensor-core kernel in chunks aligned to absolute positions;
// the TAIL (the last ATT_TAIL_R + 1 positions: the youngest cached tokens and the node's nearest ancestors, itself
// included) is added key by key in position order by the merge kernel.  For trees of depth <= ATT_TAIL_R the bulk
// lies entirely in the committed context, so a node's result does not depend on the tree it arrived in.
constexpr int ATT_TAIL_R = 8;
struct TreePrepArgs {
    int B, T, vocab, page_size;
    const int32_t* seq_slots;  // [B]
    const int32_t* tokens;     // [B][T]
    const int32_t* parents;    // [B][T]
    const int32_t* n_nodes;    // [B] or null
    const int32_t* ctx_len;    // [max_seqs] (device state)
    const int32_t* capacity;   // [max_seqs] tokens
    int max_seqs, max_pos;
    int max_keys;              // keys the attention grid of this step covers (n_chunks * chunk): longer sequences are rejected
    int32_t* Lsnap;            // [B] context length at entry
    int32_t* nn_eff;           // [B] nodes in use (0 when the sequence is rejected)
    int32_t* order;            // [B] sequences by decreasing context length (attention CTAs start the longest first)
    int32_t* status;           // [B]
    int32_t* depth;            // [B][T]
    int32_t* pos;              // [B][T] RoPE position = L + depth
    unsigned long long* anc;   // [B][T] ancestor-or-self bit masks
    unsigned long long* anc_bulk;  // [B][T] ancestors that belong to the bulk (depth < own depth - ATT_TAIL_R); 0 for shallow trees
    int32_t* erow;             // [B][T] cached positions below erow are bulk keys of the row: max(0, L + depth - ATT_TAIL_R)
    int32_t* kend_row;         // [B][T] one past the row's last bulk key slot
    int32_t* kend_seq;         // [B] max over the sequence's rows
    unsigned long long* argmax_keys;  // [B*T] reset to 0 here
};

__global__ void tree_prep_kernel(TreePrepArgs a) {
    pdl_launch_dependents();
    pdl_wait();
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= a.B) return;
    const int T = a.T;
    int st = 0;
    const int slot = a.seq_slots[b];
    int nn = a.n_nodes ? a.n_nodes[b] : T;
    int L = 0;
    if (nn < 1 || nn > T) { st |= 1; nn = 0; }   // checked before anything is indexed by it
    if (slot < 0 || slot >= a.max_seqs) {
        st |= 4;
    } else {
        L = a.ctx_len[slot];
        if (L + nn > a.capacity[slot] || L + nn > a.max_pos || L + nn > a.max_keys) st |= 4;
        for (int o = 0; o < b; ++o)   // two rows of one batch on the same sequence would race on its KV slots: the later one is rejected
            if (a.seq_slots[o] == slot) st |= 4;
    }
    for (int i = 0; i < nn; ++i) {
        const int p = a.parents[b * T + i];
        const int tk = a.tokens[b * T + i];
        if (tk < 0 || tk >= a.vocab) st |= 2;
        if (i == 0 ? (p != -1) : (p < 0 || p >= i)) { st |= 1; break; }
    }
    a.status[b] = st;
    a.Lsnap[b] = L;
    a.nn_eff[b] = st ? 0 : nn;
    {   // rank of this sequence by decreasing context length (ties by index): the attention grid walks sequences in
        // this order, so with mixed lengths (config[3]: 1,024..8,192) the long CTAs start first and the tail is short
        int rank = 0;
        for (int o = 0; o < a.B; ++o) {
            const int so = a.seq_slots[o];
            const int Lo = (so < 0 || so >= a.max_seqs) ? 0 : a.ctx_len[so];
            rank += (Lo > L || (Lo == L && o < b)) ? 1 : 0;
        }
        a.order[rank] = b;
    }
    int kend = 0;
    for (int i = 0; i < T; ++i) {
        int d = 0;
        unsigned long long m = 1ull, mb = 0ull;  // padding / rejected rows see the root only
        int e = 0, ke = 0;
        if (!st && i < nn) {
            const int p = a.parents[b * T + i];
            if (i > 0) { d = a.depth[b * T + p] + 1; m = a.anc[b * T + p] | (1ull << i); }
            e = max(0, L + d - ATT_TAIL_R);
            if (d > ATT_TAIL_R)
                for (int j = 0; j < i; ++j)
                    if (((m >> j) & 1ull) && a.depth[b * T + j] < d - ATT_TAIL_R) mb |= 1ull << j;
            ke = mb ? L + (63 - __clzll((long long)mb)) + 1 : min(L, e);
        }
        a.depth[b * T + i] = d;
        a.pos[b * T + i] = L + d;
        a.anc[b * T + i] = m;
        a.anc_bulk[b * T + i] = mb;
        a.erow[b * T + i] = e;
        a.kend_row[b * T + i] = ke;
        kend = max(kend, ke);
        a.argmax_keys[b * T + i] = 0ull;
    }
    a.kend_seq[b] = kend;
}

// ---- K11: embedding gather: residual stream (fp32) <- bf16 rows --------------------------------
__global__ void __launch_bounds__(EW_THREADS) embed_gather_kernel(const int32_t* __restrict__ tokens, int vocab,
                                                                  const __nv_bfloat16* __restrict__ table, int H,
                                                                  float* __restrict__ h) {
    pdl_launch_dependents();
    pdl_wait();
    const int m = blockIdx.x;
    const int tk = tokens[m];
    const bool ok = tk >= 0 && tk < vocab;
    const uint32_t* src = reinterpret_cast<const uint32_t*>(table + (size_t)(ok ? tk : 0) * H);
    float2* dst = reinterpret_cast<float2*>(h + (size_t)m * H);
    for (int i = threadIdx.x; i < H / 2; i += EW_THREADS) {
        const uint32_t u = ok ? __ldg(src + i) : 0u;
        dst[i] = make_float2(__uint_as_float(u << 16), __uint_as_float(u & 0xFFFF0000u));
    }
}

// ---- per-token quantization of a row already held as fp32 values produced by `val(i)` ----------
// shared tail of K3 / K6 / ev_op_quantize_rows: absmax -> scale -> codes
struct QuantOut {
    uint8_t* codes;            // [M][K]
    float* sx;                 // [M]
    const float* static_scale; // null = dynamic per-token
    float* site_amax;          // null, or calibration accumulator (atomicMax on the float's bits)
    unsigned long long* clip_count;  // null, or (static scales) this site's count of elements with |x| > 448 s: the
                                     // clipping PAPER.md:140 measures ("clip rate"); SURVEY section 8(f)-1
};
// adds this thread's count of clipped elements to the site counter: one atomic per warp that saw any
__device__ __forceinline__ void clip_add(const QuantOut& q, unsigned cnt) {
    if (!q.clip_count) return;   // uniform
    const unsigned tot = __reduce_add_sync(0xffffffffu, cnt);
    if (tot && (threadIdx.x & 31) == 0) atomicAdd(q.clip_count, (unsigned long long)tot);
}
__device__ __forceinline__ unsigned clip4(float x0, float x1, float x2, float x3, float thr) {
    return (unsigned)(fabsf(x0) > thr) + (unsigned)(fabsf(x1) > thr) + (unsigned)(fabsf(x2) > thr) + (unsigned)(fabsf(x3) > thr);
}

template <class F>
__device__ __forceinline__ void quantize_row(int m, int K, F val, const QuantOut& q, float* red) {
    float amax = 0.f;
    for (int i = threadIdx.x * 4; i < K; i += EW_THREADS * 4) {
#pragma unroll
        for (int j = 0; j < 4; ++j) amax = fmaxf(amax, fabsf(val(i + j)));
    }
    amax = block_max(amax, red);
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
    for (int i = threadIdx.x * 4; i < K; i += EW_THREADS * 4) {
        dst[i >> 2] = e4m3x4(div_rn(val(i), s), div_rn(val(i + 1), s), div_rn(val(i + 2), s), div_rn(val(i + 3), s));
        if (q.clip_count) clipped += clip4(val(i), val(i + 1), val(i + 2), val(i + 3), thr);
    }
    clip_add(q, clipped);
}

// row held in registers, spread over the CTAs of a cluster: this CTA owns the float4 numbers [c0, c1) of the
// row and thread t owns c0 + t + k*blockDim.x (k < NV4).  The absmax meets across the cluster (cluster_max).
template <int NV4>
__device__ __forceinline__ void quantize_regs(const float4 (&v)[NV4], int m, int K, int c0, int c1, const QuantOut& q, float* red,
                                              float* xch) {
    const int nthr = blockDim.x;
    float amax = 0.f;
#pragma unroll
    for (int k = 0; k < NV4; ++k)
        if (c0 + (int)threadIdx.x + k * nthr < c1)
            amax = fmaxf(amax, fmaxf(fmaxf(fabsf(v[k].x), fabsf(v[k].y)), fmaxf(fabsf(v[k].z), fabsf(v[k].w))));
    amax = cluster_max(block_max(amax, red), xch);
    float s;
    if (q.static_scale) s = *q.static_scale;
    else s = (amax == 0.f) ? 1.0f : div_rn(amax, 448.0f);
    if (threadIdx.x == 0 && cluster_ctarank() == 0) {
        q.sx[m] = s;
        if (q.site_amax) atomicMax(reinterpret_cast<int*>(q.site_amax), __float_as_int(amax));
    }
    uint32_t* dst = reinterpret_cast<uint32_t*>(q.codes + (size_t)m * K);
    const float thr = mul_rn(448.0f, s);
    unsigned clipped = 0;
#pragma unroll
    for (int k = 0; k < NV4; ++k) {
        const int i4 = c0 + (int)threadIdx.x + k * nthr;
        if (i4 < c1) {
            dst[i4] = e4m3x4(div_rn(v[k].x, s), div_rn(v[k].y, s), div_rn(v[k].z, s), div_rn(v[k].w, s));
            if (q.clip_count) clipped += clip4(v[k].x, v[k].y, v[k].z, v[k].w, thr);
        }
    }
    clip_add(q, clipped);
}
// this CTA's share [c0, c1) of a row of n4 float4s
__device__ __forceinline__ void cluster_cols(int n4, int& c0, int& c1) {
    const int nct = (int)cluster_nctarank(), r = (int)cluster_ctarank();
    const int per = ((n4 + nct - 1) / nct + 31) & ~31;   // whole 32-float4 segments: a warp's float4s never straddle two CTAs' shares
    c0 = min(n4, r * per);
    c1 = min(n4, c0 + per);
}

// ---- K3: (residual += pending linear output) + RMSNorm + quantize; one CTA of 256 threads per token;
// H % 4 == 0 and H <= 4096.  `pend` is the raw output of the previous O / down GEMM (LinOut, ev_common.cuh) or
// has p == null; the updated residual stream is written back to h.  H <= 4 * ROW_THREADS * NV4 * cluster size. ----
// Row kernels (RMSNorm, SwiGLU, attention merge): ROW_THREADS threads per CTA, a row spread over the CTAs of a
// cluster, NV4 float4s per thread in registers (instantiated for 1, 2, 4; the host picks cluster size and NV4 from
// the token count so that few rows still fill the machine and many rows keep several CTAs per SM: row_plan()).
constexpr int ROW_THREADS = 256;
constexpr int NORM_THREADS = ROW_THREADS;
constexpr int NORM_SEG_MAX = 32;   // 128-element segments of a row: hidden <= 4096
template <int NORM_NV4, int MAXS>
// <4, 1> is the many-row form (one CTA per row, M > 256): six CTAs per SM (40 registers) put the 832 rows of config[2] in ONE wave (888 slots)
// instead of 1.4 waves of four (norm class 858 -> 786 us per step)
// (every other form: four CTAs per SM = 64 registers, what the compiler chose without a bound; with an explicit 1 it took 72 - 101 and
// the GEMM that follows could no longer be resident beside it: profiles/r2_step_timeline.md)
__global__ void __launch_bounds__(NORM_THREADS, (NORM_NV4 == 4 && MAXS == 1) ? 6 : 4) rmsnorm_quant_kernel(float* __restrict__ h, int H, LinOut pend,
                                                                     const __nv_bfloat16* __restrict__ gain, float eps,
                                                                     QuantOut q, L2Prefetch pf) {
    pdl_launch_dependents();  // the next kernel (a GEMM) may start prefetching its weights now
    l2_prefetch_issue(pf);
    __shared__ float red[NORM_THREADS / 32];
    __shared__ double seg[NORM_SEG_MAX];   // segment sums of the whole row, in segment order (every CTA of the cluster gets all of them)
    __shared__ float xch_f[CLUSTER_MAX];
    const int m = blockIdx.x / cluster_nctarank();   // one token row per cluster
    int c0, c1;
    cluster_cols(H / 4, c0, c1);
    uint2 gbits[NORM_NV4];   // gains (bf16 x 4) do not depend on the previous kernel: fetched before the wait
#pragma unroll
    for (int k = 0; k < NORM_NV4; ++k) {
        const int i4 = c0 + threadIdx.x + k * NORM_THREADS;
        gbits[k] = make_uint2(0x3F803F80u, 0x3F803F80u);  // 1.0, 1.0
        if (gain && i4 < c1) gbits[k] = __ldg(reinterpret_cast<const uint2*>(gain + i4 * 4));
    }
    pdl_wait();
    trace_past_wait(pf);
    float* x = h + (size_t)m * H;
    float4 v[NORM_NV4];
    const float sxm = pend.p ? __ldg(pend.sx + m) : 0.f;
    // Mean of squares in fp64, rounded once (DESIGN.md R-accum), in ONE fixed order whatever the cluster size and the
    // float4s per thread: the row is cut into segments of 32 float4s (128 elements); a segment always belongs to one
    // warp in one k-iteration, which sums it with an xor butterfly; the segment sums are then added in segment order.
    const int nseg = (H / 4 + 31) / 32;
    const uint32_t nct = cluster_nctarank();
#pragma unroll
    for (int k = 0; k < NORM_NV4; ++k) {
        const int i4 = c0 + threadIdx.x + k * NORM_THREADS;
        const int i = i4 * 4;
        v[k] = make_float4(0.f, 0.f, 0.f, 0.f);
        double acc = 0.0;
        if (i4 < c1) {
            v[k] = *reinterpret_cast<const float4*>(x + i);
            if (pend.p) {
                const float4 y = lin_value4<MAXS>(pend, m, i, sxm);
                v[k] = make_float4(add_rn(v[k].x, y.x), add_rn(v[k].y, y.y), add_rn(v[k].z, y.z), add_rn(v[k].w, y.w));
                *reinterpret_cast<float4*>(x + i) = v[k];
            }
            acc = (((double)v[k].x * v[k].x + (double)v[k].y * v[k].y) + (double)v[k].z * v[k].z) + (double)v[k].w * v[k].w;
        }
        acc = warp_sum(acc);
        const int w4 = i4 - (int)(threadIdx.x & 31);   // the warp's first float4 (warp-uniform); every segment has exactly one owner
        const int sg = w4 >> 5;
        if ((threadIdx.x & 31) == 0 && w4 < c1) {
            if (nct == 1) seg[sg] = acc;
            else for (uint32_t r = 0; r < nct; ++r) asm volatile("st.shared::cluster.f64 [%0], %1;" ::"r"(cluster_map(seg + sg, r)), "d"(acc) : "memory");
        }
    }
    if (nct > 1) cluster_barrier(); else __syncthreads();
    double tot = 0.0;
    for (int i = 0; i < nseg; ++i) tot += seg[i];
    const float ms = (float)(tot / (double)H);
    const float r = div_rn(1.0f, sqrtf(add_rn(ms, eps)));
#pragma unroll
    for (int k = 0; k < NORM_NV4; ++k) {
        const int i4 = c0 + threadIdx.x + k * NORM_THREADS;
        const int i = i4 * 4;
        if (i4 < c1) {
            const float4 g = make_float4(__uint_as_float(gbits[k].x << 16), __uint_as_float(gbits[k].x & 0xFFFF0000u),
                                         __uint_as_float(gbits[k].y << 16), __uint_as_float(gbits[k].y & 0xFFFF0000u));
            v[k] = make_float4(mul_rn(mul_rn(v[k].x, r), g.x), mul_rn(mul_rn(v[k].y, r), g.y), mul_rn(mul_rn(v[k].z, r), g.z),
                               mul_rn(mul_rn(v[k].w, r), g.w));
        }
    }
    quantize_regs<NORM_NV4>(v, m, H, c0, c1, q, red, xch_f);
    trace_exit(pf);
}

// residual += pending linear output, nothing else (debug taps / end of a prefill pass)
__global__ void __launch_bounds__(256) apply_pending_kernel(float* __restrict__ h, int H, LinOut pend) {
    pdl_launch_dependents();
    pdl_wait();
    const int m = blockIdx.x;
    const float sxm = __ldg(pend.sx + m);
    for (int i = threadIdx.x; i < H; i += 256) h[(size_t)m * H + i] = add_rn(h[(size_t)m * H + i], lin_value(pend, m, i, sxm));
}
// y = linear output with its scales (ev_op_linear)
__global__ void __launch_bounds__(256) materialize_linear_kernel(float* __restrict__ out, int N, LinOut lin) {
    pdl_launch_dependents();
    pdl_wait();
    const int m = blockIdx.x;
    const float sxm = __ldg(lin.sx + m);
    for (int i = threadIdx.x; i < N; i += 256) out[(size_t)m * N + i] = lin_value(lin, m, i, sxm);
}

// plain per-token quantization of fp32 rows (ev_op_quantize_rows)
__global__ void __launch_bounds__(EW_THREADS) quantize_rows_kernel(const float* __restrict__ x, int K, QuantOut q) {
    __shared__ float red[EW_THREADS / 32];
    const int m = blockIdx.x;
    const float* row = x + (size_t)m * K;
    quantize_row(m, K, [&](int i) -> float { return row[i]; }, q, red);
}

// ---- K6: SwiGLU + quantize on the raw gate|up GEMM output (LinOut, ld = 2F: gate | up); one CTA of 512
// threads per token, the row of F values lives in registers; F % 4 == 0 and F <= 4 * ROW_THREADS * NV4 * cluster size. ----
__device__ __forceinline__ float swiglu_f(float g, float u) {
    // t = (g / (1 + exp(-g))) * u, fp32 ops in this order; expf is the full-range libdevice one
    return mul_rn(div_rn(g, add_rn(1.0f, expf(-g))), u);
}
constexpr int SWI_THREADS = ROW_THREADS;
template <int SWI_NV4, int MAXS>
__global__ void __launch_bounds__(SWI_THREADS) swiglu_quant_kernel(LinOut gu, int F, float* __restrict__ gu_tap, QuantOut q,
                                                                   L2Prefetch pf) {
    pdl_launch_dependents();  // the down-projection GEMM may start prefetching its weights now
    l2_prefetch_issue(pf);
    pdl_wait();
    trace_past_wait(pf);
    __shared__ float red[SWI_THREADS / 32];
    __shared__ float xch_f[CLUSTER_MAX];
    const int m = blockIdx.x / cluster_nctarank();   // one token row per cluster
    int c0, c1;
    cluster_cols(F / 4, c0, c1);
    const float sxm = __ldg(gu.sx + m);
    float4 v[SWI_NV4];
#pragma unroll
    for (int k = 0; k < SWI_NV4; ++k) {
        const int i4 = c0 + threadIdx.x + k * SWI_THREADS;
        const int i = i4 * 4;
        v[k] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (i4 < c1) {
            const float4 g = lin_value4<MAXS>(gu, m, i, sxm), u = lin_value4<MAXS>(gu, m, F + i, sxm);
            if (gu_tap) {
                *reinterpret_cast<float4*>(gu_tap + (size_t)m * 2 * F + i) = g;
                *reinterpret_cast<float4*>(gu_tap + (size_t)m * 2 * F + F + i) = u;
            }
            v[k] = make_float4(swiglu_f(g.x, u.x), swiglu_f(g.y, u.y), swiglu_f(g.z, u.z), swiglu_f(g.w, u.w));
        }
    }
    quantize_regs<SWI_NV4>(v, m, F, c0, c1, q, red, xch_f);
    trace_exit(pf);
}

// Many rows (M > ~2 rows per SM): one CTA per token, no cluster; the row of F SwiGLU values is staged in shared
// memory (4 F bytes) between the absmax pass and the quantize pass, so a thread holds only a few values in
// registers and several CTAs stay resident per SM (the register-resident form above runs one CTA per SM at F = 14336).
template <int MAXS>
__global__ void __launch_bounds__(SWI_THREADS) swiglu_quant_smem_kernel(LinOut gu, int F, float* __restrict__ gu_tap, QuantOut q,
                                                                        L2Prefetch pf) {
    extern __shared__ float4 swi_row[];   // [F / 4]
    __shared__ float red[SWI_THREADS / 32];
    pdl_launch_dependents();
    pdl_wait();
    trace_past_wait(pf);
    const int m = blockIdx.x;
    const int n4 = F / 4;
    const float sxm = __ldg(gu.sx + m);
    float amax = 0.f;
    for (int i4 = threadIdx.x; i4 < n4; i4 += SWI_THREADS) {
        const int i = i4 * 4;
        const float4 g = lin_value4<MAXS>(gu, m, i, sxm), u = lin_value4<MAXS>(gu, m, F + i, sxm);
        if (gu_tap) {
            *reinterpret_cast<float4*>(gu_tap + (size_t)m * 2 * F + i) = g;
            *reinterpret_cast<float4*>(gu_tap + (size_t)m * 2 * F + F + i) = u;
        }
        const float4 t = make_float4(swiglu_f(g.x, u.x), swiglu_f(g.y, u.y), swiglu_f(g.z, u.z), swiglu_f(g.w, u.w));
        swi_row[i4] = t;
        amax = fmaxf(amax, fmaxf(fmaxf(fabsf(t.x), fabsf(t.y)), fmaxf(fabsf(t.z), fabsf(t.w))));
    }
    amax = block_max(amax, red);   // contains the __syncthreads that publishes swi_row
    float s;
    if (q.static_scale) s = *q.static_scale;
    else s = (amax == 0.f) ? 1.0f : div_rn(amax, 448.0f);
    if (threadIdx.x == 0) {
        q.sx[m] = s;
        if (q.site_amax) atomicMax(reinterpret_cast<int*>(q.site_amax), __float_as_int(amax));
    }
    uint32_t* dst = reinterpret_cast<uint32_t*>(q.codes + (size_t)m * F);
    const float thr = mul_rn(448.0f, s);
    unsigned clipped = 0;
    for (int i4 = threadIdx.x; i4 < n4; i4 += SWI_THREADS) {
        const float4 t = swi_row[i4];   // written by this same thread
        dst[i4] = e4m3x4(div_rn(t.x, s), div_rn(t.y, s), div_rn(t.z, s), div_rn(t.w, s));
        if (q.clip_count) clipped += clip4(t.x, t.y, t.z, t.w, thr);
    }
    clip_add(q, clipped);
    trace_exit(pf);
}

// ---- K4: RoPE (positions = L + depth) on q, k of the raw QKV GEMM output + K,V -> bf16 pages; q, k, v are
// also written as fp32 to qkv_out [M][ld] (q feeds attention).  One CTA of 512 threads per token. ----
struct RopeArgs {
    LinOut lin;           // raw QKV output, ld = (Hq + 2 Hkv) * D
    float* qkv_out;       // [M][ld]
    int ld, Hq, Hkv, D, T;
    const int32_t* pos;   // [M]
    const float2* cs;     // [max_pos][D/2] (cos, sin) built on the host in fp64
    const int32_t* seq_slots;  // [B]
    const int32_t* Lsnap;      // [B]
    const int32_t* nn_eff;     // [B]
    const int32_t* page_table; // [max_seqs][max_pages]
    int max_pages, page_size;
    __nv_bfloat16* pool;       // this layer: [page][2][Hkv][page_size][D] (2-byte elements; kv_mode 2: 1-byte E4M3 codes, see pool8)
    int kv_f16;                // pool keeps the bf16-rounded values in binary16 containers (ev_common.cuh)
    uint8_t* pool8;            // kv_dtype 1 (FP8 KV cache): this layer's pool as E4M3 codes, or null
    float k_scale, v_scale;    // its static per-tensor scales: code = E4M3_sat(x / s)
    float* kv_amax;            // calibration: [2] running absmax of this layer's K (post-RoPE) and V (atomicMax on the bits), or null
    L2Prefetch pf;
};
constexpr int ROPE_THREADS = 256;
template <int MAXS>
__global__ void __launch_bounds__(ROPE_THREADS) rope_kvwrite_kernel(RopeArgs a) {
    pdl_launch_dependents();
    l2_prefetch_issue(a.pf);
    // position, destination page (tree_prep_kernel's output and the page table: complete before any kernel of the step starts,
    // ev_api.cu serial_next_launch) before griddepcontrol.wait; the wait guards the QKV GEMM's slabs and the activation scales
    const int m = blockIdx.x;
    const int b = m / a.T, node = m % a.T;
    const int D = a.D, D2 = D / 2;
    float* __restrict__ row = a.qkv_out + (size_t)m * a.ld;
    const float2* cs = a.cs + (size_t)__ldcg(a.pos + m) * D2;
    const bool write = node < __ldcg(a.nn_eff + b);
    __nv_bfloat16* kdst = nullptr;
    __nv_bfloat16* vdst = nullptr;
    if (write) {
        const int slot_tok = __ldcg(a.Lsnap + b) + node;
        const int page = a.page_table[(size_t)__ldcg(a.seq_slots + b) * a.max_pages + slot_tok / a.page_size];
        const size_t base = (size_t)page * 2 * a.Hkv * a.page_size * D + (size_t)(slot_tok % a.page_size) * D;
        kdst = a.pool + base;
        vdst = a.pool + base + (size_t)a.Hkv * a.page_size * D;
    }
    pdl_wait();
    trace_past_wait(a.pf);
    const float sxm = __ldg(a.lin.sx + m);
    const int n_rot4 = (a.Hq + a.Hkv) * D2 / 4;  // groups of 4 rotation pairs
    const int tid = blockIdx.y * blockDim.x + threadIdx.x, nthr = gridDim.y * blockDim.x;  // a row may be spread over gridDim.y CTAs
    for (int i = tid; i < n_rot4; i += nthr) {
        const int head = (i * 4) / D2, j = (i * 4) % D2;
        const float4 lo = lin_value4<MAXS>(a.lin, m, head * D + j, sxm), hi = lin_value4<MAXS>(a.lin, m, head * D + j + D2, sxm);
        const float4 c01 = __ldg(reinterpret_cast<const float4*>(cs + j)), c23 = __ldg(reinterpret_cast<const float4*>(cs + j + 2));
        float4 rlo, rhi;  // (cos, sin) pairs: c01 = (c0, s0, c1, s1), c23 = (c2, s2, c3, s3)
        rlo.x = sub_rn(mul_rn(lo.x, c01.x), mul_rn(hi.x, c01.y)); rhi.x = add_rn(mul_rn(hi.x, c01.x), mul_rn(lo.x, c01.y));
        rlo.y = sub_rn(mul_rn(lo.y, c01.z), mul_rn(hi.y, c01.w)); rhi.y = add_rn(mul_rn(hi.y, c01.z), mul_rn(lo.y, c01.w));
        rlo.z = sub_rn(mul_rn(lo.z, c23.x), mul_rn(hi.z, c23.y)); rhi.z = add_rn(mul_rn(hi.z, c23.x), mul_rn(lo.z, c23.y));
        rlo.w = sub_rn(mul_rn(lo.w, c23.z), mul_rn(hi.w, c23.w)); rhi.w = add_rn(mul_rn(hi.w, c23.z), mul_rn(lo.w, c23.w));
        *reinterpret_cast<float4*>(row + head * D + j) = rlo;
        *reinterpret_cast<float4*>(row + head * D + j + D2) = rhi;
        if (head >= a.Hq && a.kv_amax) {
            const float am = fmaxf(fmaxf(fmaxf(fabsf(rlo.x), fabsf(rlo.y)), fmaxf(fabsf(rlo.z), fabsf(rlo.w))),
                                   fmaxf(fmaxf(fabsf(rhi.x), fabsf(rhi.y)), fmaxf(fabsf(rhi.z), fabsf(rhi.w))));
            if (write) atomicMax(reinterpret_cast<int*>(a.kv_amax), __float_as_int(am));
        }
        if (head >= a.Hq && write && a.pool8) {
            uint8_t* kd = a.pool8 + (kdst - a.pool) + (size_t)(head - a.Hq) * a.page_size * D;
            *reinterpret_cast<uint32_t*>(kd + j) = e4m3x4(div_rn(rlo.x, a.k_scale), div_rn(rlo.y, a.k_scale), div_rn(rlo.z, a.k_scale), div_rn(rlo.w, a.k_scale));
            *reinterpret_cast<uint32_t*>(kd + j + D2) = e4m3x4(div_rn(rhi.x, a.k_scale), div_rn(rhi.y, a.k_scale), div_rn(rhi.z, a.k_scale), div_rn(rhi.w, a.k_scale));
        } else if (head >= a.Hq && write) {
            __nv_bfloat16* kd = kdst + (size_t)(head - a.Hq) * a.page_size * D;
            __nv_bfloat162 p0 = __floats2bfloat162_rn(rlo.x, rlo.y), p1 = __floats2bfloat162_rn(rlo.z, rlo.w);
            __nv_bfloat162 p2 = __floats2bfloat162_rn(rhi.x, rhi.y), p3 = __floats2bfloat162_rn(rhi.z, rhi.w);
            uint32_t w0 = *reinterpret_cast<uint32_t*>(&p0), w1 = *reinterpret_cast<uint32_t*>(&p1);
            uint32_t w2 = *reinterpret_cast<uint32_t*>(&p2), w3 = *reinterpret_cast<uint32_t*>(&p3);
            if (a.kv_f16) { w0 = bf16x2_to_f16x2(w0); w1 = bf16x2_to_f16x2(w1); w2 = bf16x2_to_f16x2(w2); w3 = bf16x2_to_f16x2(w3); }
            *reinterpret_cast<uint2*>(kd + j) = make_uint2(w0, w1);
            *reinterpret_cast<uint2*>(kd + j + D2) = make_uint2(w2, w3);
        }
    }
    const int voff = (a.Hq + a.Hkv) * D;
    for (int i = tid; i < a.Hkv * D / 4; i += nthr) {
        const int head = (i * 4) / D, j = (i * 4) % D;
        const float4 v = lin_value4<MAXS>(a.lin, m, voff + i * 4, sxm);
        *reinterpret_cast<float4*>(row + voff + i * 4) = v;
        if (a.kv_amax && write) atomicMax(reinterpret_cast<int*>(a.kv_amax + 1), __float_as_int(fmaxf(fmaxf(fabsf(v.x), fabsf(v.y)), fmaxf(fabsf(v.z), fabsf(v.w)))));
        if (write && a.pool8) {
            *reinterpret_cast<uint32_t*>(a.pool8 + (vdst - a.pool) + (size_t)head * a.page_size * D + j) =
                e4m3x4(div_rn(v.x, a.v_scale), div_rn(v.y, a.v_scale), div_rn(v.z, a.v_scale), div_rn(v.w, a.v_scale));
        } else if (write) {
            __nv_bfloat162 p0 = __floats2bfloat162_rn(v.x, v.y), p1 = __floats2bfloat162_rn(v.z, v.w);
            uint32_t w0 = *reinterpret_cast<uint32_t*>(&p0), w1 = *reinterpret_cast<uint32_t*>(&p1);
            if (a.kv_f16) { w0 = bf16x2_to_f16x2(w0); w1 = bf16x2_to_f16x2(w1); }
            *reinterpret_cast<uint2*>(vdst + (size_t)head * a.page_size * D + j) = make_uint2(w0, w1);
        }
    }
    trace_exit(a.pf);
}

// ---- K8 finalize + K9 greedy acceptance walk + ctx_len update: one thread per sequence ---------
struct AcceptArgs {
    int B, T, commit, force_all;
    const int32_t* tokens;
    const int32_t* parents;
    const int32_t* nn_eff;
    const int32_t* status;
    const int32_t* Lsnap;
    const int32_t* seq_slots;
    const unsigned long long* argmax_keys;  // [B*T] packed (ordered logit bits << 32 | ~index)
    int32_t* argmax_out;                    // optional [B][T]
    int32_t* accept_len;
    int32_t* accept_nodes;
    int32_t* out_tokens;
    int32_t* new_ctx_len;
    int32_t* ctx_len;                       // device state, advanced when commit
};
__global__ void accept_walk_kernel(AcceptArgs a) {
    pdl_launch_dependents();
    pdl_wait();
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= a.B) return;
    const int T = a.T, nn = a.nn_eff[b], L = a.Lsnap[b];
    const int32_t* tok = a.tokens + b * T;
    const int32_t* par = a.parents + b * T;
    int32_t* path = a.accept_nodes + b * T;
    int32_t* out = a.out_tokens + b * T;
    for (int i = 0; i < T; ++i) {
        path[i] = -1;
        out[i] = -1;
        if (a.argmax_out) a.argmax_out[b * T + i] = (i < nn) ? (int32_t)(0xFFFFFFFFu - (uint32_t)a.argmax_keys[b * T + i]) : -1;
    }
    if (nn == 0) {  // rejected sequence
        a.accept_len[b] = 0;
        a.new_ctx_len[b] = L;
        return;
    }
    int n_path = 1;
    path[0] = 0;
    if (a.force_all) {
        for (int i = 1; i < nn; ++i) path[i] = i;
        n_path = nn;
    } else {
        int cur = 0;
        while (true) {
            const int32_t want = (int32_t)(0xFFFFFFFFu - (uint32_t)a.argmax_keys[b * T + cur]);
            int nxt = -1;
            for (int c = cur + 1; c < nn; ++c)
                if (par[c] == cur && tok[c] == want) { nxt = c; break; }
            if (nxt < 0) break;
            path[n_path++] = nxt;
            cur = nxt;
        }
        for (int j = 1; j < n_path; ++j) out[j - 1] = tok[path[j]];
        out[n_path - 1] = (int32_t)(0xFFFFFFFFu - (uint32_t)a.argmax_keys[b * T + cur]);
    }
    a.accept_len[b] = n_path - 1;
    a.new_ctx_len[b] = L + n_path;
    if (a.commit) a.ctx_len[a.seq_slots[b]] = L + n_path;
}

// ---- K10: KV compaction: slot L+path[j] -> slot L+j (j = 1..a), all layers, K and V -----------
// sources are never overwritten before they are read (path[j] >= j, strictly increasing), so all
// moves of a sequence run in parallel.  grid (B, n_layers).
struct CompactArgs {
    int eb;             // bytes per pool element: 2 (bf16 / binary16 containers) or 1 (E4M3 codes)
    int T, Hkv, D, page_size, max_pages;
    long layer_stride;  // elements per layer in the pool
    __nv_bfloat16* pool;
    const int32_t* page_table;
    const int32_t* seq_slots;
    const int32_t* Lsnap;
    const int32_t* accept_len;
    const int32_t* accept_nodes;
};
__global__ void __launch_bounds__(EW_THREADS) kv_compact_kernel(CompactArgs a) {
    pdl_launch_dependents();
    pdl_wait();
    const int b = blockIdx.x, layer = blockIdx.y;
    const int n = a.accept_len[b];
    const int L = a.Lsnap[b];
    const int32_t* pt = a.page_table + (size_t)a.seq_slots[b] * a.max_pages;
    uint8_t* pool = reinterpret_cast<uint8_t*>(a.pool) + (size_t)layer * a.layer_stride * a.eb;
    const int vec_per_head = a.D * a.eb / 16;      // 16-byte vectors per (token, K|V, head) row
    const int per_tok = 2 * a.Hkv * vec_per_head;  // K|V x heads
    for (int j = 1; j <= n; ++j) {
        const int src_node = a.accept_nodes[b * a.T + j];
        if (src_node == j) continue;
        const int ss = L + src_node, ds = L + j;
        const size_t sbase = (size_t)pt[ss / a.page_size] * 2 * a.Hkv * a.page_size * a.D + (size_t)(ss % a.page_size) * a.D;
        const size_t dbase = (size_t)pt[ds / a.page_size] * 2 * a.Hkv * a.page_size * a.D + (size_t)(ds % a.page_size) * a.D;
        for (int i = threadIdx.x; i < per_tok; i += EW_THREADS) {
            const int kvh = i / vec_per_head, c = i % vec_per_head;  // kvh in [0, 2*Hkv)
            const size_t off = (size_t)kvh * a.page_size * a.D;
            *reinterpret_cast<uint4*>(pool + (dbase + off) * a.eb + (size_t)c * 16) = *reinterpret_cast<const uint4*>(pool + (sbase + off) * a.eb + (size_t)c * 16);
        }
    }
}

// ---- dense <-> paged copies for export/import (one CTA per (token, layer)) ---------------------
struct DenseCopyArgs {
    int Hkv, D, page_size, n_tokens, layer_begin;
    long layer_stride;
    __nv_bfloat16* pool;
    const int32_t* page_row;   // this sequence's page-table row
    __nv_bfloat16* dense;      // [layer][2][Hkv][n_tokens][D], always bf16
    int to_dense;
    int kv_f16;                // pool container (ev_common.cuh)
    int eb;                    // bytes per element: 2, or 1 (E4M3 codes: dense is then uint8 codes too)
};
__global__ void __launch_bounds__(128) dense_copy_kernel(DenseCopyArgs a) {
    const int t = blockIdx.x, li = blockIdx.y;
    uint8_t* pool = reinterpret_cast<uint8_t*>(a.pool) + (size_t)(a.layer_begin + li) * a.layer_stride * a.eb;
    const size_t pbase = (size_t)a.page_row[t / a.page_size] * 2 * a.Hkv * a.page_size * a.D + (size_t)(t % a.page_size) * a.D;
    const int vec_per_head = a.D * a.eb / 16;
    for (int i = threadIdx.x; i < 2 * a.Hkv * vec_per_head; i += 128) {
        const int kvh = i / vec_per_head, c = i % vec_per_head;
        uint4* p = reinterpret_cast<uint4*>(pool + (pbase + (size_t)kvh * a.page_size * a.D) * a.eb + (size_t)c * 16);
        uint4* d = reinterpret_cast<uint4*>(reinterpret_cast<uint8_t*>(a.dense) + ((((size_t)li * 2 * a.Hkv + kvh) * a.n_tokens + t) * a.D) * a.eb + (size_t)c * 16);
        if (a.to_dense) {
            uint4 v = *p;
            if (a.kv_f16) { v.x = f16x2_to_bf16x2(v.x); v.y = f16x2_to_bf16x2(v.y); v.z = f16x2_to_bf16x2(v.z); v.w = f16x2_to_bf16x2(v.w); }
            *d = v;
        } else {
            uint4 v = *d;
            if (a.kv_f16) { v.x = bf16x2_to_f16x2(v.x); v.y = bf16x2_to_f16x2(v.y); v.z = bf16x2_to_f16x2(v.z); v.w = bf16x2_to_f16x2(v.w); }
            *p = v;
        }
    }
}

__global__ void set_i32_kernel(int32_t* p, int32_t v) { *p = v; }
struct SetLensArgs { static constexpr int MAX = 64; int n; int slot[MAX]; int len[MAX]; };
__global__ void set_lens_kernel(int32_t* ctx_len, SetLensArgs a) {
    pdl_launch_dependents();
    pdl_wait();
    if ((int)threadIdx.x < a.n) ctx_len[a.slot[threadIdx.x]] = a.len[threadIdx.x];
}

// out[M][H] f32 copy (hidden taps)
__global__ void __launch_bounds__(EW_THREADS) copy_f32_kernel(const float4* __restrict__ src, float4* __restrict__ dst, long n4) {
    for (long i = blockIdx.x * (long)EW_THREADS + threadIdx.x; i < n4; i += (long)gridDim.x * EW_THREADS) dst[i] = src[i];
}

}  // namespace ev
