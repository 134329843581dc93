// Draft side ("a lightweight draft model that consumes target-model hidden states",
// PAPER.md:359-361 FP8 drafter, chain and tree drafts; architecture from the EAGLE paper the paper cites, DESIGN.md R-drafter):
// the small kernels around the decoder layer the drafter shares with the target path -
//   concat_quant_kernel : x = [embed(token) ; predecessor feature] (2H) -> per-token absmax -> E4M3 codes (input of the FC GEMM)
//   topk_kernel         : the k largest logits of every node, largest first, ties to the lower token id
//   draft_expand_kernel : one level of the static tree: a child's token = its parent's rank-th best token, its predecessor
//                         feature = its parent's predicted feature
//   gather_accepted_kernel : after a verify step, the accepted tokens and the TARGET features that precede them, per sequence
#pragma once
#include "ev_common.cuh"
#include "ev_elementwise.cuh"

namespace ev {

// ---- [embed(token) ; feature] -> codes [M][2H], scale [M]; one CTA per node ----
__global__ void __launch_bounds__(EW_THREADS) concat_quant_kernel(const int32_t* __restrict__ tokens, int vocab,
                                                                  const __nv_bfloat16* __restrict__ table, const float* __restrict__ feat,
                                                                  int H, QuantOut q) {
    pdl_launch_dependents();
    pdl_wait();
    __shared__ float red[EW_THREADS / 32];
    const int m = blockIdx.x;
    const int tk = tokens[m];
    const bool ok = tk >= 0 && tk < vocab;
    const __nv_bfloat16* erow = table + (size_t)(ok ? tk : 0) * H;
    const float* frow = feat + (size_t)m * H;
    quantize_row(m, 2 * H, [&](int i) -> float {
        if (i < H) return ok ? __bfloat162float(erow[i]) : 0.f;
        return frow[i - H];
    }, q, red);
}

// ---- top-k of a logits row: one CTA of 256 threads per node, K <= TOPK_MAX ----
constexpr int TOPK_MAX = 8;
struct TopkArgs {
    const float* logits;   // [M][V]
    int V, K, T;
    const int32_t* nn_eff; // [B] nodes in use per sequence (rows beyond it are skipped), or null
    int32_t* out;          // [M][K] token ids, largest logit first; ties: lower id first
};
__device__ __forceinline__ bool topk_better(float a, int ia, float b, int ib) { return a > b || (a == b && ia < ib); }
__global__ void __launch_bounds__(256) topk_kernel(TopkArgs a) {
    pdl_launch_dependents();
    pdl_wait();
    const int m = blockIdx.x;
    if (a.nn_eff && (m % a.T) >= a.nn_eff[m / a.T]) return;
    __shared__ float sv[256 * TOPK_MAX];
    __shared__ int si[256 * TOPK_MAX];
    float v[TOPK_MAX];
    int id[TOPK_MAX];
#pragma unroll
    for (int j = 0; j < TOPK_MAX; ++j) { v[j] = -INFINITY; id[j] = 0x7FFFFFFF; }
    const float* row = a.logits + (size_t)m * a.V;
    for (int i = threadIdx.x; i < a.V; i += 256) {
        float x = row[i];
        int xi = i;
        if (topk_better(x, xi, v[TOPK_MAX - 1], id[TOPK_MAX - 1])) {   // insertion into the sorted list (registers, unrolled)
#pragma unroll
            for (int j = 0; j < TOPK_MAX; ++j)
                if (topk_better(x, xi, v[j], id[j])) { const float tv = v[j]; const int ti = id[j]; v[j] = x; id[j] = xi; x = tv; xi = ti; }
        }
    }
#pragma unroll
    for (int j = 0; j < TOPK_MAX; ++j) { sv[threadIdx.x * TOPK_MAX + j] = v[j]; si[threadIdx.x * TOPK_MAX + j] = id[j]; }
    __syncthreads();
    // tree merge of sorted lists: stride halves, each survivor merges its neighbour's list into its own
    for (int s = 128; s >= 1; s >>= 1) {
        if ((int)threadIdx.x < s) {
            float ov[TOPK_MAX];
            int oi[TOPK_MAX];
            int pa = 0, pb = 0;
            const float* va = sv + threadIdx.x * TOPK_MAX; const int* ia = si + threadIdx.x * TOPK_MAX;
            const float* vb = sv + (threadIdx.x + s) * TOPK_MAX; const int* ib = si + (threadIdx.x + s) * TOPK_MAX;
            for (int j = 0; j < TOPK_MAX; ++j) {
                const bool ta = topk_better(va[pa], ia[pa], vb[pb], ib[pb]);
                ov[j] = ta ? va[pa] : vb[pb];
                oi[j] = ta ? ia[pa] : ib[pb];
                pa += ta ? 1 : 0; pb += ta ? 0 : 1;       // pa + pb = j + 1 <= TOPK_MAX: neither list is read past its end
            }
            for (int j = 0; j < TOPK_MAX; ++j) { sv[threadIdx.x * TOPK_MAX + j] = ov[j]; si[threadIdx.x * TOPK_MAX + j] = oi[j]; }
        }
        __syncthreads();
    }
    if ((int)threadIdx.x < a.K) a.out[(size_t)m * a.K + threadIdx.x] = si[threadIdx.x];
}

// ---- one level of the static draft tree: nodes [n0, n1) (all of depth d+1) take their token and predecessor feature from
// their parents; parents / rank are the shared topology [T]; grid (n1 - n0, B) ----
struct ExpandArgs {
    int T, H, K, n0;
    const int32_t* parents;   // [T]
    const int32_t* rank;      // [T] child rank among the parent's children
    const int32_t* topk;      // [B][T][K] of the pass that just ran
    const float* f_hat;       // [B][T][H] predicted features of that pass
    int32_t* tokens;          // [B][T]
    float* feats;             // [B][T][H]
};
__global__ void __launch_bounds__(256) draft_expand_kernel(ExpandArgs a) {
    pdl_launch_dependents();
    pdl_wait();
    const int i = a.n0 + blockIdx.x, b = blockIdx.y;
    const int p = a.parents[i];
    if (threadIdx.x == 0) a.tokens[b * a.T + i] = a.topk[((size_t)b * a.T + p) * a.K + a.rank[i]];
    const float4* src = reinterpret_cast<const float4*>(a.f_hat + ((size_t)b * a.T + p) * a.H);
    float4* dst = reinterpret_cast<float4*>(a.feats + ((size_t)b * a.T + i) * a.H);
    for (int k = threadIdx.x; k < a.H / 4; k += 256) dst[k] = src[k];
}

// ---- after a target verify step: the chain the drafter must absorb.  Row j (j <= a) of sequence b: token = the accepted
// node's token (j = 0: the root), predecessor feature = the target feature of the accepted node before it (j = 0: the
// feature carried over from the previous step); also hands out the next root (bonus token) and its predecessor feature.
// grid (T, B) ----
struct GatherArgs {
    int T, H;
    const int32_t* tokens;        // [B][T] the verified tree
    const int32_t* accept_len;    // [B]
    const int32_t* accept_nodes;  // [B][T]
    const int32_t* out_tokens;    // [B][T]
    const float* feat;            // [B][T][H] target features of the verified tree (dev_final_hidden)
    float* carry;                 // [B][H] in: predecessor feature of the old root; out: of the new root
    int32_t* ext_tokens;          // [B][T]
    float* ext_feats;             // [B][T][H]
    int32_t* ext_n;               // [B] = a + 1
    int32_t* next_root;           // [B]
};
__global__ void __launch_bounds__(256) gather_accepted_kernel(GatherArgs a) {
    const int j = blockIdx.x, b = blockIdx.y;
    const int n = a.accept_len[b];
    if (j > n) return;
    const int node = a.accept_nodes[b * a.T + j];
    if (threadIdx.x == 0) {
        a.ext_tokens[b * a.T + j] = a.tokens[b * a.T + node];
        if (j == 0) { a.ext_n[b] = n + 1; a.next_root[b] = a.out_tokens[b * a.T + n]; }
    }
    const float* src = j == 0 ? a.carry + (size_t)b * a.H : a.feat + ((size_t)b * a.T + a.accept_nodes[b * a.T + j - 1]) * a.H;
    float* dst = a.ext_feats + ((size_t)b * a.T + j) * a.H;
    for (int k = threadIdx.x; k < a.H; k += 256) dst[k] = src[k];
}
// second half (separate launch: the carry may only be overwritten after every row has read it)
__global__ void __launch_bounds__(256) carry_update_kernel(GatherArgs a) {
    const int b = blockIdx.x;
    const int n = a.accept_len[b];
    const float* src = a.feat + ((size_t)b * a.T + a.accept_nodes[b * a.T + n]) * a.H;
    for (int k = threadIdx.x; k < a.H; k += 256) a.carry[(size_t)b * a.H + k] = src[k];
}

}  // namespace ev
