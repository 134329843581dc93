// C-ABI implementation (include/eagle_verify.h): handles, quantized-weight storage, page pool,
// and the verify-step schedule.  Every step of the path runs in the kernels of ev_*.cuh; the host
// code here only validates arguments, owns memory and enqueues launches on the caller's stream.
#include "../../include/eagle_verify.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "ev_attention.cuh"
#include "ev_attention_tc.cuh"
#include "ev_common.cuh"
#include "ev_drafter.cuh"
#include "ev_elementwise.cuh"
#include "ev_gemm.cuh"

using namespace ev;

// ------------------------------------------------------------------------------------------------
namespace {

thread_local std::string g_err;
thread_local long g_launches = 0;
thread_local long g_captures = 0;

int fail(int code, const std::string& msg) {
    g_err = msg;
    return code;
}
#define CUDA_TRY(expr)                                                                                    \
    do {                                                                                                  \
        cudaError_t _e = (expr);                                                                          \
        if (_e != cudaSuccess)                                                                            \
            return fail(EV_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(_e) + " @" + std::to_string(__LINE__)); \
    } while (0)
#define LAUNCH_CHECK()                                                                                    \
    do {                                                                                                  \
        ++g_launches;                                                                                     \
        cudaError_t _e = cudaGetLastError();                                                              \
        if (_e != cudaSuccess)                                                                            \
            return fail(EV_ECUDA, std::string("kernel launch: ") + cudaGetErrorString(_e) + " @" + std::to_string(__LINE__)); \
    } while (0)
#define EV_TRY(expr)                \
    do {                            \
        int _r = (expr);            \
        if (_r != EV_OK) return _r; \
    } while (0)

typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
PFN_encodeTiled g_encode = nullptr;

int get_encode() {
    if (g_encode) return EV_OK;
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q);
    if (e != cudaSuccess || q != cudaDriverEntryPointSuccess || !fn)
        return fail(EV_ECUDA, "cuTensorMapEncodeTiled entry point not available (no CUDA driver?)");
    g_encode = (PFN_encodeTiled)fn;
    return EV_OK;
}

// 2-D uint8 tensor [rows][cols] (cols contiguous), box = [box_rows][128 bytes], 128-byte swizzle
int make_tmap(CUtensorMap* tm, const void* base, long rows, long cols, int box_rows) {
    EV_TRY(get_encode());
    cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)cols};
    cuuint32_t box[2] = {128u, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1u, 1u};
    CUresult r = g_encode(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(base), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(EV_ECUDA, "cuTensorMapEncodeTiled failed, code " + std::to_string((int)r));
    return EV_OK;
}

// KV pool as a 4-D tensor of 2-byte elements over its rows = (layer, page, K|V, head, token) of D elements:
// (64 elements of a 128-byte half row, 8 rows of a swizzle group, D/64 half rows, rows/8 groups).  A box of
// (64, 8, D/64, 2) is one whole 16-token (page, K|V, head) block - 4 KiB contiguous in HBM at D = 128 - and lands
// in shared memory as [group][half][8 rows x 128 B]: every 1-KiB swizzle atom whole, 8-row groups of one half
// D/64 KiB apart (the UMMA stride byte offset).  One TMA instruction per block instead of one per half block.
int make_tmap_kv(CUtensorMap* tm, const void* base, long rows, int D) {
    EV_TRY(get_encode());
    cuuint64_t dims[4] = {64u, 8u, (cuuint64_t)(D / 64), (cuuint64_t)(rows / 8)};
    cuuint64_t strides[3] = {(cuuint64_t)D * 2, 128u, (cuuint64_t)D * 2 * 8};
    cuuint32_t box[4] = {64u, 8u, (cuuint32_t)(D / 64), (cuuint32_t)(TCA_PAGE / 8)};
    cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    CUresult r = g_encode(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 4, const_cast<void*>(base), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(EV_ECUDA, "cuTensorMapEncodeTiled (KV pool) failed, code " + std::to_string((int)r));
    return EV_OK;
}

constexpr int N_TOK_VARIANTS = 16;  // token-tile sizes 16, 32, ..., 256

struct ActBuf {  // an E4M3 activation buffer [rows_pad][K] + per-token scales, with one TMA map per token-tile size
    uint8_t* codes = nullptr;
    float* scale = nullptr;
    long K = 0;
    CUtensorMap tm[N_TOK_VARIANTS];
    CUtensorMap tmh[N_TOK_VARIANTS];   // half tiles (8, 16, ..., 128 rows): one CTA's share of a CTA pair's token tile
    CUtensorMap* tms_dev = nullptr;    // device copy: box heights 8, 16, ..., 256 rows (the balanced partition picks per item)
};

struct QMat {  // a quantized weight matrix [N][K], codes in the GEMM's tiled HBM layout (ev_gemm.cuh)
    uint8_t* codes = nullptr;  // [n_tiles][total_kb][16 KiB]
    float* scale = nullptr;    // [N]
    long N = 0, K = 0;
    int n_tiles = 0, total_kb = 0;
};

struct LayerW {
    QMat qkv, o, gu, down;
    __nv_bfloat16* g1 = nullptr;
    __nv_bfloat16* g2 = nullptr;
    unsigned have = 0;  // bit per ev_weight_kind
};

long round_up(long x, long m) { return (x + m - 1) / m * m; }

enum ProfClass { PC_GEMM_QKV = 0, PC_GEMM_O, PC_GEMM_GATEUP, PC_GEMM_DOWN, PC_GEMM_LM, PC_ATTN, PC_ATTN_MERGE, PC_NORM_QUANT,
                 PC_ROPE_KV, PC_SWIGLU, PC_OTHER, PC_COUNT };
struct ProfRec { cudaEvent_t a, b; int cls; };

struct AttnPlan { int n_splits, split_len; };
constexpr int TRACE_CAP = 1024;
struct GraphKey {
    int B, T, commit, force_all, n_splits, split_len, need_lm, pad;
    const void* p[16];
};
struct GraphEntry { GraphKey key; cudaGraphExec_t exec; long launches; unsigned long stamp; };
constexpr size_t MAX_GRAPHS = 16;

}  // namespace

struct ev_model {
    ev_config cfg;
    int M_cap = 0, M_pad = 0, qkv_dim = 0, q_dim = 0, kv_dim = 0, max_pos = 0;
    std::vector<LayerW> layers;
    QMat lm;
    __nv_bfloat16* embed = nullptr;
    __nv_bfloat16* gf = nullptr;
    bool have_embed = false, have_lm = false;
    float2* rope_cs = nullptr;
    // workspaces
    float* h = nullptr;
    ActBuf xq, aq, tq;
    float* qkv = nullptr;
    float* attn = nullptr;
    float* o_part = nullptr;
    float* ml_part = nullptr;
    float* lin_out = nullptr;   // raw GEMM output [splits][M][N], consumed by the next element-wise kernel
    long lin_floats = 0;
    unsigned long long* trace = nullptr;   // ev_profile_enable(m, 2): [TRACE_CAP][TRACE_SLOTS] step trace, see ev_profile_trace
    bool trace_on = false;
    int n_traced = 0;
    // tree state
    int32_t *attn_order = nullptr;
    int32_t *Lsnap = nullptr, *nn_eff = nullptr, *depth = nullptr, *pos = nullptr;
    unsigned long long *anc = nullptr, *anc_bulk = nullptr, *argmax_keys = nullptr;
    int32_t *erow = nullptr, *kend_row = nullptr, *kend_seq = nullptr;   // bulk / tail cut of every row's key set (tree_prep_kernel)
    int attn_chunk = 1024, n_chunks_max = 1;   // keys per attention chunk (cfg.attn_chunk); chunk columns the partial workspace holds
    // static activation scales
    int n_sites = 0;
    float* static_scales = nullptr;  // device [n_sites]
    float* site_amax = nullptr;      // device [n_sites]
    float* w_amax = nullptr;         // device scalar: absmax of the matrix being quantized (per-tensor weight scales)
    unsigned long long* clip_counts = nullptr;  // device [n_sites]: elements clipped by the static scales since the last reset
    bool calibrated = false, recording = false;
    // FP8 KV cache (cfg.kv_dtype 1): static per-tensor scales of every layer's K and V cache, [2 * n_layers] = (K, V) per layer
    float* kv_amax = nullptr;          // device: calibration accumulators
    std::vector<float> kv_scales;      // host copy (kernel arguments)
    bool kv_calibrated = false;
    int num_sms = 148;
    int cut_pairs = 74;   // pieces of the canonical K cuts of every layer matrix (ev_gemm.cuh): a constant of the library, NOT the
                          // SM count of the device, so results do not change with the GPU the model runs on (148 SMs = 74 pairs)
    int row_cluster = 0;  // EV_ROW_CLUSTER override (bring-up)
    bool profile = false;
    // L2 weight stream (PfPlanner): on for token counts <= l2pf_max_m; bytes the stream may run ahead / per launch
    int l2pf_max_m = 0;
    long l2pf_cap = 88L << 20, l2pf_maxq = 40L << 20;
    unsigned l2pf_mask = 0xFFFFFFFFu;
    std::vector<ProfRec> prof;
    size_t prof_used = 0;
    // captured verify steps (CUDA graphs), keyed by everything a launch depends on
    bool use_graph = true;
    cudaStream_t cap_stream = nullptr;
    std::vector<GraphEntry> graphs;
    unsigned long graph_clock = 0;
    // draft side (ev_drafter.cuh): EAGLE front end and tree-expansion workspaces; all null / empty on a target model
    QMat fc;                         // EV_W_DRAFT_FC [H][2H]
    bool have_fc = false, shared_head = false;
    ActBuf fq;                       // codes of [embed ; feature], K = 2H
    float* logits_ws = nullptr;      // [M_cap][vocab] when top-k is asked for without a logits output
    int32_t* d_topk = nullptr;       // [M_cap][TOPK_MAX]
    float* d_fhat = nullptr;         // [M_cap][H] predicted features of the last drafter pass
    float* d_feats = nullptr;        // [M_cap][H] predecessor features of the tree being drafted
    int32_t* d_scratch = nullptr;    // required verify outputs of the drafter passes nobody reads
    int32_t* d_topo = nullptr;       // [2][T] parents, child ranks of the static topology
    int32_t* d_lvl_n = nullptr;      // [levels][max_batch] nodes in use per level
    std::vector<int32_t> h_topo;     // host copy of the topology last uploaded
    int32_t* d_tree_par = nullptr;   // [M_cap] that topology replicated per sequence (row stride T)
    int32_t* d_chain_par = nullptr;  // [M_cap] chain parents (i - 1) at row stride chain_T
    int chain_T = 0;
    std::vector<void*> allocs;
    std::vector<ev_cache*> caches;   // caches created on this model (their model pointer is cleared if the model dies first)
};

struct ev_cache {
    ev_model* model = nullptr;
    long n_pages = 0;
    int max_seqs = 0, max_pages = 0;
    long layer_stride = 0;  // elements
    __nv_bfloat16* pool = nullptr;
    int32_t* page_table = nullptr;  // device [max_seqs][max_pages]
    int32_t* ctx_len = nullptr;     // device [max_seqs]
    int32_t* capacity = nullptr;    // device [max_seqs]
    std::vector<int> free_pages;
    std::vector<std::vector<int>> seq_pages;
    std::vector<char> seq_used;
    std::vector<int> len_bound;  // host-side upper bound of each sequence's ctx_len (sizes the key-split grid)
    CUtensorMap tmKV;            // whole pool, for the tcgen05 attention kernel
    bool tc_attn = false;        // page_size == 16 and the pool fits 32-bit row coordinates
    bool kv_f16 = false;         // the pool keeps the bf16-rounded K/V values in binary16 containers (tcgen05 attention; ev_common.cuh)
    bool kv_fp8 = false;         // the pool keeps E4M3 codes, one byte per element (cfg.kv_dtype 1)
    int eb = 2;                  // bytes per pool element
    // prefill staging
    int32_t *pf_tokens = nullptr, *pf_parents = nullptr, *pf_nn = nullptr, *pf_slots = nullptr;
    int32_t *pf_out = nullptr;
};

namespace {

// records a CUDA-event pair around the launches issued in its scope when profiling is on
struct ProfScope {
    ev_model* m; cudaStream_t st; ProfRec* r = nullptr;
    ProfScope(ev_model* m_, cudaStream_t st_, int cls) : m(m_), st(st_) {
        if (!m->profile) return;
        if (m->prof_used == m->prof.size()) {
            ProfRec n;
            cudaEventCreate(&n.a); cudaEventCreate(&n.b);
            m->prof.push_back(n);
        }
        r = &m->prof[m->prof_used++];
        r->cls = cls;
        cudaEventRecord(r->a, st);
    }
    ~ProfScope() { if (r) cudaEventRecord(r->b, st); }
};

template <class T>
int dev_alloc(ev_model* m, T** p, size_t count) {
    void* q = nullptr;
    cudaError_t e = cudaMalloc(&q, count * sizeof(T) > 0 ? count * sizeof(T) : 16);
    if (e != cudaSuccess) return fail(EV_ENOMEM, std::string("cudaMalloc: ") + cudaGetErrorString(e));
    if (m) m->allocs.push_back(q);
    *p = (T*)q;
    return EV_OK;
}

int alloc_actbuf(ev_model* m, ActBuf* b, long K) {
    b->K = K;
    EV_TRY(dev_alloc(m, &b->codes, (size_t)m->M_pad * K));
    EV_TRY(dev_alloc(m, &b->scale, (size_t)m->M_pad));
    cudaMemset(b->codes, 0, (size_t)m->M_pad * K);
    for (int i = 0; i < N_TOK_VARIANTS; ++i) EV_TRY(make_tmap(&b->tm[i], b->codes, m->M_pad, K, 16 * (i + 1)));
    for (int i = 0; i < N_TOK_VARIANTS; ++i) EV_TRY(make_tmap(&b->tmh[i], b->codes, m->M_pad, K, 8 * (i + 1)));
    CUtensorMap all[2 * N_TOK_VARIANTS];
    for (int i = 0; i < 2 * N_TOK_VARIANTS; ++i) EV_TRY(make_tmap(&all[i], b->codes, m->M_pad, K, 8 * (i + 1)));
    EV_TRY(dev_alloc(m, &b->tms_dev, (size_t)2 * N_TOK_VARIANTS));
    CUDA_TRY(cudaMemcpy(b->tms_dev, all, sizeof(all), cudaMemcpyHostToDevice));
    return EV_OK;
}

int alloc_qmat(ev_model* m, QMat* q, long N, long K) {
    q->N = N;
    q->K = K;
    q->n_tiles = (int)round_up((N + GEMM_WROWS - 1) / GEMM_WROWS, 2);   // whole PAIRS of 128-channel tiles (canonical K cuts, CTA pairs)
    q->total_kb = (int)((K + GEMM_BK - 1) / GEMM_BK);
    const size_t bytes = (size_t)q->n_tiles * q->total_kb * GEMM_WTILE;
    EV_TRY(dev_alloc(m, &q->codes, bytes));
    EV_TRY(dev_alloc(m, &q->scale, (size_t)N));
    if (cudaMemset(q->codes, 0, bytes) != cudaSuccess) return fail(EV_ECUDA, "memset");  // K / N padding stays zero
    return EV_OK;
}


// Every kernel of the step is launched with the programmatic-stream-serialization attribute (PDL): it may
// become resident while its predecessor is still running, and executes griddepcontrol.wait before touching
// anything the predecessor wrote.  Under stream capture these launches become programmatic graph edges.
// ONE launch per step goes without it: the kernel right after tree_prep_kernel (serial_next_launch()).  It then starts only
// when tree_prep_kernel has completed, and since a PDL kernel can become resident only after every CTA of its predecessor has
// started, no later kernel of the step runs a single instruction before that either: the per-step metadata tree_prep_kernel
// writes (Lsnap, nn_eff, order, erow, ...) may be read ahead of griddepcontrol.wait (tree_attn_tc_kernel does).
bool g_use_pdl = true;
thread_local bool g_serial_next = false;
void serial_next_launch() { g_serial_next = true; }
template <class... KArgs, class... Args>
int launch_kc(int cluster, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[2];
    int na = 0;
    const bool serial = g_serial_next;
    g_serial_next = false;
    if (g_use_pdl && !serial) {
        at[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    if (cluster > 1) {  // grid.x counts CTAs: a multiple of the cluster size
        at[na].id = cudaLaunchAttributeClusterDimension;
        at[na].val.clusterDim.x = cluster; at[na].val.clusterDim.y = 1; at[na].val.clusterDim.z = 1;
        ++na;
    }
    cfg.attrs = at;
    cfg.numAttrs = na;
    cudaError_t e = cudaLaunchKernelEx(&cfg, kern, args...);
    if (e != cudaSuccess) return fail(EV_ECUDA, std::string("kernel launch: ") + cudaGetErrorString(e));
    ++g_launches;
    return EV_OK;
}
template <class... KArgs, class... Args>
int launch_k(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    return launch_kc(1, kern, grid, block, smem, st, args...);
}
// Shape of a row kernel launch (RMSNorm / SwiGLU / attention merge; ev_elementwise.cuh): cl CTAs of ROW_THREADS
// threads per token row (one cluster), nv4 float4s per thread.  Few rows are spread over many CTAs so that they
// still occupy every SM (cl up to 8); many rows keep nv4 <= 4 so that several CTAs stay resident per SM.
struct RowPlan { int cl, nv4; };
int pow2_ceil(long x) { int p = 1; while (p < x) p <<= 1; return p; }
RowPlan row_plan(const ev_model* m, int M, int row_floats, int cl_par_max = CLUSTER_MAX) {
    const long row4 = (row_floats + 3) / 4;
    int cl_par = 1;
    while (cl_par < cl_par_max && (long)M * cl_par * 2 <= 4L * m->num_sms) cl_par <<= 1;
    cl_par = std::min(cl_par, pow2_ceil((row4 + ROW_THREADS - 1) / ROW_THREADS));
    const int cl_need = pow2_ceil((row4 + 4L * ROW_THREADS - 1) / (4L * ROW_THREADS));
    RowPlan p;
    p.cl = std::max(cl_par, cl_need);
    if (m->row_cluster > 0) p.cl = std::max(pow2_ceil(m->row_cluster), cl_need);
    p.cl = std::min(p.cl, CLUSTER_MAX);
    p.nv4 = pow2_ceil((row4 + (long)ROW_THREADS * p.cl - 1) / ((long)ROW_THREADS * p.cl));
    return p;
}
#define ROW_DISPATCH(plan, KERN, ...)                                                                          \
    do {                                                                                                       \
        if ((plan).nv4 == 1) EV_TRY(launch_kc((plan).cl, KERN<1>, __VA_ARGS__));                               \
        else if ((plan).nv4 == 2) EV_TRY(launch_kc((plan).cl, KERN<2>, __VA_ARGS__));                          \
        else if ((plan).nv4 == 4) EV_TRY(launch_kc((plan).cl, KERN<4>, __VA_ARGS__));                          \
        else return fail(EV_EINVAL, "row too long for the row kernels");                                       \
    } while (0)

// row kernels that consume a LinOut: also instantiated for the slab-count bound (1 / 3 / 8) so that the
// no-split case (M > 256) does not issue seven predicated-off slab loads and adds per element
#define ROW_DISPATCH_S(plan, splits, KERN, ...)                                                                \
    do {                                                                                                       \
        const int s_ = (splits);                                                                               \
        if (s_ <= 1) ROW_DISPATCH_S1(plan, 1, KERN, __VA_ARGS__);                                              \
        else if (s_ <= 3) ROW_DISPATCH_S1(plan, 3, KERN, __VA_ARGS__);                                         \
        else ROW_DISPATCH_S1(plan, 8, KERN, __VA_ARGS__);                                                      \
    } while (0)
#define ROW_DISPATCH_S1(plan, S, KERN, ...)                                                                    \
    do {                                                                                                       \
        if ((plan).nv4 == 1) EV_TRY(launch_kc((plan).cl, KERN<1, S>, __VA_ARGS__));                            \
        else if ((plan).nv4 == 2) EV_TRY(launch_kc((plan).cl, KERN<2, S>, __VA_ARGS__));                       \
        else if ((plan).nv4 == 4) EV_TRY(launch_kc((plan).cl, KERN<4, S>, __VA_ARGS__));                       \
        else return fail(EV_EINVAL, "row too long for the row kernels");                                       \
    } while (0)

// cudaFuncSetAttribute is per device: one flag per (kernel instantiation, device)
inline bool& attr_flag(bool (&flags)[64]) {
    int dev = 0;
    cudaGetDevice(&dev);
    return flags[dev & 63];
}

template <int EPI, bool PAIR>
int launch_gemm(cudaStream_t st, const CUtensorMap& tmX, const CUtensorMap& tmXh, const GemmArgs& a, int grid, int smem) {
    static bool flags[64] = {};
    bool& attr_set = attr_flag(flags);
    if (!attr_set) {
        CUDA_TRY(cudaFuncSetAttribute(gemm_e4m3_kernel<EPI, PAIR>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        attr_set = true;
    }
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(gemm_threads<EPI, PAIR>());
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;  // PDL: weight prefetch overlaps the previous kernel
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    if (PAIR) {  // CTA pairs: clusters of 2 CTAs along x
        at[1].id = cudaLaunchAttributeClusterDimension;
        at[1].val.clusterDim.x = 2; at[1].val.clusterDim.y = 1; at[1].val.clusterDim.z = 1;
        cfg.numAttrs = 2;
    }
    CUDA_TRY(cudaLaunchKernelEx(&cfg, gemm_e4m3_kernel<EPI, PAIR>, tmX, tmXh, a));
    ++g_launches;
    return EV_OK;
}

template <int MAXS>
int launch_swiglu_s(ev_model* m, cudaStream_t st, bool smem_form, RowPlan rp, int M, const LinOut& gu, int F, float* tap, const QuantOut& q,
                    const L2Prefetch& pf) {
    if (smem_form) {
        static bool flags[64] = {};
        bool& attr_set = attr_flag(flags);
        if (!attr_set) {
            CUDA_TRY(cudaFuncSetAttribute(swiglu_quant_smem_kernel<MAXS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024));
            attr_set = true;
        }
        return launch_k(swiglu_quant_smem_kernel<MAXS>, dim3(M), dim3(SWI_THREADS), (size_t)F * 4, st, gu, F, tap, q, pf);
    }
    if (rp.nv4 == 1) return launch_kc(rp.cl, swiglu_quant_kernel<1, MAXS>, dim3(M * rp.cl), dim3(SWI_THREADS), 0, st, gu, F, tap, q, pf);
    if (rp.nv4 == 2) return launch_kc(rp.cl, swiglu_quant_kernel<2, MAXS>, dim3(M * rp.cl), dim3(SWI_THREADS), 0, st, gu, F, tap, q, pf);
    if (rp.nv4 == 4) return launch_kc(rp.cl, swiglu_quant_kernel<4, MAXS>, dim3(M * rp.cl), dim3(SWI_THREADS), 0, st, gu, F, tap, q, pf);
    return fail(EV_EINVAL, "row too long for the row kernels");
}
int launch_swiglu(ev_model* m, cudaStream_t st, bool smem_form, RowPlan rp, int M, const LinOut& gu, int F, float* tap, const QuantOut& q,
                  const L2Prefetch& pf) {
    if (gu.splits <= 1) return launch_swiglu_s<1>(m, st, smem_form, rp, M, gu, F, tap, q, pf);
    if (gu.splits <= 3) return launch_swiglu_s<3>(m, st, smem_form, rp, M, gu, F, tap, q, pf);
    return launch_swiglu_s<8>(m, st, smem_form, rp, M, gu, F, tap, q, pf);
}

// Host side of the L2 weight stream (L2Prefetch, ev_common.cuh).  segs = the weight matrices of the step in
// the order the GEMMs consume them.  Every kernel launch of the step takes the next slice: at most `maxq`
// bytes, and never more than `cap` bytes ahead of the start of the most recently launched GEMM's weights
// (that GEMM may still be reading them when the slice is issued, one PDL stage early).
struct PfPlanner {
    std::vector<std::pair<const uint8_t*, size_t>> segs;
    std::vector<size_t> start;   // prefix sums, start[i] = first stream byte of segs[i]; start.back() = total
    size_t cursor = 0;           // stream bytes already covered (prefetched, or read directly by their GEMM)
    int next_gemm = 0;
    size_t cap = 0, maxq = 0;
    bool on = false;
    unsigned mask = 0xFFFFFFFFu;   // which launches of a layer may issue (bit = position in the layer's 10-kernel sequence:
    int n_take = 0, per_layer = 10, n_layer_launches = 0;   // norm1 qkv rope attn merge o norm2 gu swiglu down; bit 10 = final norm / LM head)
    unsigned long long* trace = nullptr;  // step trace (ev_profile_trace): 4 slots per launch, in launch order
    int n_traced = 0, trace_cap = 0;
    void add(const uint8_t* p, size_t n) {
        if (start.empty()) start.push_back(0);
        segs.push_back({p, n});
        start.push_back(start.back() + n);
    }
    L2Prefetch take(bool is_gemm) {
        L2Prefetch pf;
        pf.p[0] = pf.p[1] = nullptr; pf.n[0] = pf.n[1] = 0;
        pf.trace = (trace && n_traced < trace_cap) ? trace + TRACE_SLOTS * (size_t)n_traced++ : nullptr;
        if (!on || segs.empty()) return pf;
        if (is_gemm && next_gemm < (int)segs.size()) {  // this GEMM reads its own weights: nothing of them is left to prefetch
            cursor = std::max(cursor, start[next_gemm + 1]);
            ++next_gemm;
        }
        const int pos = n_take < n_layer_launches ? n_take % per_layer : per_layer;
        ++n_take;
        if (!((mask >> pos) & 1u)) return pf;
        const size_t consumed = start[std::max(0, next_gemm - 1)];
        const size_t ahead = cursor - std::min(cursor, consumed);
        if (ahead >= cap) return pf;
        size_t quota = std::min(maxq, cap - ahead);
        quota -= quota % L2PF_CHUNK;
        int piece = 0;
        while (quota > 0 && piece < 2 && cursor < start.back()) {
            int si = (int)(std::upper_bound(start.begin(), start.end(), cursor) - start.begin()) - 1;
            const size_t off = cursor - start[si];
            size_t n = std::min(quota, segs[si].second - off);
            n -= n % L2PF_CHUNK;
            if (n == 0) { cursor = start[si + 1]; continue; }
            pf.p[piece] = segs[si].first + off;
            pf.n[piece] = (unsigned)n;
            ++piece;
            cursor += n;
            quota -= n;
            if (segs[si].second - off - n < L2PF_CHUNK) cursor = start[si + 1];
        }
        return pf;
    }
};

// one W8A8 linear.  epi == EPI_RAW: raw accumulators go to m->lin_out as [slabs][M][N]; *lin describes them for
// the consumer kernel.  epi == EPI_ARGMAX (LM head): scales applied, argmax keys updated, optional logits.
// Two forms (ev_gemm.cuh), both cutting K at the matrix's canonical cuts (cut_G = m->cut_pairs pieces over the
// flattened (pair tile, K-block) space), so a token's result does not depend on how many tokens share the launch:
//   M <= 256 (one token tile): stream-K over CTA pairs of single CTAs, piece c = work of pair c, slabs added by the consumer;
//   M  > 256: cta_group::2 pairs own whole (pair tile, token tile) items, running fp32 sum over the pieces in the epilogue.
int run_linear(ev_model* m, cudaStream_t st, const QMat& w, const ActBuf& x, int M, int epi, LinOut* lin, float* logits,
               unsigned long long* keys, int prof_cls, PfPlanner* pfp = nullptr, const void* warm1 = nullptr, int warm1_bytes = 0) {
    ProfScope prof_scope(m, st, prof_cls);
    if (lin) {
        lin->p = m->lin_out; lin->splits = 1; lin->ld = (int)w.N; lin->split_stride = (long)M * w.N;
        lin->sx = x.scale; lin->sw = w.scale; lin->sk_G = lin->sk_U = lin->sk_kb = 0;
    }
    GemmArgs a;
    a.M = M; a.N = (int)w.N; a.total_kb = w.total_kb; a.n_tiles = w.n_tiles;   // n_tiles is even (alloc_qmat)
    a.m_tiles = (M + 255) / 256;
    const bool pair = a.m_tiles >= 2;   // cta_group::2 kernel
    if (pair && epi == EPI_RAW) {
        // Token tiling of the many-row form is a scheduling choice (rows are independent, the K cuts do not move): an item is
        // (pair of channel tiles, token tile) and the CTA pairs take whole items.  When the default (fewest, widest tiles) does not
        // even fill ONE round of pairs, narrower tiles put more pairs to work at no cost in rounds: config[4] (480 rows) QKV 48 -> 72
        // items on 74 pairs (735 -> 665 us per step), down 32 -> 64 items (1,378 -> 1,094).  Beyond one round it does not pay - the
        // count rounds x tile width predicts -31 % for QKV at 832 rows (96 items of 208 -> 144 items of 144) and -17 % for gate|up at
        // 480; measured +5 % and +73 %: narrower tiles re-read W and pay the per-item hand-overs more often.
        const int pairs_avail = std::max(1, m->num_sms / 2), n_pairs_ = a.n_tiles / 2;
        if (n_pairs_ * a.m_tiles < pairs_avail)
            for (int mt = a.m_tiles + 1; mt <= 8 && n_pairs_ * mt <= pairs_avail; ++mt) a.m_tiles = mt;
    }
    a.tok = (int)round_up((M + a.m_tiles - 1) / a.m_tiles, 16);
    // balanced partition (ev_gemm.cuh, GemmArgs::bal): several token tiles -> items of up to 256 tokens cut from an even deal.
    // Used for the LM head (1002 n tiles: 27 items per CTA pair, 588 -> 548 us at M = 832).  The layer GEMMs have 1-6
    // items per pair; there the extra partial items (a 32-token item costs as much W traffic as a 208-token one)
    // outweigh the partial last wave: O 26 -> 33 us, down 54 -> 82 us, gate|up 98 -> 104 us.
    a.bal = (pair && epi == EPI_ARGMAX) ? 1 : 0;
    a.bal_blocks = (M + 15) / 16;
    a.tms = x.tms_dev;
    if (a.bal) a.tok = 256;   // the largest item: sizes the stages and the two accumulators
    const int stage_bytes = GEMM_WTILE + (pair ? a.tok / 2 : a.tok) * GEMM_BK;
    a.stages = std::min(GEMM_MAX_STAGES, GEMM_SMEM_BUDGET / stage_bytes);
    if (a.stages < 2) return fail(EV_EINVAL, "token tile too large");
    a.W = w.codes; a.sx = x.scale; a.sw = w.scale; a.argmax_keys = keys;
    a.out = (epi == EPI_RAW) ? m->lin_out : logits;
    a.ldo = (int)w.N;
    a.pf.p[0] = a.pf.p[1] = nullptr; a.pf.n[0] = a.pf.n[1] = 0; a.pf.trace = nullptr;
    a.warm[0] = (epi == EPI_RAW) ? w.scale : nullptr; a.warm_bytes[0] = (epi == EPI_RAW) ? (int)(w.N * sizeof(float)) : 0;
    a.warm[1] = warm1; a.warm_bytes[1] = warm1 ? warm1_bytes : 0;
    if (pfp) a.pf = pfp->take(true);
    a.k_splits = 1;
    a.kb_per_split = a.total_kb;
    a.sk_units = 0;
    a.cut_G = a.cut_U = 0;
    const int n_pairs = a.n_tiles / 2;
    const int U = n_pairs * a.total_kb;             // K-block units of the (pair tile, K-block) space
    const int cutG = std::min(std::min(m->cut_pairs, U), 7 * n_pairs);   // canonical pieces: matrix shape and a model constant only; <= 8 pieces per tile
    int pmax = 1;                                   // most pieces any pair tile is cut into
    for (int t = 0; t < n_pairs; ++t)
        pmax = std::max(pmax, sk_first_cta((t + 1) * a.total_kb - 1, cutG, U) - sk_first_cta(t * a.total_kb, cutG, U) + 1);
    int grid;
    if (epi == EPI_ARGMAX) {          // LM head: whole K per item, no cuts
        a.mc = pair ? 1 : 0;
        grid = pair ? 2 * std::min(n_pairs * a.bal_blocks, m->num_sms / 2) : std::min(a.n_tiles, m->num_sms);
    } else if (!pair) {               // stream-K: piece c = CTAs 2c, 2c+1
        if (pmax > 8 || (long)pmax * M * a.N > m->lin_floats) return fail(EV_EINVAL, "K cuts: more than 8 pieces per tile or slab workspace too small");
        a.mc = 1;
        a.sk_units = U;
        grid = 2 * cutG;
        if (lin) { lin->splits = pmax; lin->sk_G = cutG; lin->sk_U = U; lin->sk_kb = a.total_kb; }
    } else {                          // CTA pairs, whole items, running sum over the same pieces
        a.mc = 1;
        a.cut_G = cutG; a.cut_U = U;
        grid = 2 * std::min(n_pairs * a.m_tiles, m->num_sms / 2);
    }
    const int smem = a.stages * stage_bytes + 512 + 2048 + 8192 + 1024;  // stages + barriers + sx staging + argmax keys + alignment slack
    const CUtensorMap& tmX = x.tm[a.tok / 16 - 1];
    const CUtensorMap& tmXh = x.tmh[a.tok / 16 - 1];
    if (epi == EPI_RAW) return pair ? launch_gemm<EPI_RAW, true>(st, tmX, tmXh, a, grid, smem) : launch_gemm<EPI_RAW, false>(st, tmX, tmXh, a, grid, smem);
    return pair ? launch_gemm<EPI_ARGMAX, true>(st, tmX, tmXh, a, grid, smem) : launch_gemm<EPI_ARGMAX, false>(st, tmX, tmXh, a, grid, smem);
}

QuantOut quant_out(ev_model* m, ActBuf& b, int site) {
    QuantOut q;
    q.codes = b.codes;
    q.sx = b.scale;
    q.static_scale = (m->cfg.act_scale_mode == 1 && !m->recording) ? m->static_scales + site : nullptr;
    q.site_amax = m->recording ? m->site_amax + site : nullptr;
    q.clip_count = q.static_scale ? m->clip_counts + site : nullptr;
    return q;
}

int copy_f32(cudaStream_t st, const float* src, float* dst, long n) {
    CUDA_TRY(cudaMemcpyAsync(dst, src, (size_t)n * sizeof(float), cudaMemcpyDeviceToDevice, st));
    return EV_OK;
}

template <int D, bool FP8, bool SMALL = false>
int launch_attn_tc(cudaStream_t st, const CUtensorMap& tm, const TcAttnArgs& a, dim3 grid) {
    static bool flags[64] = {};
    bool& attr_set = attr_flag(flags);
    if (!attr_set) {
        CUDA_TRY(cudaFuncSetAttribute(tree_attn_tc_kernel<D, FP8, SMALL>, cudaFuncAttributeMaxDynamicSharedMemorySize, TcaCfg<D, FP8, SMALL>::SMEM));
        attr_set = true;
    }
    return launch_k(tree_attn_tc_kernel<D, FP8, SMALL>, grid, dim3(TcaCfg<D, FP8, SMALL>::THREADS), TcaCfg<D, FP8, SMALL>::SMEM, st, tm, a);
}

template <int D>
int launch_attn(cudaStream_t st, const AttnArgs& a, dim3 grid) {
    constexpr int smem = 2 * 2 * ATT_CH * D * 2 + ATT_WARPS * 3 * 16 * D * 2;
    static bool flags[64] = {};
    bool& attr_set = attr_flag(flags);
    if (!attr_set) {
        CUDA_TRY(cudaFuncSetAttribute(tree_attn_partial_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        attr_set = true;
    }
    return launch_k(tree_attn_partial_kernel<D>, grid, dim3(ATT_THREADS), smem, st, a);
}


// Attention grid: n_chunks chunk columns of cfg.attn_chunk keys each (ev_attention.cuh).  The chunk length is a constant
// of the model - which keys share a chunk never depends on the batch - so the plan only says how many chunk columns the
// grid has: enough for the longest sequence the host knows of (len_bound, an upper bound of ctx_len; the kernels read the
// true lengths on the device, CTAs of empty chunks leave at once, and tree_prep rejects a sequence the grid does not cover).
AttnPlan plan_attention(ev_model* m, ev_cache* c, const ev_verify_in* in) {
    const int T = in->n_nodes_max;
    int max_keys = 0;
    for (int i = 0; i < c->max_seqs; ++i)
        if (c->seq_used[i]) max_keys = std::max(max_keys, c->len_bound[i]);
    max_keys += T;
    if (in->commit)   // the host does not see which nodes are accepted: every sequence may grow by T (ev_verify_host and ev_cache_get_len tighten the bound)
        for (int i = 0; i < c->max_seqs; ++i)
            if (c->seq_used[i]) c->len_bound[i] = std::min(c->len_bound[i] + T, (int)c->seq_pages[i].size() * m->cfg.page_size);
    AttnPlan p;
    p.split_len = m->attn_chunk;
    int need = std::max(1, (max_keys + p.split_len - 1) / p.split_len);
    // short chunks (models built for one or two sequences): a growing sequence crosses a chunk boundary every few dozen steps and
    // every new column count is a new CUDA graph - round the column count up to a power of two (the CTAs of empty columns leave at once)
    if (p.split_len <= 512) need = pow2_ceil(need);
    p.n_splits = std::min(m->n_chunks_max, need);
    return p;
}

// the verify-step schedule; max_keys_hint: upper bound of ctx_len + T over the
// batch known to the host (sizes the key-split grid; the kernels read the true lengths on the device)
int run_forward(ev_model* m, ev_cache* c, const ev_verify_in* in, ev_verify_out* out, cudaStream_t st, bool need_lm, AttnPlan plan) {
    const ev_config& cfg = m->cfg;
    const int B = in->n_seqs, T = in->n_nodes_max, M = B * T;
    const int H = cfg.hidden, D = cfg.head_dim, F = cfg.ffn;

    TreePrepArgs tp;
    tp.B = B; tp.T = T; tp.vocab = cfg.vocab; tp.page_size = cfg.page_size;
    tp.seq_slots = in->dev_seq_slots; tp.tokens = in->dev_tokens; tp.parents = in->dev_parents; tp.n_nodes = in->dev_n_nodes;
    tp.ctx_len = c->ctx_len; tp.capacity = c->capacity; tp.max_seqs = c->max_seqs; tp.max_pos = m->max_pos;
    tp.Lsnap = m->Lsnap; tp.nn_eff = m->nn_eff; tp.status = out->dev_status; tp.depth = m->depth; tp.pos = m->pos;
    tp.anc = m->anc; tp.argmax_keys = m->argmax_keys; tp.order = m->attn_order;
    tp.anc_bulk = m->anc_bulk; tp.erow = m->erow; tp.kend_row = m->kend_row; tp.kend_seq = m->kend_seq;
    tp.max_keys = plan.n_splits * plan.split_len;
    EV_TRY(launch_k(tree_prep_kernel, dim3((B + 63) / 64), dim3(64), 0, st, tp));

    const float* ovr = in->dev_hidden_override;
    if (ovr) {
        EV_TRY(copy_f32(st, ovr, m->h, (long)M * H));
    } else if (in->dev_features) {
        // draft model (ev_drafter.cuh): layer-0 input = FC(Q8([embed(token) ; predecessor feature]))
        QuantOut q;
        q.codes = m->fq.codes; q.sx = m->fq.scale; q.static_scale = nullptr; q.site_amax = nullptr; q.clip_count = nullptr;
        serial_next_launch();
        EV_TRY(launch_k(concat_quant_kernel, dim3(M), dim3(EW_THREADS), 0, st, in->dev_tokens, cfg.vocab, m->embed, in->dev_features, H, q));
        LinOut fl;
        EV_TRY(run_linear(m, st, m->fc, m->fq, M, EPI_RAW, &fl, nullptr, nullptr, PC_OTHER));
        EV_TRY(launch_k(materialize_linear_kernel, dim3(M), dim3(256), 0, st, m->h, H, fl));
    } else {
        serial_next_launch();
        EV_TRY(launch_k(embed_gather_kernel, dim3(M), dim3(EW_THREADS), 0, st, in->dev_tokens, cfg.vocab, m->embed, H, m->h));
    }
    if (out->dev_hidden) EV_TRY(copy_f32(st, m->h, out->dev_hidden, (long)M * H));

    // L2 weight stream: the step's weight matrices in consumption order (PfPlanner)
    PfPlanner pfp;
    pfp.on = M <= m->l2pf_max_m && !m->profile;
    pfp.cap = (size_t)m->l2pf_cap; pfp.maxq = (size_t)m->l2pf_maxq;
    pfp.trace = m->trace_on ? m->trace : nullptr; pfp.trace_cap = TRACE_CAP;
    pfp.mask = m->l2pf_mask; pfp.n_layer_launches = 10 * cfg.n_layers;
    if (pfp.on) {
        auto qbytes = [](const QMat& q) { return (size_t)q.n_tiles * q.total_kb * GEMM_WTILE; };
        for (int l = 0; l < cfg.n_layers; ++l) {
            LayerW& w = m->layers[l];
            pfp.add(w.qkv.codes, qbytes(w.qkv)); pfp.add(w.o.codes, qbytes(w.o));
            pfp.add(w.gu.codes, qbytes(w.gu)); pfp.add(w.down.codes, qbytes(w.down));
        }
        if (need_lm) pfp.add(m->lm.codes, qbytes(m->lm));
    }

    const int n_splits = plan.n_splits, split_len = plan.split_len;
    const RowPlan rp_h = row_plan(m, M, H), rp_f = row_plan(m, M, F, CLUSTER_MAX), rp_q = row_plan(m, M, m->q_dim);
    // many rows: one CTA per row, row staged in smem.  Measured cross-over with the register / cluster form: 480 rows 950 (smem) vs 778 us
    // per step (clusters of 4), 832 rows 1,222 vs 1,379
    const bool swi_smem = M > 4 * m->num_sms && (size_t)F * 4 <= 160 * 1024;
    const int rope_gy = (long)M * 4 <= 4L * m->num_sms ? 4 : 2;
    const int row_groups = (T * (cfg.n_q_heads / cfg.n_kv_heads) + 16 * ATT_WARPS - 1) / (16 * ATT_WARPS);

    LinOut pend;           // raw output of the last O / down GEMM, not yet added to the residual stream
    pend.p = nullptr;
    LinOut none;
    none.p = nullptr; none.splits = 0; none.ld = 0; none.split_stride = 0; none.sx = nullptr; none.sw = nullptr;
    none.sk_G = none.sk_U = none.sk_kb = 0;
    pend = none;
    auto materialize = [&]() -> int {  // h += pending (only for debug taps; the fast path fuses this into RMSNorm)
        if (!pend.p) return EV_OK;
        EV_TRY(launch_k(apply_pending_kernel, dim3(M), dim3(256), 0, st, m->h, H, pend));
        pend = none;
        return EV_OK;
    };
    const bool lockstep = ovr && !in->override_first_only;
    for (int l = 0; l < cfg.n_layers; ++l) {
        LayerW& w = m->layers[l];
        const bool tap = (out->tap_layer == l);
        if (lockstep && l > 0) { pend = none; EV_TRY(copy_f32(st, ovr + (size_t)l * M * H, m->h, (long)M * H)); }
        // --- attention block ---
        {
            ProfScope ps(m, st, PC_NORM_QUANT);
            ROW_DISPATCH_S(rp_h, pend.p ? pend.splits : 1, rmsnorm_quant_kernel, dim3(M * rp_h.cl), dim3(NORM_THREADS), 0, st, m->h, H, pend, w.g1, cfg.rms_eps, quant_out(m, m->xq, 4 * l + 0), pfp.take(false));
            pend = none;
        }
        if (tap && out->dev_tap_xq) CUDA_TRY(cudaMemcpyAsync(out->dev_tap_xq, m->xq.codes, (size_t)M * H, cudaMemcpyDeviceToDevice, st));
        if (tap && out->dev_tap_sx) EV_TRY(copy_f32(st, m->xq.scale, out->dev_tap_sx, M));
        RopeArgs ra;
        EV_TRY(run_linear(m, st, w.qkv, m->xq, M, EPI_RAW, &ra.lin, nullptr, nullptr, PC_GEMM_QKV, &pfp));
        ra.qkv_out = m->qkv; ra.ld = m->qkv_dim; ra.Hq = cfg.n_q_heads; ra.Hkv = cfg.n_kv_heads; ra.D = D; ra.T = T;
        ra.pos = m->pos; ra.cs = m->rope_cs; ra.seq_slots = in->dev_seq_slots; ra.Lsnap = m->Lsnap; ra.nn_eff = m->nn_eff;
        ra.page_table = c->page_table; ra.max_pages = c->max_pages; ra.page_size = cfg.page_size;
        ra.pool = c->pool + (size_t)l * c->layer_stride;
        ra.kv_f16 = c->kv_f16;
        ra.pool8 = c->kv_fp8 ? reinterpret_cast<uint8_t*>(c->pool) + (size_t)l * c->layer_stride : nullptr;
        ra.k_scale = c->kv_fp8 ? m->kv_scales[2 * l] : 1.f; ra.v_scale = c->kv_fp8 ? m->kv_scales[2 * l + 1] : 1.f;
        ra.kv_amax = m->recording ? m->kv_amax + 2 * l : nullptr;
        ra.pf = pfp.take(false);
        {
            ProfScope ps(m, st, PC_ROPE_KV);
            if (ra.lin.splits <= 1) EV_TRY(launch_k(rope_kvwrite_kernel<1>, dim3(M, rope_gy), dim3(ROPE_THREADS), 0, st, ra));
            else if (ra.lin.splits <= 3) EV_TRY(launch_k(rope_kvwrite_kernel<3>, dim3(M, rope_gy), dim3(ROPE_THREADS), 0, st, ra));
            else EV_TRY(launch_k(rope_kvwrite_kernel<8>, dim3(M, rope_gy), dim3(ROPE_THREADS), 0, st, ra));
        }
        if (tap && out->dev_tap_qkv) EV_TRY(copy_f32(st, m->qkv, out->dev_tap_qkv, (long)M * m->qkv_dim));
        AttnArgs aa;
        aa.q = m->qkv; aa.q_ld = m->qkv_dim; aa.T = T; aa.G = cfg.n_q_heads / cfg.n_kv_heads; aa.Hq = cfg.n_q_heads;
        aa.Hkv = cfg.n_kv_heads; aa.pool = ra.pool; aa.page_table = c->page_table; aa.max_pages = c->max_pages;
        aa.page_size = cfg.page_size; aa.seq_slots = in->dev_seq_slots; aa.Lsnap = m->Lsnap; aa.nn_eff = m->nn_eff; aa.order = m->attn_order;
        aa.anc_bulk = m->anc_bulk; aa.erow = m->erow; aa.kend_seq = m->kend_seq;
        aa.chunk = split_len; aa.n_chunks = n_splits; aa.scale = 1.0f / sqrtf((float)D);
        aa.o_part = m->o_part; aa.ml_part = m->ml_part;
        // chunks per CTA (tcgen05 kernel): about four CTAs per SM-slot over the launch; a scheduling choice only
        const long units = (long)B * cfg.n_kv_heads * row_groups;
        aa.cpg = (c->kv_f16 || c->kv_fp8) ? (int)std::min<long>(n_splits, std::max<long>(1, units * n_splits / (4L * m->num_sms))) : 1;
        dim3 agrid((n_splits + aa.cpg - 1) / aa.cpg, cfg.n_kv_heads * row_groups, B);
        {
            ProfScope ps(m, st, PC_ATTN);
            if (c->kv_f16 || c->kv_fp8) {
                TcAttnArgs ta;
                ta.a = aa;
                ta.row0 = (int)((long)l * c->n_pages * 2 * cfg.n_kv_heads * TCA_PAGE);
                ta.pool8 = reinterpret_cast<const uint8_t*>(c->pool);
                ta.k_scale = c->kv_fp8 ? m->kv_scales[2 * l] : 1.f; ta.v_scale = c->kv_fp8 ? m->kv_scales[2 * l + 1] : 1.f;
                ta.pf = pfp.take(false);
                const dim3 tgrid(agrid.y, agrid.x, agrid.z);   // the tcgen05 kernel takes (kv head x row group, chunk column, sequence)
                if (c->kv_fp8) EV_TRY((launch_attn_tc<128, true>(st, c->tmKV, ta, tgrid)));
                else if (D == 128 && (long)aa.cpg * aa.chunk <= 8 * TCA_BN) EV_TRY((launch_attn_tc<128, false, true>(st, c->tmKV, ta, tgrid)));   // short key ranges: small rings, more L1
                else if (D == 128) EV_TRY((launch_attn_tc<128, false>(st, c->tmKV, ta, tgrid))); else EV_TRY((launch_attn_tc<64, false>(st, c->tmKV, ta, tgrid)));
            } else {
                if (D == 128) EV_TRY(launch_attn<128>(st, aa, agrid)); else EV_TRY(launch_attn<64>(st, aa, agrid));
            }
        }
        MergeArgs ma;
        ma.T = T; ma.Hq = cfg.n_q_heads; ma.Hkv = cfg.n_kv_heads; ma.D = D; ma.n_chunks = n_splits; ma.chunk = split_len;
        ma.Lsnap = m->Lsnap; ma.nn_eff = m->nn_eff; ma.seq_slots = in->dev_seq_slots; ma.erow = m->erow; ma.kend_row = m->kend_row;
        ma.anc = m->anc; ma.anc_bulk = m->anc_bulk; ma.o_part = m->o_part; ma.ml_part = m->ml_part;
        ma.qkv = m->qkv; ma.q_ld = m->qkv_dim; ma.pool = ra.pool; ma.page_table = c->page_table; ma.max_pages = c->max_pages;
        ma.page_size = cfg.page_size; ma.kv_f16 = c->kv_f16 ? 1 : 0; ma.scale = aa.scale;
        ma.pool8 = ra.pool8; ma.k_scale = ra.k_scale; ma.v_scale = ra.v_scale;
        ma.attn = (tap && out->dev_tap_attn) ? out->dev_tap_attn : nullptr;
        ma.q = quant_out(m, m->aq, 4 * l + 1);
        ma.pf = pfp.take(false);
        {
            ProfScope ps(m, st, PC_ATTN_MERGE);
            const int Gq = cfg.n_q_heads / cfg.n_kv_heads;
            // many rows: one warp per kv head (from 256 rows on: config[3], 256 rows, 789 us per step in clusters of 2 vs 720 this way)
            if ((rp_q.cl == 1 || M >= 256) && D == 128 && cfg.n_kv_heads <= 8 && (Gq == 4 || Gq == 1)) {
                if (Gq == 4) EV_TRY(launch_k(attn_merge_rowkv_kernel<4>, dim3(M), dim3(32 * cfg.n_kv_heads), 0, st, ma));
                else EV_TRY(launch_k(attn_merge_rowkv_kernel<1>, dim3(M), dim3(32 * cfg.n_kv_heads), 0, st, ma));
            } else {
                ROW_DISPATCH(rp_q, attn_merge_quant_kernel, dim3(M * rp_q.cl), dim3(MERGE_THREADS), 0, st, ma);
            }
        }
        if (tap && out->dev_tap_aq) CUDA_TRY(cudaMemcpyAsync(out->dev_tap_aq, m->aq.codes, (size_t)M * m->q_dim, cudaMemcpyDeviceToDevice, st));
        if (tap && out->dev_tap_sa) EV_TRY(copy_f32(st, m->aq.scale, out->dev_tap_sa, M));
        EV_TRY(run_linear(m, st, w.o, m->aq, M, EPI_RAW, &pend, nullptr, nullptr, PC_GEMM_O, &pfp, w.g2, H * 2));
        if (tap && out->dev_tap_hmid) { EV_TRY(materialize()); EV_TRY(copy_f32(st, m->h, out->dev_tap_hmid, (long)M * H)); }
        // --- MLP block ---
        {
            ProfScope ps(m, st, PC_NORM_QUANT);
            ROW_DISPATCH_S(rp_h, pend.p ? pend.splits : 1, rmsnorm_quant_kernel, dim3(M * rp_h.cl), dim3(NORM_THREADS), 0, st, m->h, H, pend, w.g2, cfg.rms_eps, quant_out(m, m->xq, 4 * l + 2), pfp.take(false));
            pend = none;
        }
        LinOut gul;
        EV_TRY(run_linear(m, st, w.gu, m->xq, M, EPI_RAW, &gul, nullptr, nullptr, PC_GEMM_GATEUP, &pfp));
        {
            ProfScope ps(m, st, PC_SWIGLU);
            EV_TRY(launch_swiglu(m, st, swi_smem, rp_f, M, gul, F, (tap ? out->dev_tap_gu : nullptr), quant_out(m, m->tq, 4 * l + 3), pfp.take(false)));
        }
        if (tap && out->dev_tap_tq) CUDA_TRY(cudaMemcpyAsync(out->dev_tap_tq, m->tq.codes, (size_t)M * F, cudaMemcpyDeviceToDevice, st));
        if (tap && out->dev_tap_st) EV_TRY(copy_f32(st, m->tq.scale, out->dev_tap_st, M));
        EV_TRY(run_linear(m, st, w.down, m->tq, M, EPI_RAW, &pend, nullptr, nullptr, PC_GEMM_DOWN, &pfp,
                          (l + 1 < cfg.n_layers) ? m->layers[l + 1].g1 : m->gf, H * 2));
        if (out->dev_hidden) { EV_TRY(materialize()); EV_TRY(copy_f32(st, m->h, out->dev_hidden + (size_t)(l + 1) * M * H, (long)M * H)); }
    }
    if (out->dev_final_hidden) {   // the "feature" an EAGLE drafter consumes: the residual stream after the last layer
        EV_TRY(materialize());
        EV_TRY(copy_f32(st, m->h, out->dev_final_hidden, (long)M * H));
    }
    if (need_lm) {
        if (lockstep) { pend = none; EV_TRY(copy_f32(st, ovr + (size_t)cfg.n_layers * M * H, m->h, (long)M * H)); }
        {
            ProfScope ps(m, st, PC_NORM_QUANT);
            ROW_DISPATCH_S(rp_h, pend.p ? pend.splits : 1, rmsnorm_quant_kernel, dim3(M * rp_h.cl), dim3(NORM_THREADS), 0, st, m->h, H, pend, m->gf, cfg.rms_eps, quant_out(m, m->xq, 4 * cfg.n_layers), pfp.take(false));
            pend = none;
        }
        float* lg = out->dev_logits ? out->dev_logits : (out->dev_topk ? m->logits_ws : nullptr);
        EV_TRY(run_linear(m, st, m->lm, m->xq, M, EPI_ARGMAX, nullptr, lg, m->argmax_keys, PC_GEMM_LM, &pfp));
        if (out->dev_topk) {
            TopkArgs ta;
            ta.logits = lg; ta.V = cfg.vocab; ta.K = out->topk; ta.T = T; ta.nn_eff = m->nn_eff; ta.out = out->dev_topk;
            EV_TRY(launch_k(topk_kernel, dim3(M), dim3(256), 0, st, ta));
        }
    }
    m->n_traced = pfp.n_traced;
    AcceptArgs ac;
    ac.B = B; ac.T = T; ac.commit = in->commit; ac.force_all = in->force_accept_all;
    ac.tokens = in->dev_tokens; ac.parents = in->dev_parents; ac.nn_eff = m->nn_eff; ac.status = out->dev_status;
    ac.Lsnap = m->Lsnap; ac.seq_slots = in->dev_seq_slots; ac.argmax_keys = m->argmax_keys; ac.argmax_out = out->dev_argmax;
    ac.accept_len = out->dev_accept_len; ac.accept_nodes = out->dev_accept_nodes; ac.out_tokens = out->dev_out_tokens;
    ac.new_ctx_len = out->dev_new_ctx_len; ac.ctx_len = c->ctx_len;
    EV_TRY(launch_k(accept_walk_kernel, dim3((B + 63) / 64), dim3(64), 0, st, ac));
    if (in->commit && !in->force_accept_all) {
        CompactArgs ca;
        ca.eb = c->eb; ca.T = T; ca.Hkv = cfg.n_kv_heads; ca.D = D; ca.page_size = cfg.page_size; ca.max_pages = c->max_pages;
        ca.layer_stride = c->layer_stride; ca.pool = c->pool; ca.page_table = c->page_table; ca.seq_slots = in->dev_seq_slots;
        ca.Lsnap = m->Lsnap; ca.accept_len = out->dev_accept_len; ca.accept_nodes = out->dev_accept_nodes;
        EV_TRY(launch_k(kv_compact_kernel, dim3(dim3(B, cfg.n_layers)), dim3(EW_THREADS), 0, st, ca));
    }
    return EV_OK;
}

// captured steps bake kernel arguments (gain pointers, scales passed by value): any change of model state drops them
void drop_graphs(ev_model* m) {
    if (m->graphs.empty()) return;
    cudaDeviceSynchronize();
    for (auto& g : m->graphs) cudaGraphExecDestroy(g.exec);
    m->graphs.clear();
}

int check_ready(ev_model* m, bool need_lm) {
    if (!m->have_embed) return fail(EV_ESTATE, "embedding not set");
    const unsigned need = (1u << EV_W_Q) | (1u << EV_W_K) | (1u << EV_W_V) | (1u << EV_W_O) | (1u << EV_W_GATE) |
                          (1u << EV_W_UP) | (1u << EV_W_DOWN);
    for (size_t l = 0; l < m->layers.size(); ++l)
        if ((m->layers[l].have & need) != need) return fail(EV_ESTATE, "layer " + std::to_string(l) + ": weights missing");
    if (need_lm && !m->have_lm) return fail(EV_ESTATE, "lm_head not set");
    if (m->cfg.act_scale_mode == 1 && !m->calibrated && !m->recording)
        return fail(EV_ESTATE, "static activation scales: model not calibrated");
    if (m->cfg.kv_dtype == 1 && !m->kv_calibrated && !m->recording)
        return fail(EV_ESTATE, "FP8 KV cache: K/V scales not calibrated (ev_model_calibrate or ev_model_set_kv_scales)");
    return EV_OK;
}

}  // namespace

// ================================================================================================
// ---- static scratch for callers that may not allocate (ev_op_linear_static, include/eagle_verify.h) ----------------
// The K-piece slabs of gemm_e4m3_kernel (its scratch: raw fp32 accumulators [pieces][M][N] that the consumer sums) in a
// file-scope device array instead of the model's cudaMalloc'ed workspace.  16 MiB of device memory on every GPU that loads
// the library, held until the process exits.  In host code the NAME `ev_static_slabs` is a host-side stand-in, not a device
// address (a kernel given it faults, or on a GPU that can reach host memory silently uses the wrong memory): host code
// asks cudaGetSymbolAddress for the address, once per device with that device current, and passes THAT to the kernel.
constexpr long EV_STATIC_SLAB_FLOATS = 4L << 20;   // 4 Mi floats = 16 MiB
static __device__ __align__(256) float ev_static_slabs[EV_STATIC_SLAB_FLOATS];
namespace {
// device address of ev_static_slabs on the CURRENT device (resolved on first use per device; ev_model_create does it at set-up)
int static_slabs_ptr(float** out) {
    static float* ptrs[64] = {};
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    float*& p = ptrs[dev & 63];
    if (!p) {
        void* q = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&q, ev_static_slabs);
        if (e != cudaSuccess || !q) return fail(EV_ECUDA, std::string("cudaGetSymbolAddress(ev_static_slabs): ") + cudaGetErrorString(e));
        p = static_cast<float*>(q);
    }
    *out = p;
    return EV_OK;
}
}  // namespace

extern "C" {

const char* ev_last_error(void) { return g_err.c_str(); }
long ev_launch_count(int reset) {
    long v = g_launches;
    if (reset) g_launches = 0;
    return v;
}
long ev_capture_count(int reset) {
    long v = g_captures;
    if (reset) g_captures = 0;
    return v;
}
int ev_version(void) { return 2; }

int ev_model_create(const ev_config* cfg, ev_model** out) {
    if (!cfg || !out) return fail(EV_EINVAL, "null argument");
    *out = nullptr;
    if (cfg->n_layers < 1 || cfg->hidden < 16 || cfg->n_q_heads < 1 || cfg->n_kv_heads < 1 || cfg->ffn < 16 || cfg->vocab < 1)
        return fail(EV_EINVAL, "bad model dimensions");
    if (cfg->head_dim != 64 && cfg->head_dim != 128) return fail(EV_EINVAL, "head_dim must be 64 or 128");
    if (cfg->n_q_heads % cfg->n_kv_heads) return fail(EV_EINVAL, "n_q_heads must be a multiple of n_kv_heads");
    if (cfg->hidden % 16 || cfg->ffn % 16) return fail(EV_EINVAL, "hidden and ffn must be multiples of 16 (TMA row pitch)");
    if (cfg->hidden > 4096 || cfg->ffn > 16384 || cfg->n_q_heads * cfg->head_dim > 4096)
        return fail(EV_EINVAL, "hidden <= 4096, ffn <= 16384, n_q_heads*head_dim <= 4096 (register-resident rows)");
    if (cfg->page_size < 1 || cfg->page_size > 256) return fail(EV_EINVAL, "page_size out of range");
    if (cfg->max_tree_nodes < 1 || cfg->max_tree_nodes > EV_MAX_TREE_NODES) return fail(EV_EINVAL, "max_tree_nodes must be 1..64");
    if (cfg->max_batch < 1 || cfg->max_ctx < 1) return fail(EV_EINVAL, "max_batch / max_ctx must be positive");
    if (cfg->act_scale_mode != 0 && cfg->act_scale_mode != 1) return fail(EV_EINVAL, "act_scale_mode must be 0 or 1");
    if (cfg->weight_scale_mode != 0 && cfg->weight_scale_mode != 1) return fail(EV_EINVAL, "weight_scale_mode must be 0 or 1");
    if (cfg->attn_chunk < 0 || cfg->attn_chunk % 64) return fail(EV_EINVAL, "attn_chunk must be 0 (default) or a multiple of 64");
    if (cfg->kv_dtype != 0 && cfg->kv_dtype != 1) return fail(EV_EINVAL, "kv_dtype must be 0 (bf16) or 1 (E4M3)");
    if (cfg->kv_dtype == 1 && (cfg->page_size != 16 || cfg->head_dim != 128)) return fail(EV_EINVAL, "kv_dtype 1 needs page_size 16 and head_dim 128");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(EV_ECUDA, "no CUDA device");
    ev_model* m = new ev_model();
    m->cfg = *cfg;
    m->M_cap = cfg->max_batch * cfg->max_tree_nodes;
    m->M_pad = (int)round_up(m->M_cap, 256);
    m->q_dim = cfg->n_q_heads * cfg->head_dim;
    m->kv_dim = cfg->n_kv_heads * cfg->head_dim;
    m->qkv_dim = m->q_dim + 2 * m->kv_dim;
    m->max_pos = cfg->max_ctx;
    m->n_sites = 4 * cfg->n_layers + 1;
    m->layers.resize(cfg->n_layers);
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&m->num_sms, cudaDevAttrMultiProcessorCount, dev);
    { float* sp = nullptr; if (static_slabs_ptr(&sp) != EV_OK) { delete m; return EV_ECUDA; } }   // set-up of ev_op_linear_static's scratch address on this device
#ifdef EV_BRINGUP   // bring-up builds only (-DEV_BRINGUP): the shipped library reads no environment variable
    if (getenv("EV_L2PF_MAX_M")) m->l2pf_max_m = atoi(getenv("EV_L2PF_MAX_M"));      // 0 = off
    if (getenv("EV_L2PF_MASK")) m->l2pf_mask = (unsigned)strtoul(getenv("EV_L2PF_MASK"), nullptr, 0);
    if (getenv("EV_L2PF_CAP_MB")) m->l2pf_cap = (long)atoi(getenv("EV_L2PF_CAP_MB")) << 20;
    if (getenv("EV_L2PF_MAXQ_MB")) m->l2pf_maxq = (long)atoi(getenv("EV_L2PF_MAXQ_MB")) << 20;
    m->row_cluster = getenv("EV_ROW_CLUSTER") ? atoi(getenv("EV_ROW_CLUSTER")) : 0;
    m->use_graph = !(getenv("EV_GRAPH") && atoi(getenv("EV_GRAPH")) == 0);          // on by default
    g_use_pdl = !(getenv("EV_PDL") && atoi(getenv("EV_PDL")) == 0);                // on by default
#endif
    const long H = cfg->hidden, F = cfg->ffn, V = cfg->vocab;
    int rc = EV_OK;
    auto A = [&](int r) { if (rc == EV_OK) rc = r; };
    for (auto& L : m->layers) {
        A(alloc_qmat(m, &L.qkv, m->qkv_dim, H));
        A(alloc_qmat(m, &L.o, H, m->q_dim));
        A(alloc_qmat(m, &L.gu, 2 * F, H));
        A(alloc_qmat(m, &L.down, H, F));
    }
    A(alloc_qmat(m, &m->lm, V, H));
    A(dev_alloc(m, &m->embed, (size_t)V * H));
    A(dev_alloc(m, &m->h, (size_t)m->M_pad * H));
    A(alloc_actbuf(m, &m->xq, H));
    A(alloc_actbuf(m, &m->aq, m->q_dim));
    A(alloc_actbuf(m, &m->tq, F));
    A(dev_alloc(m, &m->qkv, (size_t)m->M_pad * m->qkv_dim));
    A(dev_alloc(m, &m->attn, (size_t)m->M_pad * m->q_dim));
    // default chunk length: short for models built for one or two sequences (every chunk is its own CTA: latency), long
    // for batched serving (fewer partial outputs per row); a function of the config only, hence fixed for the model's life
    m->attn_chunk = cfg->attn_chunk > 0 ? cfg->attn_chunk : (cfg->max_batch <= 2 ? 256 : (cfg->max_batch < 16 ? 2048 : 4096));
    m->n_chunks_max = (cfg->max_ctx + m->attn_chunk - 1) / m->attn_chunk;
    A(dev_alloc(m, &m->o_part, (size_t)m->M_cap * m->n_chunks_max * m->q_dim));
    A(dev_alloc(m, &m->ml_part, (size_t)m->M_cap * m->n_chunks_max * cfg->n_q_heads * 2));
    {
        const long widest = std::max<long>(std::max<long>(2 * F, m->qkv_dim), H);
        m->lin_floats = std::max<long>((long)m->M_pad * widest, 8L * std::min(m->M_pad, 256) * widest);
    }
    A(dev_alloc(m, &m->lin_out, (size_t)m->lin_floats));
    A(dev_alloc(m, &m->Lsnap, (size_t)cfg->max_batch));
    A(dev_alloc(m, &m->nn_eff, (size_t)cfg->max_batch));
    A(dev_alloc(m, &m->attn_order, (size_t)cfg->max_batch));
    A(dev_alloc(m, &m->depth, (size_t)m->M_cap));
    A(dev_alloc(m, &m->pos, (size_t)m->M_cap));
    A(dev_alloc(m, &m->anc, (size_t)m->M_cap));
    A(dev_alloc(m, &m->anc_bulk, (size_t)m->M_cap));
    A(dev_alloc(m, &m->erow, (size_t)m->M_cap));
    A(dev_alloc(m, &m->kend_row, (size_t)m->M_cap));
    A(dev_alloc(m, &m->kend_seq, (size_t)cfg->max_batch));
    A(dev_alloc(m, &m->argmax_keys, (size_t)m->M_cap));
    A(dev_alloc(m, &m->static_scales, (size_t)m->n_sites));
    A(dev_alloc(m, &m->site_amax, (size_t)m->n_sites));
    A(dev_alloc(m, &m->w_amax, (size_t)1));
    A(dev_alloc(m, &m->clip_counts, (size_t)m->n_sites));
    A(dev_alloc(m, &m->kv_amax, (size_t)2 * cfg->n_layers));
    m->kv_scales.assign((size_t)2 * cfg->n_layers, 1.0f);
    cudaMemset(m->clip_counts, 0, (size_t)m->n_sites * 8);
    A(dev_alloc(m, &m->rope_cs, (size_t)m->max_pos * (cfg->head_dim / 2)));
    if (rc == EV_OK) {
        // RoPE table: angle = p * theta^(-2j/d) in fp64, cos/sin rounded to fp32 (DESIGN.md R-rope)
        const int D2 = cfg->head_dim / 2;
        std::vector<float2> tab((size_t)m->max_pos * D2);
        std::vector<double> inv(D2);
        for (int j = 0; j < D2; ++j) inv[j] = std::pow((double)cfg->rope_theta, -(2.0 * j) / (double)cfg->head_dim);
        for (long p = 0; p < m->max_pos; ++p)
            for (int j = 0; j < D2; ++j) {
                const double ang = (double)p * inv[j];
                tab[(size_t)p * D2 + j] = make_float2((float)std::cos(ang), (float)std::sin(ang));
            }
        if (cudaMemcpy(m->rope_cs, tab.data(), tab.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess)
            rc = fail(EV_ECUDA, "rope table upload failed");
    }
    if (rc != EV_OK) {
        std::string keep = g_err;
        ev_model_destroy(m);
        g_err = keep;
        return rc;
    }
    *out = m;
    return EV_OK;
}

static void ev_cache_detach(ev_cache* c) { c->model = nullptr; }
int ev_model_destroy(ev_model* m) {
    if (!m) return EV_OK;
    cudaDeviceSynchronize();
    for (void* p : m->allocs) cudaFree(p);
    for (auto& r : m->prof) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    for (auto& g : m->graphs) cudaGraphExecDestroy(g.exec);
    if (m->cap_stream) cudaStreamDestroy(m->cap_stream);
    for (ev_cache* c : m->caches) ev_cache_detach(c);
    delete m;
    return EV_OK;
}

int ev_model_set_weight(ev_model* m, int kind, int layer, const void* dev_bf16, long rows, long cols, void* stream) {
    if (!m || !dev_bf16) return fail(EV_EINVAL, "null argument");
    cudaStream_t st = (cudaStream_t)stream;
    const ev_config& c = m->cfg;
    const long H = c.hidden, F = c.ffn, V = c.vocab;
    const bool per_layer = (kind >= EV_W_Q && kind <= EV_W_DOWN) || kind == EV_W_NORM1 || kind == EV_W_NORM2;
    if (per_layer && (layer < 0 || layer >= c.n_layers)) return fail(EV_EINVAL, "layer out of range");
    auto shape_is = [&](long r, long k) { return rows == r && cols == k; };
    auto bad_shape = [&]() { return fail(EV_EINVAL, "weight shape does not match the model config"); };
    auto quant = [&](QMat& q, long row_off) -> int {
        const float* t_amax = nullptr;
        if (c.weight_scale_mode == 1) {   // per-tensor: the matrix's absmax first (cols % 8 == 0: rows * cols / 8 uint4s)
            CUDA_TRY(cudaMemsetAsync(m->w_amax, 0, sizeof(float), st));
            const long n8 = rows * cols / 8;
            tensor_absmax_bf16_kernel<<<(unsigned)std::min<long>((n8 + 255) / 256, 4L * m->num_sms), 256, 0, st>>>(
                (const __nv_bfloat16*)dev_bf16, n8, m->w_amax);
            LAUNCH_CHECK();
            t_amax = m->w_amax;
        }
        quantize_weight_rows_kernel<<<(unsigned)rows, EW_THREADS, 0, st>>>((const __nv_bfloat16*)dev_bf16, cols, q.codes, q.total_kb,
                                                                          row_off, q.scale, t_amax);
        LAUNCH_CHECK();
        return EV_OK;
    };
    switch (kind) {
        case EV_W_EMBED:
            if (!shape_is(V, H)) return bad_shape();
            CUDA_TRY(cudaMemcpyAsync(m->embed, dev_bf16, (size_t)V * H * 2, cudaMemcpyDeviceToDevice, st));
            m->have_embed = true;
            return EV_OK;
        case EV_W_Q: if (!shape_is(m->q_dim, H)) return bad_shape(); EV_TRY(quant(m->layers[layer].qkv, 0)); break;
        case EV_W_K: if (!shape_is(m->kv_dim, H)) return bad_shape(); EV_TRY(quant(m->layers[layer].qkv, m->q_dim)); break;
        case EV_W_V: if (!shape_is(m->kv_dim, H)) return bad_shape(); EV_TRY(quant(m->layers[layer].qkv, m->q_dim + m->kv_dim)); break;
        case EV_W_O: if (!shape_is(H, m->q_dim)) return bad_shape(); EV_TRY(quant(m->layers[layer].o, 0)); break;
        case EV_W_GATE: if (!shape_is(F, H)) return bad_shape(); EV_TRY(quant(m->layers[layer].gu, 0)); break;
        case EV_W_UP: if (!shape_is(F, H)) return bad_shape(); EV_TRY(quant(m->layers[layer].gu, F)); break;
        case EV_W_DOWN: if (!shape_is(H, F)) return bad_shape(); EV_TRY(quant(m->layers[layer].down, 0)); break;
        case EV_W_LM_HEAD:
            if (!shape_is(V, H)) return bad_shape();
            EV_TRY(quant(m->lm, 0));
            m->have_lm = true;
            return EV_OK;
        case EV_W_NORM1: case EV_W_NORM2: case EV_W_NORMF: {
            if (!(shape_is(1, H) || shape_is(H, 1))) return bad_shape();
            __nv_bfloat16** dst = kind == EV_W_NORM1 ? &m->layers[layer].g1 : kind == EV_W_NORM2 ? &m->layers[layer].g2 : &m->gf;
            if (!*dst) { EV_TRY(dev_alloc(m, dst, (size_t)H)); drop_graphs(m); }   // a graph captured before held a null gain pointer
            CUDA_TRY(cudaMemcpyAsync(*dst, dev_bf16, (size_t)H * 2, cudaMemcpyDeviceToDevice, st));
            return EV_OK;
        }
        case EV_W_DRAFT_FC: {
            if (!shape_is(H, 2 * H)) return bad_shape();
            if (!m->fc.codes) {
                EV_TRY(alloc_qmat(m, &m->fc, H, 2 * H));
                EV_TRY(alloc_actbuf(m, &m->fq, 2 * H));
                EV_TRY(dev_alloc(m, &m->d_topk, (size_t)m->M_cap * TOPK_MAX));
                EV_TRY(dev_alloc(m, &m->d_fhat, (size_t)m->M_cap * H));
                EV_TRY(dev_alloc(m, &m->d_feats, (size_t)m->M_cap * H));
                EV_TRY(dev_alloc(m, &m->d_scratch, (size_t)2 * m->M_cap + 4 * c.max_batch));
                EV_TRY(dev_alloc(m, &m->d_topo, (size_t)2 * EV_MAX_TREE_NODES));
                EV_TRY(dev_alloc(m, &m->d_lvl_n, (size_t)(EV_MAX_TREE_NODES + 1) * c.max_batch));
                EV_TRY(dev_alloc(m, &m->d_tree_par, (size_t)m->M_cap));
                EV_TRY(dev_alloc(m, &m->d_chain_par, (size_t)m->M_cap));
                drop_graphs(m);
            }
            EV_TRY(quant(m->fc, 0));
            m->have_fc = true;
            return EV_OK;
        }
        default: return fail(EV_EINVAL, "unknown weight kind");
    }
    m->layers[layer].have |= 1u << kind;
    return EV_OK;
}

int ev_model_get_quantized(ev_model* m, int kind, int layer, uint8_t* dev_codes_out, float* dev_scales_out, long rows, long cols,
                           void* stream) {
    if (!m || !dev_codes_out || !dev_scales_out) return fail(EV_EINVAL, "null argument");
    if (kind >= EV_W_Q && kind <= EV_W_DOWN && (layer < 0 || layer >= m->cfg.n_layers)) return fail(EV_EINVAL, "layer out of range");
    const long F = m->cfg.ffn;
    QMat* q = nullptr;
    long off = 0, n = 0;
    switch (kind) {
        case EV_W_Q: q = &m->layers[layer].qkv; off = 0; n = m->q_dim; break;
        case EV_W_K: q = &m->layers[layer].qkv; off = m->q_dim; n = m->kv_dim; break;
        case EV_W_V: q = &m->layers[layer].qkv; off = m->q_dim + m->kv_dim; n = m->kv_dim; break;
        case EV_W_O: q = &m->layers[layer].o; n = q->N; break;
        case EV_W_GATE: q = &m->layers[layer].gu; off = 0; n = F; break;
        case EV_W_UP: q = &m->layers[layer].gu; off = F; n = F; break;
        case EV_W_DOWN: q = &m->layers[layer].down; n = q->N; break;
        case EV_W_LM_HEAD: q = &m->lm; n = q->N; break;
        default: return fail(EV_EINVAL, "kind is not a quantized matrix");
    }
    if (rows != n || cols != q->K) return fail(EV_EINVAL, "rows/cols do not match the matrix");
    cudaStream_t st = (cudaStream_t)stream;
    untile_weight_kernel<<<(unsigned)n, 256, 0, st>>>(q->codes, q->total_kb, off, n, q->K, dev_codes_out);
    LAUNCH_CHECK();
    CUDA_TRY(cudaMemcpyAsync(dev_scales_out, q->scale + off, (size_t)n * 4, cudaMemcpyDeviceToDevice, st));
    return EV_OK;
}

int ev_model_get_static_scales(ev_model* m, float* host_out) {
    if (!m || !host_out) return fail(EV_EINVAL, "null argument");
    if (!m->calibrated) return fail(EV_ESTATE, "not calibrated");
    CUDA_TRY(cudaMemcpy(host_out, m->static_scales, m->n_sites * sizeof(float), cudaMemcpyDeviceToHost));
    return EV_OK;
}
int ev_model_get_clip_counts(ev_model* m, unsigned long long* host_out, int reset) {
    if (!m || !host_out) return fail(EV_EINVAL, "null argument");
    CUDA_TRY(cudaDeviceSynchronize());
    CUDA_TRY(cudaMemcpy(host_out, m->clip_counts, m->n_sites * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
    if (reset) CUDA_TRY(cudaMemset(m->clip_counts, 0, m->n_sites * sizeof(unsigned long long)));
    return EV_OK;
}
int ev_model_set_static_scales(ev_model* m, const float* host_in) {
    if (!m || !host_in) return fail(EV_EINVAL, "null argument");
    CUDA_TRY(cudaMemcpy(m->static_scales, host_in, m->n_sites * sizeof(float), cudaMemcpyHostToDevice));
    m->calibrated = true;
    return EV_OK;
}
int ev_model_get_kv_scales(ev_model* m, float* host_out) {
    if (!m || !host_out) return fail(EV_EINVAL, "null argument");
    if (!m->kv_calibrated) return fail(EV_ESTATE, "not calibrated");
    memcpy(host_out, m->kv_scales.data(), m->kv_scales.size() * sizeof(float));
    return EV_OK;
}
int ev_model_set_kv_scales(ev_model* m, const float* host_in) {
    if (!m || !host_in) return fail(EV_EINVAL, "null argument");
    for (size_t i = 0; i < m->kv_scales.size(); ++i)
        if (!(host_in[i] > 0.f)) return fail(EV_EINVAL, "K/V cache scales must be positive");
    memcpy(m->kv_scales.data(), host_in, m->kv_scales.size() * sizeof(float));
    m->kv_calibrated = true;
    drop_graphs(m);
    return EV_OK;
}

// ---- cache ---------------------------------------------------------------------------------------
static int cache_create(ev_model* m, long n_pages, int max_seqs, bool fp8, ev_cache** out);
int ev_cache_create(ev_model* m, long n_pages, int max_seqs, ev_cache** out) {
    if (!m) return fail(EV_EINVAL, "bad argument");
    return cache_create(m, n_pages, max_seqs, m->cfg.kv_dtype == 1, out);
}
static int cache_create(ev_model* m, long n_pages, int max_seqs, bool fp8, ev_cache** out) {
    if (!m || !out || n_pages < 1 || max_seqs < 1) return fail(EV_EINVAL, "bad argument");
    *out = nullptr;
    ev_cache* c = new ev_cache();
    c->model = m;
    c->kv_fp8 = fp8;
    c->eb = fp8 ? 1 : 2;
    c->n_pages = n_pages;
    c->max_seqs = max_seqs;
    const ev_config& cfg = m->cfg;
    c->max_pages = (cfg.max_ctx + cfg.page_size - 1) / cfg.page_size;
    c->layer_stride = n_pages * 2L * cfg.n_kv_heads * cfg.page_size * cfg.head_dim;
    const size_t pool_elems = (size_t)cfg.n_layers * c->layer_stride;
    bool ok = cudaMalloc((void**)&c->pool, pool_elems * c->eb) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&c->page_table, (size_t)max_seqs * c->max_pages * 4) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&c->ctx_len, (size_t)max_seqs * 4) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&c->capacity, (size_t)max_seqs * 4) == cudaSuccess;
    const size_t pf = (size_t)m->M_cap;
    ok = ok && cudaMalloc((void**)&c->pf_tokens, pf * 4) == cudaSuccess && cudaMalloc((void**)&c->pf_parents, pf * 4) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&c->pf_nn, (size_t)cfg.max_batch * 4) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&c->pf_slots, (size_t)cfg.max_batch * 4) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&c->pf_out, (pf * 2 + (size_t)cfg.max_batch * 3) * 4) == cudaSuccess;
    if (!ok) {
        ev_cache_destroy(c);
        return fail(EV_ENOMEM, "KV pool allocation failed");
    }
    cudaMemset(c->pool, 0, pool_elems * c->eb);
    {
        const long rows = (long)cfg.n_layers * n_pages * 2 * cfg.n_kv_heads * cfg.page_size;
        if (cfg.page_size == TCA_PAGE && rows < (1L << 31)) {
            if (make_tmap_kv(&c->tmKV, c->pool, rows, cfg.head_dim) != EV_OK) {
                std::string keep = g_err;
                ev_cache_destroy(c);
                g_err = keep;
                return EV_ECUDA;
            }
            c->tc_attn = true;
            c->kv_f16 = !fp8;
        }
    }
    if (fp8 && !(c->tc_attn && cfg.head_dim == 128)) {
        ev_cache_destroy(c);
        return fail(EV_EINVAL, "kv_dtype 1 (FP8 KV cache) needs page_size 16 and head_dim 128");
    }
    cudaMemset(c->page_table, 0, (size_t)max_seqs * c->max_pages * 4);
    cudaMemset(c->ctx_len, 0, (size_t)max_seqs * 4);
    cudaMemset(c->capacity, 0, (size_t)max_seqs * 4);
    c->free_pages.resize(n_pages);
    for (long i = 0; i < n_pages; ++i) c->free_pages[i] = (int)(n_pages - 1 - i);  // pop_back yields 0,1,2,...
    c->seq_pages.resize(max_seqs);
    c->seq_used.assign(max_seqs, 0);
    c->len_bound.assign(max_seqs, 0);
    m->caches.push_back(c);
    *out = c;
    return EV_OK;
}

int ev_cache_destroy(ev_cache* c) {
    if (!c) return EV_OK;
    cudaDeviceSynchronize();
    if (c->model) {  // captured steps that reference this cache's buffers die with it
        auto& cs = c->model->caches;
        cs.erase(std::remove(cs.begin(), cs.end(), c), cs.end());
        auto& gs = c->model->graphs;
        for (size_t i = gs.size(); i-- > 0;)
            if (gs[i].key.p[0] == (const void*)c) { cudaGraphExecDestroy(gs[i].exec); gs.erase(gs.begin() + i); }
    }
    cudaFree(c->pool); cudaFree(c->page_table); cudaFree(c->ctx_len); cudaFree(c->capacity);
    cudaFree(c->pf_tokens); cudaFree(c->pf_parents); cudaFree(c->pf_nn); cudaFree(c->pf_slots); cudaFree(c->pf_out);
    delete c;
    return EV_OK;
}

int ev_cache_add_seq(ev_cache* c, int capacity_tokens, const int* host_pages, int* seq_slot_out) {
    if (!c || !seq_slot_out || capacity_tokens < 1) return fail(EV_EINVAL, "bad argument");
    const int P = c->model->cfg.page_size;
    const int need = (capacity_tokens + P - 1) / P;
    if (need > c->max_pages) return fail(EV_ECAPACITY, "capacity exceeds max_ctx");
    int slot = -1;
    for (int i = 0; i < c->max_seqs; ++i)
        if (!c->seq_used[i]) { slot = i; break; }
    if (slot < 0) return fail(EV_ECAPACITY, "no free sequence slot");
    std::vector<int> pages;
    if (host_pages) {
        for (int i = 0; i < need; ++i) {
            const int pg = host_pages[i];
            auto it = std::find(c->free_pages.begin(), c->free_pages.end(), pg);
            if (pg < 0 || pg >= c->n_pages || it == c->free_pages.end()) {
                for (int q : pages) c->free_pages.push_back(q);
                return fail(EV_EINVAL, "requested page is not free");
            }
            c->free_pages.erase(it);
            pages.push_back(pg);
        }
    } else {
        if ((long)c->free_pages.size() < need) return fail(EV_ECAPACITY, "out of KV pages");
        for (int i = 0; i < need; ++i) { pages.push_back(c->free_pages.back()); c->free_pages.pop_back(); }
    }
    std::vector<int32_t> row(c->max_pages, 0);
    for (int i = 0; i < need; ++i) row[i] = pages[i];
    const int32_t cap = need * P, zero = 0;
    CUDA_TRY(cudaMemcpy(c->page_table + (size_t)slot * c->max_pages, row.data(), row.size() * 4, cudaMemcpyHostToDevice));
    CUDA_TRY(cudaMemcpy(c->capacity + slot, &cap, 4, cudaMemcpyHostToDevice));
    CUDA_TRY(cudaMemcpy(c->ctx_len + slot, &zero, 4, cudaMemcpyHostToDevice));
    c->seq_pages[slot] = pages;
    c->seq_used[slot] = 1;
    c->len_bound[slot] = 0;
    *seq_slot_out = slot;
    return EV_OK;
}

int ev_cache_free_seq(ev_cache* c, int slot) {
    if (!c || slot < 0 || slot >= c->max_seqs || !c->seq_used[slot]) return fail(EV_EINVAL, "bad sequence slot");
    for (int pg : c->seq_pages[slot]) c->free_pages.push_back(pg);
    c->seq_pages[slot].clear();
    c->seq_used[slot] = 0;
    const int32_t zero = 0;
    CUDA_TRY(cudaMemcpy(c->capacity + slot, &zero, 4, cudaMemcpyHostToDevice));
    CUDA_TRY(cudaMemcpy(c->ctx_len + slot, &zero, 4, cudaMemcpyHostToDevice));
    return EV_OK;
}

int ev_cache_set_len(ev_cache* c, int slot, int ctx_len, void* stream) {
    if (!c || slot < 0 || slot >= c->max_seqs || !c->seq_used[slot] || ctx_len < 0) return fail(EV_EINVAL, "bad argument");
    if (ctx_len > (int)c->seq_pages[slot].size() * c->model->cfg.page_size) return fail(EV_ECAPACITY, "ctx_len exceeds capacity");
    set_i32_kernel<<<1, 1, 0, (cudaStream_t)stream>>>(c->ctx_len + slot, ctx_len);
    LAUNCH_CHECK();
    c->len_bound[slot] = ctx_len;
    return EV_OK;
}
int ev_cache_set_lens(ev_cache* c, int n, const int* host_slots, const int* host_lens, void* stream) {
    if (!c || !host_slots || !host_lens || n < 1 || n > c->model->cfg.max_batch) return fail(EV_EINVAL, "bad argument");
    for (int i = 0; i < n; ++i) {
        const int s = host_slots[i];
        if (s < 0 || s >= c->max_seqs || !c->seq_used[s] || host_lens[i] < 0) return fail(EV_EINVAL, "bad slot or length");
        if (host_lens[i] > (int)c->seq_pages[s].size() * c->model->cfg.page_size) return fail(EV_ECAPACITY, "ctx_len exceeds capacity");
    }
    SetLensArgs a;
    if (n > SetLensArgs::MAX) return fail(EV_EINVAL, "at most 64 sequences per call");
    a.n = n;
    for (int i = 0; i < n; ++i) { a.slot[i] = host_slots[i]; a.len[i] = host_lens[i]; c->len_bound[host_slots[i]] = host_lens[i]; }
    set_lens_kernel<<<1, 64, 0, (cudaStream_t)stream>>>(c->ctx_len, a);
    LAUNCH_CHECK();
    return EV_OK;
}
int ev_cache_get_len(ev_cache* c, int slot, int* ctx_len, void* stream) {
    if (!c || !ctx_len || slot < 0 || slot >= c->max_seqs || !c->seq_used[slot]) return fail(EV_EINVAL, "bad argument");
    int32_t v = 0;
    CUDA_TRY(cudaMemcpyAsync(&v, c->ctx_len + slot, 4, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CUDA_TRY(cudaStreamSynchronize((cudaStream_t)stream));
    *ctx_len = v;
    c->len_bound[slot] = v;
    return EV_OK;
}

static int dense_copy(ev_cache* c, int slot, int lb, int le, int n_tokens, void* dense, int to_dense, cudaStream_t st) {
    if (!c || !dense || slot < 0 || slot >= c->max_seqs || !c->seq_used[slot]) return fail(EV_EINVAL, "bad argument");
    const ev_config& cfg = c->model->cfg;
    if (lb < 0 || le > cfg.n_layers || lb >= le || n_tokens < 1) return fail(EV_EINVAL, "bad layer / token range");
    if (n_tokens > (int)c->seq_pages[slot].size() * cfg.page_size) return fail(EV_ECAPACITY, "n_tokens exceeds capacity");
    DenseCopyArgs a;
    a.Hkv = cfg.n_kv_heads; a.D = cfg.head_dim; a.page_size = cfg.page_size; a.n_tokens = n_tokens; a.layer_begin = lb;
    a.layer_stride = c->layer_stride; a.pool = c->pool; a.page_row = c->page_table + (size_t)slot * c->max_pages;
    a.dense = (__nv_bfloat16*)dense; a.to_dense = to_dense; a.kv_f16 = c->kv_f16; a.eb = c->eb;
    dense_copy_kernel<<<dim3(n_tokens, le - lb), 128, 0, st>>>(a);
    LAUNCH_CHECK();
    return EV_OK;
}
int ev_cache_export_seq(ev_cache* c, int slot, int lb, int le, int n_tokens, void* dense, void* stream) {
    return dense_copy(c, slot, lb, le, n_tokens, dense, 1, (cudaStream_t)stream);
}
int ev_cache_import_seq(ev_cache* c, int slot, int lb, int le, int n_tokens, const void* dense, int set_len, void* stream) {
    EV_TRY(dense_copy(c, slot, lb, le, n_tokens, const_cast<void*>(dense), 0, (cudaStream_t)stream));
    if (set_len) return ev_cache_set_len(c, slot, n_tokens, stream);
    return EV_OK;
}

// ---- verify ----------------------------------------------------------------------------------------
int ev_verify(ev_model* m, ev_cache* c, const ev_verify_in* in, ev_verify_out* out, void* stream) {
    if (!m || !c || !in || !out) return fail(EV_EINVAL, "null argument");
    if (c->model != m) return fail(EV_EINVAL, "cache belongs to another model");
    if (in->n_seqs < 1 || in->n_nodes_max < 1) return fail(EV_EINVAL, "n_seqs and n_nodes_max must be positive");
    if (in->n_seqs > m->cfg.max_batch || in->n_nodes_max > m->cfg.max_tree_nodes)
        return fail(EV_ECAPACITY, "batch or tree size exceeds the model's max_batch / max_tree_nodes");
    if (!in->dev_seq_slots || !in->dev_tokens || !in->dev_parents) return fail(EV_EINVAL, "null input array");
    if (!out->dev_accept_len || !out->dev_accept_nodes || !out->dev_out_tokens || !out->dev_new_ctx_len || !out->dev_status)
        return fail(EV_EINVAL, "null required output array");
    const bool need_lm = !in->force_accept_all || m->recording;
    EV_TRY(check_ready(m, need_lm));
    if (in->dev_features && !m->have_fc) return fail(EV_ESTATE, "dev_features given but EV_W_DRAFT_FC is not set (not a draft model)");
    if (out->dev_topk) {
        if (out->topk < 1 || out->topk > TOPK_MAX) return fail(EV_EINVAL, "topk must be 1..8");
        if (!out->dev_logits && !m->logits_ws) {   // setup-time allocation (first use), not on the steady path
            EV_TRY(dev_alloc(m, &m->logits_ws, (size_t)m->M_cap * m->cfg.vocab));
        }
    }
    cudaStream_t st = (cudaStream_t)stream;
    const AttnPlan plan = plan_attention(m, c, in);
    // Fast path: the whole step (~330 launches, PDL edges included) is captured once per distinct argument set
    // and replayed as one CUDA graph.  Debug taps, lock-step overrides, profiling and calibration run eagerly.
    bool graph_ok = m->use_graph && !m->profile && !m->recording && !in->dev_hidden_override && !out->dev_hidden &&
                    (out->tap_layer < 0 || out->tap_layer >= m->cfg.n_layers);
    if (graph_ok) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) graph_ok = false;  // caller captures
    }
    if (!graph_ok) return run_forward(m, c, in, out, st, need_lm, plan);
    GraphKey key;
    memset(&key, 0, sizeof(key));
    key.B = in->n_seqs; key.T = in->n_nodes_max; key.commit = in->commit; key.force_all = in->force_accept_all;
    key.n_splits = plan.n_splits; key.split_len = plan.split_len; key.need_lm = need_lm;
    const void* ptrs[16] = {c, in->dev_seq_slots, in->dev_tokens, in->dev_parents, in->dev_n_nodes, out->dev_accept_len,
                            out->dev_accept_nodes, out->dev_out_tokens, out->dev_new_ctx_len, out->dev_status, out->dev_argmax,
                            out->dev_logits, in->dev_features, out->dev_final_hidden, out->dev_topk, (const void*)(size_t)out->topk};
    memcpy(key.p, ptrs, sizeof(ptrs));
    GraphEntry* hit = nullptr;
    for (auto& g : m->graphs)
        if (memcmp(&g.key, &key, sizeof(key)) == 0) { hit = &g; break; }
    if (!hit) {
        if (!m->cap_stream) CUDA_TRY(cudaStreamCreateWithFlags(&m->cap_stream, cudaStreamNonBlocking));
        const long before = g_launches;
        ++g_captures;
        CUDA_TRY(cudaStreamBeginCapture(m->cap_stream, cudaStreamCaptureModeRelaxed));
        const int rc = run_forward(m, c, in, out, m->cap_stream, need_lm, plan);
        cudaGraph_t graph = nullptr;
        const cudaError_t e = cudaStreamEndCapture(m->cap_stream, &graph);
        const long n_launch = g_launches - before;
        g_launches = before;
        if (rc != EV_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
        if (e != cudaSuccess || !graph) return fail(EV_ECUDA, std::string("graph capture: ") + cudaGetErrorString(e));
        cudaGraphExec_t exec = nullptr;
        const cudaError_t e2 = cudaGraphInstantiate(&exec, graph, 0);
        cudaGraphDestroy(graph);
        if (e2 != cudaSuccess) return fail(EV_ECUDA, std::string("graph instantiate: ") + cudaGetErrorString(e2));
        if (m->graphs.size() >= MAX_GRAPHS) {  // evict the least recently used
            size_t lru = 0;
            for (size_t i = 1; i < m->graphs.size(); ++i)
                if (m->graphs[i].stamp < m->graphs[lru].stamp) lru = i;
            cudaGraphExecDestroy(m->graphs[lru].exec);
            m->graphs.erase(m->graphs.begin() + lru);
        }
        GraphEntry ge;
        ge.key = key; ge.exec = exec; ge.launches = n_launch; ge.stamp = 0;
        m->graphs.push_back(ge);
        hit = &m->graphs.back();
    }
    hit->stamp = ++m->graph_clock;
    CUDA_TRY(cudaGraphLaunch(hit->exec, st));
    g_launches += hit->launches;
    return EV_OK;
}

int ev_cache_prefill(ev_model* m, ev_cache* c, int n_seqs, const int* host_seq_slots, const int32_t* host_token_ids,
                     const int* host_lens, void* stream) {
    if (!m || !c || !host_seq_slots || !host_token_ids || !host_lens || n_seqs < 1) return fail(EV_EINVAL, "bad argument");
    cudaStream_t st = (cudaStream_t)stream;
    const int T = m->cfg.max_tree_nodes, Bmax = m->cfg.max_batch;
    std::vector<long> off(n_seqs + 1, 0);
    for (int i = 0; i < n_seqs; ++i) {
        if (host_lens[i] < 0) return fail(EV_EINVAL, "negative length");
        off[i + 1] = off[i] + host_lens[i];
    }
    std::vector<int> done(n_seqs, 0);
    std::vector<int32_t> tok((size_t)Bmax * T), par((size_t)Bmax * T), nn(Bmax), slots(Bmax);
    ev_verify_out o;
    memset(&o, 0, sizeof(o));
    o.tap_layer = -1;
    o.dev_accept_len = c->pf_out;
    o.dev_new_ctx_len = c->pf_out + Bmax;
    o.dev_status = c->pf_out + 2 * Bmax;
    o.dev_accept_nodes = c->pf_out + 3 * Bmax;
    o.dev_out_tokens = o.dev_accept_nodes + (size_t)m->M_cap;
    while (true) {
        int B = 0;
        for (int i = 0; i < n_seqs && B < Bmax; ++i) {
            const int rem = host_lens[i] - done[i];
            if (rem <= 0) continue;
            const int n = std::min(rem, T);
            for (int j = 0; j < T; ++j) {
                tok[(size_t)B * T + j] = j < n ? host_token_ids[off[i] + done[i] + j] : 0;
                par[(size_t)B * T + j] = j - 1;
            }
            nn[B] = n;
            slots[B] = host_seq_slots[i];
            done[i] += n;
            ++B;
        }
        if (B == 0) break;
        CUDA_TRY(cudaMemcpyAsync(c->pf_tokens, tok.data(), (size_t)B * T * 4, cudaMemcpyHostToDevice, st));
        CUDA_TRY(cudaMemcpyAsync(c->pf_parents, par.data(), (size_t)B * T * 4, cudaMemcpyHostToDevice, st));
        CUDA_TRY(cudaMemcpyAsync(c->pf_nn, nn.data(), (size_t)B * 4, cudaMemcpyHostToDevice, st));
        CUDA_TRY(cudaMemcpyAsync(c->pf_slots, slots.data(), (size_t)B * 4, cudaMemcpyHostToDevice, st));
        ev_verify_in in;
        memset(&in, 0, sizeof(in));
        in.n_seqs = B; in.n_nodes_max = T; in.dev_seq_slots = c->pf_slots; in.dev_tokens = c->pf_tokens;
        in.dev_parents = c->pf_parents; in.dev_n_nodes = c->pf_nn; in.commit = 1; in.force_accept_all = 1;
        EV_TRY(ev_verify(m, c, &in, &o, stream));
        CUDA_TRY(cudaStreamSynchronize(st));  // host staging buffers are reused by the next pass
        std::vector<int32_t> status(B);
        CUDA_TRY(cudaMemcpy(status.data(), o.dev_status, (size_t)B * 4, cudaMemcpyDeviceToHost));
        for (int i = 0; i < B; ++i)
            if (status[i]) return fail(status[i] & EV_SEQ_OVER_CAPACITY ? EV_ECAPACITY : EV_EINVAL,
                                       "prefill: sequence rejected, status " + std::to_string(status[i]));
    }
    return EV_OK;
}

int ev_model_calibrate(ev_model* m, const float* dev_hidden, int n_tok, float* dev_layer_inputs, void* stream) {
    if (!m || !dev_hidden || n_tok < 1) return fail(EV_EINVAL, "bad argument");
    if (n_tok > m->cfg.max_ctx) return fail(EV_ECAPACITY, "n_tok exceeds max_ctx");
    cudaStream_t st = (cudaStream_t)stream;
    const ev_config& cfg = m->cfg;
    const int T = cfg.max_tree_nodes, H = cfg.hidden;
    ev_cache* c = nullptr;
    EV_TRY(cache_create(m, (n_tok + cfg.page_size - 1) / cfg.page_size + 1, 1, false, &c));   // the calibration pass itself runs on a bf16 cache
    int slot = -1, rc = ev_cache_add_seq(c, n_tok, nullptr, &slot);
    float* taps = nullptr;
    if (rc == EV_OK && dev_layer_inputs && cudaMalloc((void**)&taps, (size_t)(cfg.n_layers + 1) * T * H * 4) != cudaSuccess)
        rc = fail(EV_ENOMEM, "calibration tap buffer");
    if (rc == EV_OK && cudaMemsetAsync(m->site_amax, 0, m->n_sites * 4, st) != cudaSuccess) rc = fail(EV_ECUDA, "memset");
    if (rc == EV_OK && cudaMemsetAsync(m->kv_amax, 0, (size_t)2 * cfg.n_layers * 4, st) != cudaSuccess) rc = fail(EV_ECUDA, "memset");
    m->recording = true;
    std::vector<int32_t> tok(T, 0), par(T);
    for (int j = 0; j < T; ++j) par[j] = j - 1;
    ev_verify_out o;
    memset(&o, 0, sizeof(o));
    o.tap_layer = -1;
    o.dev_accept_len = c->pf_out; o.dev_new_ctx_len = c->pf_out + 1; o.dev_status = c->pf_out + 2;
    o.dev_accept_nodes = c->pf_out + 3; o.dev_out_tokens = c->pf_out + 3 + T;
    o.dev_hidden = taps;
    for (int p0 = 0; rc == EV_OK && p0 < n_tok; p0 += T) {
        const int n = std::min(T, n_tok - p0);
        const int32_t nn = n, sl = slot;
        auto cp = [&](void* d, const void* s, size_t b) { if (rc == EV_OK && cudaMemcpyAsync(d, s, b, cudaMemcpyHostToDevice, st) != cudaSuccess) rc = fail(EV_ECUDA, "H2D copy"); };
        cp(c->pf_tokens, tok.data(), (size_t)T * 4);
        cp(c->pf_parents, par.data(), (size_t)T * 4);
        cp(c->pf_nn, &nn, 4);
        cp(c->pf_slots, &sl, 4);
        ev_verify_in in;
        memset(&in, 0, sizeof(in));
        in.n_seqs = 1; in.n_nodes_max = n; in.dev_seq_slots = c->pf_slots; in.dev_tokens = c->pf_tokens;
        in.dev_parents = c->pf_parents; in.dev_n_nodes = c->pf_nn; in.commit = 1; in.force_accept_all = 1;
        in.dev_hidden_override = dev_hidden + (size_t)p0 * H; in.override_first_only = 1;
        if (rc == EV_OK) rc = ev_verify(m, c, &in, &o, stream);
        if (rc == EV_OK && taps)
            for (int l = 0; l <= cfg.n_layers && rc == EV_OK; ++l)
                if (cudaMemcpyAsync(dev_layer_inputs + ((size_t)l * n_tok + p0) * H, taps + (size_t)l * n * H, (size_t)n * H * 4,
                                    cudaMemcpyDeviceToDevice, st) != cudaSuccess) rc = fail(EV_ECUDA, "tap copy");
        if (rc == EV_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = fail(EV_ECUDA, "calibration pass failed");
    }
    m->recording = false;
    if (rc == EV_OK) {
        std::vector<float> amax(m->n_sites), sc(m->n_sites);
        if (cudaMemcpy(amax.data(), m->site_amax, m->n_sites * 4, cudaMemcpyDeviceToHost) != cudaSuccess) rc = fail(EV_ECUDA, "D2H copy");
        for (int i = 0; i < m->n_sites; ++i) sc[i] = amax[i] > 0.f ? amax[i] / 448.0f : 1.0f;
        if (rc == EV_OK && cudaMemcpy(m->static_scales, sc.data(), m->n_sites * 4, cudaMemcpyHostToDevice) != cudaSuccess) rc = fail(EV_ECUDA, "H2D copy");
        if (rc == EV_OK) m->calibrated = true;
        std::vector<float> kva((size_t)2 * cfg.n_layers);
        if (rc == EV_OK && cudaMemcpy(kva.data(), m->kv_amax, kva.size() * 4, cudaMemcpyDeviceToHost) != cudaSuccess) rc = fail(EV_ECUDA, "D2H copy");
        if (rc == EV_OK) {   // FP8 KV cache scales: per-tensor absmax of K (post-RoPE) and V over the calibration tokens / 448
            for (size_t i = 0; i < kva.size(); ++i) m->kv_scales[i] = kva[i] > 0.f ? kva[i] / 448.0f : 1.0f;
            m->kv_calibrated = true;
        }
        drop_graphs(m);
    }
    std::string keep = g_err;
    if (taps) cudaFree(taps);
    ev_cache_destroy(c);
    g_err = keep;
    return rc;
}

// ---- draft side ----------------------------------------------------------------------------------------
int ev_model_share_head(ev_model* d, ev_model* t) {
    if (!d || !t || d == t) return fail(EV_EINVAL, "bad argument");
    if (d->cfg.hidden != t->cfg.hidden || d->cfg.vocab != t->cfg.vocab) return fail(EV_EINVAL, "drafter and target differ in hidden / vocab");
    if (!t->have_embed || !t->have_lm) return fail(EV_ESTATE, "target embedding / LM head not set");
    d->embed = t->embed; d->lm = t->lm; d->gf = t->gf;     // borrowed: the drafter's own (unused) buffers stay in its alloc list
    d->have_embed = d->have_lm = d->shared_head = true;
    drop_graphs(d);
    return EV_OK;
}

static int draft_pass(ev_model* m, ev_cache* c, int B, int T, const int32_t* slots, const int32_t* tokens, const int32_t* parents,
                      const int32_t* n_nodes, const float* feats, bool commit_all, int topk, cudaStream_t st) {
    ev_verify_in in;
    memset(&in, 0, sizeof(in));
    in.n_seqs = B; in.n_nodes_max = T; in.dev_seq_slots = slots; in.dev_tokens = tokens; in.dev_parents = parents;
    in.dev_n_nodes = n_nodes; in.commit = commit_all ? 1 : 0; in.force_accept_all = commit_all ? 1 : 0; in.dev_features = feats;
    ev_verify_out o;
    memset(&o, 0, sizeof(o));
    o.tap_layer = -1;
    const int Bm = m->cfg.max_batch;
    o.dev_accept_len = m->d_scratch; o.dev_new_ctx_len = m->d_scratch + Bm; o.dev_status = m->d_scratch + 2 * Bm;
    o.dev_accept_nodes = m->d_scratch + 4 * Bm; o.dev_out_tokens = o.dev_accept_nodes + m->M_cap;
    if (!commit_all) { o.dev_final_hidden = m->d_fhat; o.dev_topk = m->d_topk; o.topk = topk; }
    return ev_verify(m, c, &in, &o, (void*)st);
}

int ev_draft_tree(ev_model* m, ev_cache* c, const ev_draft_args* a, void* stream) {
    if (!m || !c || !a || !a->dev_seq_slots || !a->host_parents || !a->dev_root_tokens || !a->dev_root_feats || !a->dev_tokens || !a->dev_parents)
        return fail(EV_EINVAL, "null argument");
    if (!m->have_fc) return fail(EV_ESTATE, "not a draft model (EV_W_DRAFT_FC not set)");
    const int B = a->n_seqs, T = a->n_nodes, H = m->cfg.hidden;
    if (B < 1 || B > m->cfg.max_batch || T < 1 || T > m->cfg.max_tree_nodes) return fail(EV_ECAPACITY, "batch or tree size exceeds the model's maxima");
    cudaStream_t st = (cudaStream_t)stream;
    // topology: depths must be non-decreasing in node order (levels are prefixes); child ranks; widest fan-out = top-k
    std::vector<int> depth(T, 0), rank(T, 0), nchild(T, 0);
    if (a->host_parents[0] != -1) return fail(EV_EINVAL, "parents[0] must be -1");
    for (int i = 1; i < T; ++i) {
        const int p = a->host_parents[i];
        if (p < 0 || p >= i) return fail(EV_EINVAL, "parents[i] must be in [0, i)");
        depth[i] = depth[p] + 1;
        if (depth[i] < depth[i - 1]) return fail(EV_EINVAL, "nodes must be ordered by depth");
        rank[i] = nchild[p]++;
    }
    int K = 1;
    for (int i = 0; i < T; ++i) K = std::max(K, nchild[i]);
    if (K > TOPK_MAX) return fail(EV_EINVAL, "a node has more than 8 children");
    const int D = depth[T - 1];
    std::vector<int32_t> topo(2 * T);
    for (int i = 0; i < T; ++i) { topo[i] = a->host_parents[i]; topo[T + i] = rank[i]; }
    if (m->h_topo != topo) {   // new topology: upload it (setup; the steady loop reuses it)
        CUDA_TRY(cudaStreamSynchronize(st));
        m->h_topo = topo;
        CUDA_TRY(cudaMemcpy(m->d_topo, topo.data(), topo.size() * 4, cudaMemcpyHostToDevice));
        std::vector<int32_t> lv((size_t)(D + 1) * m->cfg.max_batch), par((size_t)m->cfg.max_batch * T);
        for (int d = 0; d <= D; ++d) {
            int n = 0;
            while (n < T && depth[n] <= d) ++n;
            for (int b = 0; b < m->cfg.max_batch; ++b) lv[(size_t)d * m->cfg.max_batch + b] = n;
        }
        for (int b = 0; b < m->cfg.max_batch; ++b) memcpy(&par[(size_t)b * T], a->host_parents, (size_t)T * 4);
        CUDA_TRY(cudaMemcpy(m->d_lvl_n, lv.data(), lv.size() * 4, cudaMemcpyHostToDevice));
        CUDA_TRY(cudaMemcpy(m->d_tree_par, par.data(), par.size() * 4, cudaMemcpyHostToDevice));
    }
    // the per-sequence parents arrays ev_verify consumes, root tokens and root features into the tree's row 0 (all on the stream)
    CUDA_TRY(cudaMemcpyAsync(a->dev_parents, m->d_tree_par, (size_t)B * T * 4, cudaMemcpyDeviceToDevice, st));
    CUDA_TRY(cudaMemcpy2DAsync(a->dev_tokens, (size_t)T * 4, a->dev_root_tokens, 4, 4, B, cudaMemcpyDeviceToDevice, st));
    CUDA_TRY(cudaMemcpy2DAsync(m->d_feats, (size_t)T * H * 4, a->dev_root_feats, (size_t)H * 4, (size_t)H * 4, B, cudaMemcpyDeviceToDevice, st));
    for (int d = 0; d <= D; ++d) {
        int n0 = 0;
        while (n0 < T && depth[n0] <= d) ++n0;
        if (d == D && n0 != T) return fail(EV_EINVAL, "topology depth mismatch");
        EV_TRY(draft_pass(m, c, B, T, a->dev_seq_slots, a->dev_tokens, a->dev_parents, m->d_lvl_n + (size_t)d * m->cfg.max_batch, m->d_feats,
                          false, K, st));
        if (d == D) break;
        int n1 = n0;
        while (n1 < T && depth[n1] == d + 1) ++n1;
        ExpandArgs ea;
        ea.T = T; ea.H = H; ea.K = K; ea.n0 = n0; ea.parents = m->d_topo; ea.rank = m->d_topo + T; ea.topk = m->d_topk; ea.f_hat = m->d_fhat;
        ea.tokens = a->dev_tokens; ea.feats = m->d_feats;
        EV_TRY(launch_k(draft_expand_kernel, dim3(n1 - n0, B), dim3(256), 0, st, ea));
    }
    return EV_OK;
}

int ev_draft_extend(ev_model* m, ev_cache* c, int n_seqs, int n_nodes, const int32_t* dev_seq_slots, const int32_t* dev_tokens,
                    const float* dev_feats, const int32_t* dev_n, void* stream) {
    if (!m || !c || !dev_seq_slots || !dev_tokens || !dev_feats || !dev_n) return fail(EV_EINVAL, "null argument");
    if (!m->have_fc) return fail(EV_ESTATE, "not a draft model (EV_W_DRAFT_FC not set)");
    if (n_seqs < 1 || n_seqs > m->cfg.max_batch || n_nodes < 1 || n_nodes > m->cfg.max_tree_nodes) return fail(EV_ECAPACITY, "batch or chain too large");
    cudaStream_t st = (cudaStream_t)stream;
    if (m->chain_T != n_nodes) {   // chain parents (row i: i - 1) at this row stride: uploaded once per stride (setup)
        std::vector<int32_t> par((size_t)m->cfg.max_batch * n_nodes);
        for (int b = 0; b < m->cfg.max_batch; ++b)
            for (int i = 0; i < n_nodes; ++i) par[(size_t)b * n_nodes + i] = i - 1;
        CUDA_TRY(cudaStreamSynchronize(st));
        CUDA_TRY(cudaMemcpy(m->d_chain_par, par.data(), par.size() * 4, cudaMemcpyHostToDevice));
        m->chain_T = n_nodes;
    }
    return draft_pass(m, c, n_seqs, n_nodes, dev_seq_slots, dev_tokens, m->d_chain_par, dev_n, dev_feats, true, 0, st);
}

int ev_gather_accepted(int n_seqs, int n_nodes, int hidden, const int32_t* dev_tokens, const int32_t* dev_accept_len,
                       const int32_t* dev_accept_nodes, const int32_t* dev_out_tokens, const float* dev_feat, float* dev_carry,
                       int32_t* dev_ext_tokens, float* dev_ext_feats, int32_t* dev_ext_n, int32_t* dev_next_root, void* stream) {
    if (n_seqs < 1 || n_nodes < 1 || hidden < 1 || !dev_tokens || !dev_accept_len || !dev_accept_nodes || !dev_out_tokens || !dev_feat ||
        !dev_carry || !dev_ext_tokens || !dev_ext_feats || !dev_ext_n || !dev_next_root)
        return fail(EV_EINVAL, "bad argument");
    cudaStream_t st = (cudaStream_t)stream;
    GatherArgs g;
    g.T = n_nodes; g.H = hidden; g.tokens = dev_tokens; g.accept_len = dev_accept_len; g.accept_nodes = dev_accept_nodes;
    g.out_tokens = dev_out_tokens; g.feat = dev_feat; g.carry = dev_carry; g.ext_tokens = dev_ext_tokens; g.ext_feats = dev_ext_feats;
    g.ext_n = dev_ext_n; g.next_root = dev_next_root;
    gather_accepted_kernel<<<dim3(n_nodes, n_seqs), 256, 0, st>>>(g);
    LAUNCH_CHECK();
    carry_update_kernel<<<n_seqs, 256, 0, st>>>(g);
    LAUNCH_CHECK();
    return EV_OK;
}

// ---- single operators --------------------------------------------------------------------------------
int ev_op_quantize_rows(ev_model* m, const float* dev_x, int M, int K, float static_scale, uint8_t* dev_codes, float* dev_sx,
                        void* stream) {
    if (!m || !dev_x || !dev_codes || !dev_sx || M < 1 || K < 4 || K % 4) return fail(EV_EINVAL, "bad argument");
    cudaStream_t st = (cudaStream_t)stream;
    QuantOut q;
    q.codes = dev_codes; q.sx = dev_sx; q.static_scale = nullptr; q.site_amax = nullptr; q.clip_count = nullptr;
    if (static_scale > 0.f) {
        CUDA_TRY(cudaMemcpyAsync(m->site_amax, &static_scale, 4, cudaMemcpyHostToDevice, st));
        CUDA_TRY(cudaStreamSynchronize(st));
        q.static_scale = m->site_amax;
    }
    quantize_rows_kernel<<<M, EW_THREADS, 0, st>>>(dev_x, K, q);
    LAUNCH_CHECK();
    return EV_OK;
}

int ev_op_linear(ev_model* m, int kind, int layer, const uint8_t* dev_codes_x, const float* dev_sx, int M, float* dev_out,
                 void* stream) {
    if (!m || !dev_codes_x || !dev_sx || !dev_out || M < 1) return fail(EV_EINVAL, "bad argument");
    if (M > m->M_cap) return fail(EV_ECAPACITY, "M exceeds max_batch * max_tree_nodes");
    cudaStream_t st = (cudaStream_t)stream;
    QMat* w = nullptr;
    ActBuf* x = nullptr;
    if (kind != EV_W_LM_HEAD && (layer < 0 || layer >= m->cfg.n_layers)) return fail(EV_EINVAL, "layer out of range");
    // fused storage: Q/K/V and GATE/UP are computed together (the kernel the step uses)
    switch (kind) {
        case EV_W_Q: w = &m->layers[layer].qkv; x = &m->xq; break;
        case EV_W_O: w = &m->layers[layer].o; x = &m->aq; break;
        case EV_W_GATE: w = &m->layers[layer].gu; x = &m->xq; break;
        case EV_W_DOWN: w = &m->layers[layer].down; x = &m->tq; break;
        case EV_W_LM_HEAD: w = &m->lm; x = &m->xq; break;
        default: return fail(EV_EINVAL, "ev_op_linear: kind must be Q (=fused QKV), O, GATE (=fused gate|up), DOWN or LM_HEAD");
    }
    CUDA_TRY(cudaMemcpyAsync(x->codes, dev_codes_x, (size_t)M * w->K, cudaMemcpyDeviceToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(x->scale, dev_sx, (size_t)M * 4, cudaMemcpyDeviceToDevice, st));
    if (kind == EV_W_LM_HEAD) {
        CUDA_TRY(cudaMemsetAsync(m->argmax_keys, 0, (size_t)M * 8, st));
        return run_linear(m, st, *w, *x, M, EPI_ARGMAX, nullptr, dev_out, m->argmax_keys, PC_OTHER);
    }
    LinOut lin;
    EV_TRY(run_linear(m, st, *w, *x, M, EPI_RAW, &lin, nullptr, nullptr, PC_OTHER));
    materialize_linear_kernel<<<M, 256, 0, st>>>(dev_out, (int)w->N, lin);
    LAUNCH_CHECK();
    return EV_OK;
}

// ev_op_linear for callers that may not allocate: the same GEMM kernel, same K cuts, same consumer - the kernel's scratch
// (K-piece slabs) lives in the file-scope device array ev_static_slabs instead of the model's workspace.  No cudaMalloc /
// cudaFree / allocating library call on this path (the address was resolved at set-up).
int ev_op_linear_static(ev_model* m, int kind, int layer, const uint8_t* dev_codes_x, const float* dev_sx, int M, float* dev_out,
                        void* stream) {
    if (!m || !dev_codes_x || !dev_sx || !dev_out || M < 1) return fail(EV_EINVAL, "bad argument");
    if (M > m->M_cap) return fail(EV_ECAPACITY, "M exceeds max_batch * max_tree_nodes");
    cudaStream_t st = (cudaStream_t)stream;
    QMat* w = nullptr;
    ActBuf* x = nullptr;
    if (layer < 0 || layer >= m->cfg.n_layers) return fail(EV_EINVAL, "layer out of range");
    switch (kind) {
        case EV_W_Q: w = &m->layers[layer].qkv; x = &m->xq; break;
        case EV_W_O: w = &m->layers[layer].o; x = &m->aq; break;
        case EV_W_GATE: w = &m->layers[layer].gu; x = &m->xq; break;
        case EV_W_DOWN: w = &m->layers[layer].down; x = &m->tq; break;
        default: return fail(EV_EINVAL, "ev_op_linear_static: kind must be Q (=fused QKV), O, GATE (=fused gate|up) or DOWN");
    }
    // worst case of the slab layout: 8 pieces per tile below 257 rows, one slab above (run_linear)
    const long need = (M <= 256 ? 8L : 1L) * M * (long)w->N;
    if (need > EV_STATIC_SLAB_FLOATS)
        return fail(EV_ECAPACITY, "ev_op_linear_static: (M <= 256 ? 8 : 1) * M * N = " + std::to_string(need) + " floats exceeds the static scratch of " +
                                      std::to_string(EV_STATIC_SLAB_FLOATS) + " floats (16 MiB); use ev_op_linear");
    float* slabs = nullptr;
    EV_TRY(static_slabs_ptr(&slabs));
    CUDA_TRY(cudaMemcpyAsync(x->codes, dev_codes_x, (size_t)M * w->K, cudaMemcpyDeviceToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(x->scale, dev_sx, (size_t)M * 4, cudaMemcpyDeviceToDevice, st));
    // the GEMM takes its slab pointer from the model: point it at the static array for this one launch.  Every slab element the
    // consumer reads is written by this launch's GEMM (pieces cover their tiles completely), so nothing has to start at zero.
    float* const saved_out = m->lin_out;
    const long saved_floats = m->lin_floats;
    m->lin_out = slabs; m->lin_floats = EV_STATIC_SLAB_FLOATS;
    LinOut lin;
    const int rc = run_linear(m, st, *w, *x, M, EPI_RAW, &lin, nullptr, nullptr, PC_OTHER);
    m->lin_out = saved_out; m->lin_floats = saved_floats;
    if (rc != EV_OK) return rc;
    materialize_linear_kernel<<<M, 256, 0, st>>>(dev_out, (int)w->N, lin);
    LAUNCH_CHECK();
    return EV_OK;
}


// ---- host-buffer entry point: copies in, one verify step, copies out, synchronises ---------------------
int ev_verify_host(ev_model* m, ev_cache* c, int n_seqs, int n_nodes, const int32_t* host_seq_slots,
                   const int32_t* host_tokens, const int32_t* host_parents, const int32_t* host_n_nodes, int commit,
                   int32_t* host_accept_len, int32_t* host_accept_nodes, int32_t* host_out_tokens,
                   int32_t* host_new_ctx_len, int32_t* host_status, void* stream) {
    if (!m || !c || !host_seq_slots || !host_tokens || !host_parents || !host_accept_len || !host_accept_nodes ||
        !host_out_tokens || !host_new_ctx_len || !host_status)
        return fail(EV_EINVAL, "null argument");
    if (n_seqs < 1 || n_nodes < 1) return fail(EV_EINVAL, "n_seqs and n_nodes must be positive");
    if (n_seqs > m->cfg.max_batch || n_nodes > m->cfg.max_tree_nodes) return fail(EV_ECAPACITY, "batch or tree too large");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t BT = (size_t)n_seqs * n_nodes;
    CUDA_TRY(cudaMemcpyAsync(c->pf_tokens, host_tokens, BT * 4, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(c->pf_parents, host_parents, BT * 4, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(c->pf_slots, host_seq_slots, (size_t)n_seqs * 4, cudaMemcpyHostToDevice, st));
    if (host_n_nodes) CUDA_TRY(cudaMemcpyAsync(c->pf_nn, host_n_nodes, (size_t)n_seqs * 4, cudaMemcpyHostToDevice, st));
    const int Bmax = m->cfg.max_batch;
    ev_verify_in in;
    memset(&in, 0, sizeof(in));
    in.n_seqs = n_seqs; in.n_nodes_max = n_nodes; in.dev_seq_slots = c->pf_slots; in.dev_tokens = c->pf_tokens;
    in.dev_parents = c->pf_parents; in.dev_n_nodes = host_n_nodes ? c->pf_nn : nullptr; in.commit = commit;
    ev_verify_out o;
    memset(&o, 0, sizeof(o));
    o.tap_layer = -1;
    o.dev_accept_len = c->pf_out; o.dev_new_ctx_len = c->pf_out + Bmax; o.dev_status = c->pf_out + 2 * Bmax;
    o.dev_accept_nodes = c->pf_out + 3 * Bmax; o.dev_out_tokens = o.dev_accept_nodes + (size_t)m->M_cap;
    EV_TRY(ev_verify(m, c, &in, &o, stream));
    CUDA_TRY(cudaMemcpyAsync(host_accept_len, o.dev_accept_len, (size_t)n_seqs * 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(host_new_ctx_len, o.dev_new_ctx_len, (size_t)n_seqs * 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(host_status, o.dev_status, (size_t)n_seqs * 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(host_accept_nodes, o.dev_accept_nodes, BT * 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(host_out_tokens, o.dev_out_tokens, BT * 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (commit)   // the true new lengths are on the host now: tighten the bounds plan_attention advanced by T
        for (int i = 0; i < n_seqs; ++i) {
            const int s = host_seq_slots[i];
            if (s >= 0 && s < c->max_seqs && c->seq_used[s] && host_status[i] == 0) c->len_bound[s] = host_new_ctx_len[i];
        }
    return EV_OK;
}

// ---- per-kernel-class device timing (CUDA events on the launching stream) ----------------------------------
int ev_profile_enable(ev_model* m, int on) {
    if (!m) return fail(EV_EINVAL, "null argument");
    m->profile = on == 1;
    m->prof_used = 0;
    const bool want_trace = on == 2;
    if (want_trace && !m->trace) {
        EV_TRY(dev_alloc(m, &m->trace, (size_t)TRACE_CAP * TRACE_SLOTS));
        CUDA_TRY(cudaMemset(m->trace, 0xFF, (size_t)TRACE_CAP * TRACE_SLOTS * 8));
    }
    if (want_trace != m->trace_on) {   // the trace slots are kernel arguments: captured steps are re-captured with / without them
        m->trace_on = want_trace;
        drop_graphs(m);
    }
    return EV_OK;
}
int ev_profile_read(ev_model* m, double* host_ms_by_class, long* host_count_by_class, int n_classes) {
    if (!m || !host_ms_by_class || !host_count_by_class || n_classes < 1) return fail(EV_EINVAL, "bad argument");
    for (int i = 0; i < n_classes; ++i) { host_ms_by_class[i] = 0.0; host_count_by_class[i] = 0; }
    CUDA_TRY(cudaDeviceSynchronize());
    for (size_t i = 0; i < m->prof_used; ++i) {
        float ms = 0.f;
        CUDA_TRY(cudaEventElapsedTime(&ms, m->prof[i].a, m->prof[i].b));
        const int c = m->prof[i].cls < n_classes ? m->prof[i].cls : n_classes - 1;
        host_ms_by_class[c] += ms;
        host_count_by_class[c] += 1;
    }
    m->prof_used = 0;
    return EV_OK;
}

// bring-up: copies the per-CTA GEMM phase timestamps of the last launch (EV_GEMM_DBG & 16) to the host
int ev_profile_trace(ev_model* m, unsigned long long* host_out, int max_entries, int* n_out) {
    if (!m || !host_out || !n_out) return fail(EV_EINVAL, "null argument");
    if (!m->trace || !m->trace_on) return fail(EV_ESTATE, "step trace is off (ev_profile_enable(model, 2) turns it on)");
    CUDA_TRY(cudaDeviceSynchronize());
    const int n = std::min(std::min(max_entries, m->n_traced), TRACE_CAP);
    CUDA_TRY(cudaMemcpy(host_out, m->trace, (size_t)n * TRACE_SLOTS * 8, cudaMemcpyDeviceToHost));
    for (int i = 0; i < n; ++i)
        for (int j = 2; j < TRACE_SLOTS; ++j) host_out[TRACE_SLOTS * i + j] = ~host_out[TRACE_SLOTS * i + j];
    CUDA_TRY(cudaMemset(m->trace, 0xFF, (size_t)TRACE_CAP * TRACE_SLOTS * 8));
    *n_out = n;
    return EV_OK;
}

}  // extern "C"

#include "ev_engine.inc"
