/*
 * eagle_verify.h - C ABI of the B200 (sm_100a) FP8 EAGLE tree-verification library.
 *
 * The one hot path this library implements (BASELINE.json:north_star): the target model's
 * forward pass over all nodes of a draft-token tree against a paged bf16 KV cache, with FP8
 * (E4M3) W8A8 linear layers, followed by greedy acceptance and the KV append:
 *     verify(tree, cache) -> accepted tokens + bonus token + compacted KV.
 * Paper passages that define the operations (PAPER.md = the paper text, section / line):
 *   - PAPER.md:98  (sec. 3.2) FP8 (E4M3) weight-and-activation quantization (W8A8), min-max
 *     post-training quantization, static scales from calibration data.
 *   - PAPER.md:361 (App. E)   draft trees "verified in a single forward pass of the target model
 *     via tree attention"; greedy drafts = a single candidate chain.
 *   - PAPER.md:92  (sec. 3.1) verification preserves the target model's output (lossless).
 * Readings of everything the paper leaves open are listed in DESIGN.md section 3.
 *
 * Conventions
 *   - Plain C, no C++/torch types.  Every function returns 0 (EV_OK) or a negative ev_status;
 *     none throws, aborts or prints.  ev_last_error() gives a thread-local message.
 *   - "dev_" pointers are CUDA device pointers (e.g. tensor.data_ptr()); "host_" pointers are
 *     host memory.  `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *   - Ownership: the caller owns every buffer it passes and must keep it alive until the stream
 *     has passed the call.  The library owns handles, quantized weights, the page pool and its
 *     workspaces; they are released by the matching *_destroy.
 *   - Asynchrony: calls taking a stream only enqueue work; outputs are valid after the caller
 *     synchronises that stream.  ev_verify in steady state performs no host synchronisation and no allocation:
 *     it replays a CUDA graph.  The FIRST call with a new (batch, tree size, buffer set, attention chunk-column count)
 *     captures and instantiates that graph (host work of a few ms; ev_capture_count counts them) and, when top-k is asked
 *     for without a logits buffer, allocates a logits workspace once.  Data-dependent failures (bad parent index, token id out
 *     of range, sequence over capacity or beyond the attention grid, two rows of one batch on the same sequence) are reported
 *     per sequence in ev_verify_out.dev_status, not by return code.
 *   - Batch invariance: every reduction's order is a function of the token's own data (DESIGN.md R-invariant): a row's
 *     results do not depend on the other rows of the call, on the tree it arrives in (depth <= 8), or on the GPU.
 *   - The shipped library reads no environment variable (bring-up switches exist only in -DEV_BRINGUP builds).
 *   - Layouts: all matrices row-major.  Weights [out_channels][in_channels] (K contiguous).
 *     Hidden states / logits [token][channel].  Batched tree arrays [B][T] with T = n_nodes_max.
 *   - A tree: node 0 is the root = the last emitted token, whose KV is not yet cached
 *     (DESIGN.md R-root); parents[0] = -1 and 0 <= parents[i] < i.  T <= 64.
 *     Node i sits at position ctx_len + depth(i) (north_star (3)) and its K/V are written to
 *     slot ctx_len + i of the sequence during the forward pass.
 */
#ifndef EAGLE_VERIFY_H
#define EAGLE_VERIFY_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define EV_MAX_TREE_NODES 64

typedef enum {
    EV_OK = 0,
    EV_EINVAL = -1,    /* bad argument (null pointer, shape mismatch, unsupported config) */
    EV_ENOMEM = -2,    /* device or host allocation failed */
    EV_ECAPACITY = -3, /* page pool / sequence slots / workspace exhausted */
    EV_ECUDA = -4,     /* a CUDA runtime or driver call failed; see ev_last_error() */
    EV_ESTATE = -5     /* call not valid in the handle's current state (e.g. weights missing) */
} ev_status;

/* per-sequence status bits written to ev_verify_out.dev_status */
#define EV_SEQ_OK 0
#define EV_SEQ_BAD_TREE 1     /* parents[] malformed or n_nodes out of range */
#define EV_SEQ_BAD_TOKEN 2    /* a token id outside [0, vocab) */
#define EV_SEQ_OVER_CAPACITY 4 /* ctx_len + n_nodes exceeds the sequence's reserved pages */

typedef struct ev_model ev_model;
typedef struct ev_cache ev_cache;

typedef struct {
    int n_layers, hidden, n_q_heads, n_kv_heads;
    int head_dim;         /* 64 or 128 */
    int ffn, vocab;
    float rms_eps, rope_theta;
    int page_size;        /* tokens per KV page; 16 */
    int act_scale_mode;   /* 0 = dynamic per-token activation scales; 1 = static calibrated */
    int max_batch;        /* B upper bound per ev_verify call */
    int max_tree_nodes;   /* T upper bound, <= EV_MAX_TREE_NODES */
    int max_ctx;          /* upper bound on ctx_len + tree nodes of any sequence (RoPE table) */
    int weight_scale_mode; /* 0 = one E4M3 scale per output channel (BASELINE.json:north_star); 1 = one scale per
                            * weight matrix, absmax / 448 over the whole matrix ("per-tensor";
                            * SURVEY section 8(f)-1; each of Q, K, V, gate, up keeps its own scale) */
    int attn_chunk;        /* keys per attention chunk: 0 = default (1024), else a multiple of 64.  A node's key set is reduced in
                            * chunks aligned to ABSOLUTE key positions plus a short tail, so its
                            * result does not depend on batch, tree or GPU; the chunk length is part of the model's arithmetic:
                            * two models with different attn_chunk agree only to fp32 rounding */
    int kv_dtype;          /* 0 = bf16 KV cache (BASELINE.json configs; values rounded to bf16, held in IEEE binary16 containers: exact for
                            * 2^-17 <= |x| <= 65504, 2^-25 absolute below, saturating above); 1 = FP8 (E4M3) KV cache, one byte per
                            * element ("quantizing the KV cache to FP8 halves the storage"): K (after
                            * RoPE) and V are stored as E4M3_sat(x / s) with ONE static scale per layer for K and one for V, set by
                            * ev_model_calibrate (absmax over the calibration tokens / 448) or ev_model_set_kv_scales; needs page_size
                            * 16 and head_dim 128 */
} ev_config;

typedef enum {
    EV_W_EMBED = 0, /* [vocab][hidden] bf16, kept bf16 */
    EV_W_Q = 1, EV_W_K = 2, EV_W_V = 3, EV_W_O = 4, EV_W_GATE = 5, EV_W_UP = 6, EV_W_DOWN = 7,
    EV_W_LM_HEAD = 8,                    /* 1..8: quantized to E4M3 on arrival */
    EV_W_NORM1 = 9, EV_W_NORM2 = 10, EV_W_NORMF = 11, /* RMSNorm gains [hidden] bf16; default 1.0 */
    EV_W_DRAFT_FC = 12  /* draft models only: [hidden][2*hidden] bf16 -> E4M3, the EAGLE front end that maps
                           [embedding ; predecessor feature] to the draft layer's input (no bias) */
} ev_weight_kind;

/* ---- model: quantize / calibrate weights -------------------------------------------------- */

/* Creates an empty model (allocates quantized-weight storage, workspaces sized from max_batch *
 * max_tree_nodes, the fp64-built RoPE table).  Errors: EV_EINVAL, EV_ENOMEM, EV_ECUDA. */
int ev_model_create(const ev_config* cfg, ev_model** out);

/* Uploads one weight.  dev_bf16: [rows][cols] bf16 on the device, read during the call's stream
 * work and not retained.  Matrices EV_W_Q..EV_W_LM_HEAD are quantized per output channel (row):
 * s_w[n] = max_k|W[n,k]| / 448 (1 for a zero row), code = E4M3_RNE_sat(W[n,k] / s_w[n])
 * (PAPER.md:98 min-max PTQ; BASELINE.json per-output-channel).  rows/cols must match cfg. */
int ev_model_set_weight(ev_model*, int kind, int layer, const void* dev_bf16, long rows, long cols,
                        void* stream);

/* Copies a quantized matrix (kinds 1..8) out of the library: E4M3 codes row-major [rows][cols] into
 * dev_codes_out and fp32 per-output-channel scales [rows] into dev_scales_out (both caller-owned device
 * buffers).  Internally the codes live in the GEMM's tiled, swizzled HBM layout; this call un-tiles.
 * rows/cols must equal the matrix shape.  Q/K/V (and GATE/UP) are sub-ranges of fused storage. */
int ev_model_get_quantized(ev_model*, int kind, int layer, uint8_t* dev_codes_out, float* dev_scales_out,
                           long rows, long cols, void* stream);

/* Static activation scales (act_scale_mode 1; "Static quantization sets scales offline
 * from activation statistics collected on calibration data"; DESIGN.md R-static): runs
 * dev_hidden [n_tok][hidden] fp32 as the layer-0 residual stream of n_tok causal tokens at positions
 * 0..n_tok-1 with dynamic scales, records per quantization site (4 per layer + LM head input) the
 * absmax over all tokens and channels, and sets scale = absmax / 448 for every later call.
 * Any n_tok <= max_ctx (processed in chunks of max_tree_nodes tokens against a temporary cache).
 * Setup call: synchronises the stream internally.  dev_layer_inputs (optional, may be NULL) receives the residual
 * stream entering every layer and after the last: [n_layers+1][n_tok][hidden] fp32. */
int ev_model_calibrate(ev_model*, const float* dev_hidden, int n_tok, float* dev_layer_inputs,
                       void* stream);

/* Copies the 4*n_layers+1 static scales to host_out in site order
 * (layer-major: qkv_in, o_in, gateup_in, down_in; then lm_in).  Synchronous. */
int ev_model_get_static_scales(ev_model*, float* host_out);
/* Overrides them (same order); used to replay externally calibrated scales. */
int ev_model_set_static_scales(ev_model*, const float* host_in);
/* FP8 KV cache scales (kv_dtype 1): 2*n_layers floats, (K, V) per layer.  get: after calibration; set: replays external scales
 * (all > 0).  Both synchronous host calls; set drops the captured CUDA graphs. */
int ev_model_get_kv_scales(ev_model*, float* host_out);
int ev_model_set_kv_scales(ev_model*, const float* host_in);
/* Clip counters (Fig. 4 "clip rate"): with static scales
 * (act_scale_mode == 1) every activation quantizer counts the elements it saturates, |x| > 448 * s_site,
 * per site, in the order of ev_model_get_static_scales, accumulated over all calls since the last reset
 * (calibration passes do not count).  Copies the 4*n_layers+1 counters to host_out (host memory owned by the
 * caller); reset != 0 zeroes them afterwards.  Synchronous (waits for the device).  All zero in dynamic
 * mode.  Returns EV_EINVAL on null arguments. */
int ev_model_get_clip_counts(ev_model*, unsigned long long* host_out, int reset);

int ev_model_destroy(ev_model*);

/* ---- paged bf16 KV cache ------------------------------------------------------------------- */

/* Pool of n_pages pages; each page holds page_size tokens for all layers.
 * Device layout: [layer][page][K|V][kv_head][page_size][head_dim], 2 bytes per element (bf16 VALUES in IEEE binary16
 * containers when page_size is 16 - the tcgen05 attention kernel's operand format, see ev_config.kv_dtype - plain bf16
 * otherwise) or 1 byte per element (E4M3 codes, kv_dtype 1). */
int ev_cache_create(ev_model*, long n_pages, int max_seqs, ev_cache** out);

/* Reserves ceil(capacity_tokens / page_size) pages for a new sequence (ctx_len = 0) and returns
 * its slot.  host_pages (optional): explicit physical page ids to use (tests of page-order
 * invariance); NULL = take from the free list.  EV_ECAPACITY when pages or slots run out. */
int ev_cache_add_seq(ev_cache*, int capacity_tokens, const int* host_pages, int* seq_slot_out);
int ev_cache_free_seq(ev_cache*, int seq_slot);

/* Context KV by definition: the K/V the quantized model yields for the token ids under causal
 * attention, appended after each sequence's current ctx_len.  host_token_ids: the sequences' ids
 * concatenated (host memory); host_lens[i] ids for sequence host_seq_slots[i].  Runs chain trees of
 * up to max_tree_nodes tokens per sequence per pass with every node accepted (no LM head).
 * Setup call: synchronises the stream after every pass. */
int ev_cache_prefill(ev_model*, ev_cache*, int n_seqs, const int* host_seq_slots,
                     const int32_t* host_token_ids, const int* host_lens, void* stream);

/* Dense export/import of one sequence's first n_tokens slots for layers [layer_begin, layer_end):
 * dev_dense: [layer][K|V][kv_head][n_tokens][head_dim] bf16 (kv_dtype 1: uint8 E4M3 codes).  import also sets
 * ctx_len = n_tokens when set_len != 0. */
int ev_cache_export_seq(ev_cache*, int seq_slot, int layer_begin, int layer_end, int n_tokens,
                        void* dev_dense, void* stream);
int ev_cache_import_seq(ev_cache*, int seq_slot, int layer_begin, int layer_end, int n_tokens,
                        const void* dev_dense, int set_len, void* stream);

/* ctx_len lives on the device (ev_verify with commit advances it without host involvement).
 * set: enqueued on the stream.  get: synchronises the stream. */
int ev_cache_set_len(ev_cache*, int seq_slot, int ctx_len, void* stream);
int ev_cache_get_len(ev_cache*, int seq_slot, int* ctx_len, void* stream);
/* Sets the ctx_len of up to 64 sequences with one launch (rewinds a batch between timed steps). */
int ev_cache_set_lens(ev_cache*, int n, const int* host_slots, const int* host_lens, void* stream);
int ev_cache_destroy(ev_cache*);

/* ---- verify --------------------------------------------------------------------------------- */

typedef struct {
    int n_seqs;                 /* B <= max_batch */
    int n_nodes_max;            /* T <= max_tree_nodes; row stride of the [B][T] arrays */
    const int32_t* dev_seq_slots; /* [B] cache slots */
    const int32_t* dev_tokens;  /* [B][T] node tokens; [b][0] = root */
    const int32_t* dev_parents; /* [B][T] parent indices; [b][0] = -1 */
    const int32_t* dev_n_nodes; /* [B] nodes in use per sequence, or NULL = all T */
    int commit;                 /* 1 = compact accepted KV to slots L..L+a and set ctx_len = L+a+1 */
    int force_accept_all;       /* 1 = (prefill) treat every node as accepted; chain trees only */
    const float* dev_hidden_override; /* lock-step debug: [n_layers+1][B*T][hidden]; layer l reads
                                     its input from slice l instead of the previous layer's output
                                     (slice n_layers feeds the LM head); or NULL */
    int override_first_only;    /* 1 = only slice 0 (replaces the embedding) is read */
    const float* dev_features;  /* draft models (EV_W_DRAFT_FC set): [B*T][hidden] predecessor feature of every node; the
                                   layer-0 input is FC(Q8([embed(token) ; feature])) instead of the embedding; or NULL */
} ev_verify_in;

typedef struct {
    int32_t* dev_accept_len;    /* [B] a = accepted draft tokens, 0..depth */
    int32_t* dev_accept_nodes;  /* [B][T] accepted path incl. root at [0] (a+1 valid) = KV-compaction
                                   source indices; rest -1 */
    int32_t* dev_out_tokens;    /* [B][T] accepted tokens then the bonus token (a+1 valid); rest -1 */
    int32_t* dev_new_ctx_len;   /* [B] L + a + 1 (whether or not commit is set) */
    int32_t* dev_status;        /* [B] EV_SEQ_* bits */
    int32_t* dev_argmax;        /* optional [B][T] target argmax per node (lowest id on ties) */
    float* dev_logits;          /* optional [B*T][vocab] */
    float* dev_hidden;          /* optional [n_layers+1][B*T][hidden] residual stream taps */
    /* optional per-kernel taps of one layer (all may be NULL) */
    int tap_layer;
    uint8_t* dev_tap_xq;  float* dev_tap_sx;     /* RMSNorm1+quant: [M][hidden] codes, [M] scales */
    float* dev_tap_qkv;                          /* after RoPE: [M][(Hq+2Hkv)*d] (K,V pre-bf16) */
    float* dev_tap_attn;                         /* attention output [M][Hq*d] fp32 */
    uint8_t* dev_tap_aq;  float* dev_tap_sa;     /* its quantization */
    float* dev_tap_hmid;                         /* residual after O-proj [M][hidden] */
    float* dev_tap_gu;                           /* gate|up GEMM output [M][2*ffn] */
    uint8_t* dev_tap_tq;  float* dev_tap_st;     /* SwiGLU + quant: [M][ffn] codes, [M] scales */
    float* dev_final_hidden;    /* optional [B*T][hidden]: the residual stream after the last layer = the "feature" an EAGLE
                                   drafter consumes (target) / predicts (draft model); graph-captured like the rest */
    int32_t* dev_topk;          /* optional [B*T][topk]: the topk tokens with the largest logits per node, largest first,
                                   ties to the lower id (tree expansion); topk <= 8 */
    int topk;
} ev_verify_out;

/* One verify step for B sequences.  M = B*T rows are processed together by
 * every decoder layer.  Required outputs: accept_len, accept_nodes, out_tokens, new_ctx_len, status.
 * Errors (host-detectable only): EV_EINVAL, EV_ECAPACITY (B or T over the model's maxima), EV_ESTATE
 * (weights missing / not calibrated in static mode), EV_ECUDA (launch failure). */
int ev_verify(ev_model*, ev_cache*, const ev_verify_in*, ev_verify_out*, void* stream);

/* The same step with HOST buffers: copies tokens/parents/slots (and n_nodes, may be NULL) to the device,
 * runs ev_verify, copies the five result arrays back ([B] or [B][n_nodes] int32) and synchronises the
 * stream.  Host buffers should be pinned for the copies to be asynchronous.  This is the end-to-end
 * call bench.py times. */
int ev_verify_host(ev_model*, ev_cache*, int n_seqs, int n_nodes, const int32_t* host_seq_slots,
                   const int32_t* host_tokens, const int32_t* host_parents, const int32_t* host_n_nodes,
                   int commit, int32_t* host_accept_len, int32_t* host_accept_nodes,
                   int32_t* host_out_tokens, int32_t* host_new_ctx_len, int32_t* host_status, void* stream);

/* ---- draft side (architecture from the EAGLE paper the paper cites) -----------
 * A draft model is an ev_model with n_layers = 1 of the target's shape, its seven layer matrices, EV_W_DRAFT_FC, and the
 * target's embedding / final norm / LM head (ev_model_share_head: pointers, no copy; the target must outlive the drafter).
 * It keeps its own ev_cache.  Node p's input is [embed(token_p) ; feature_{p-1}]: committed positions use the TARGET's
 * features (ev_draft_extend after every verify step), draft nodes the drafter's own prediction for their parent. */
int ev_model_share_head(ev_model* drafter, ev_model* target);

typedef struct {
    int n_seqs, n_nodes;               /* B, T */
    const int32_t* dev_seq_slots;      /* [B] slots in the drafter's cache */
    const int32_t* host_parents;       /* [T] ONE static topology for the batch, nodes ordered by depth, parents[0] = -1 */
    const int32_t* dev_root_tokens;    /* [B] last emitted token of every sequence */
    const float* dev_root_feats;       /* [B][hidden] target feature preceding the root */
    int32_t* dev_tokens;               /* out [B][T]: the drafted tree's tokens (node 0 = root) */
    int32_t* dev_parents;              /* out [B][T]: the topology per sequence, as ev_verify takes it */
} ev_draft_args;
/* Expands the static tree level by level on the stream (no host sync): level d runs the drafter over the nodes of depth <= d
 * (rows are independent given their ancestors, so re-running earlier levels changes nothing), takes every node's top-k
 * tokens, and gives the child of rank r the parent's (r+1)-th best token and the parent's predicted feature.  The
 * drafter's cache is NOT advanced (draft nodes are scratch).  A chain topology is greedy drafting. */
int ev_draft_tree(ev_model* drafter, ev_cache* dcache, const ev_draft_args*, void* stream);
/* Commits tokens to the drafter's cache with the given predecessor features: dev_tokens [B][T], dev_feats [B][T][hidden],
 * dev_n [B] tokens in use per sequence (chains; every node kept; ctx_len += n). */
int ev_draft_extend(ev_model* drafter, ev_cache* dcache, int n_seqs, int n_nodes, const int32_t* dev_seq_slots,
                    const int32_t* dev_tokens, const float* dev_feats, const int32_t* dev_n, void* stream);
/* After a target verify step: builds ev_draft_extend's inputs from the accepted path - row j <= a of sequence b holds the
 * accepted node's token and the TARGET feature of the accepted node before it (row 0: dev_carry[b], the feature preceding the
 * old root) - then dev_next_root[b] = the bonus token and dev_carry[b] = the feature of the last accepted node.  All device
 * pointers: tokens/accept_nodes/out_tokens [B][T], accept_len [B], feat [B][T][hidden] (ev_verify_out.dev_final_hidden),
 * carry [B][hidden], ext_tokens [B][T], ext_feats [B][T][hidden], ext_n [B], next_root [B]. */
int ev_gather_accepted(int n_seqs, int n_nodes, int hidden, const int32_t* dev_tokens, const int32_t* dev_accept_len,
                       const int32_t* dev_accept_nodes, const int32_t* dev_out_tokens, const float* dev_feat, float* dev_carry,
                       int32_t* dev_ext_tokens, float* dev_ext_feats, int32_t* dev_ext_n, int32_t* dev_next_root, void* stream);

/* ---- serving shell: continuous batching around verify ("continuous batching") -------------
 * An engine owns a set of requests.  Every ev_engine_step is one iteration of iteration-level scheduling: waiting requests are
 * admitted while batch rows and KV pages are free (their prompt is prefilled into the target cache and, with a drafter,
 * into the drafter's cache with the target's features), then ONE speculative step runs for all active requests together
 * (draft tree -> verify -> accept -> KV compaction -> drafter extend), emitted tokens are appended to each request's output
 * and finished requests leave, freeing their pages - the next step's batch has a different composition.  Because every
 * kernel of the path is batch-invariant, a request's tokens do not depend on which other requests share its steps.
 * Without a drafter (drafter == NULL) the step is plain decoding (one node per sequence). */
typedef struct ev_engine ev_engine;
typedef struct {
    int max_batch;                /* rows per step, <= both models' max_batch */
    int n_nodes;                  /* T of the static draft topology (ignored without a drafter) */
    const int32_t* host_parents;  /* [T] topology, nodes ordered by depth (copied) */
} ev_engine_config;
int ev_engine_create(ev_model* target, ev_cache* tcache, ev_model* drafter, ev_cache* dcache, const ev_engine_config*, ev_engine** out);
/* Queues a request: host_prompt[n_prompt] (n_prompt >= 2, copied), generate max_new_tokens tokens.  Returns its id. */
int ev_engine_submit(ev_engine*, const int32_t* host_prompt, int n_prompt, int max_new_tokens, int* request_id);
/* One scheduling iteration on the stream; synchronises it (results come back to the host every step).  Outputs: requests active
 * during the step, requests that finished in it, requests still waiting for rows or pages. */
int ev_engine_step(ev_engine*, int* n_active, int* n_finished, int* n_waiting, void* stream);
/* Copies up to cap generated tokens of a request to host_tokens_out; *n_out = tokens generated so far (capped at
 * max_new_tokens), *finished = 1 once it has left the batch. */
int ev_engine_poll(ev_engine*, int request_id, int32_t* host_tokens_out, int cap, int* n_out, int* finished);
int ev_engine_destroy(ev_engine*);

/* ---- single operators (per-kernel parity tests; same kernels the step uses) ------------------ */

/* y[M][N] = (codes_x . W_kind^T) * s_x[m] * s_w[n] with the product GEMM kernel. */
int ev_op_linear(ev_model*, int kind, int layer, const uint8_t* dev_codes_x, const float* dev_sx,
                 int M, float* dev_out, void* stream);
/* ev_op_linear for callers that may not allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc).  Same GEMM kernel, same canonical K cuts, same result bit for bit; kinds Q (= fused QKV),
 * O, GATE (= fused gate|up), DOWN.  The kernel's scratch - the fp32 K-piece slabs [pieces][M][N] its consumer sums - lives in a
 * file-scope `static __device__` array of EV_STATIC_SCRATCH_BYTES (16 MiB, resident on every GPU that loads the library until
 * the process exits) instead of the model's workspace; its device address is resolved with cudaGetSymbolAddress once per
 * device at ev_model_create.  The call performs no cudaMalloc / cudaFree / allocating library call.
 *   dev_codes_x [M][K] E4M3 codes, dev_sx [M] fp32 scales, dev_out [M][N] fp32: device pointers, caller-owned.
 *   Limit: (M <= 256 ? 8 : 1) * M * N * 4 bytes <= EV_STATIC_SCRATCH_BYTES (the worst-case slab layout), else EV_ECAPACITY
 *   (ev_last_error names both numbers) - e.g. M <= 60 for every layer GEMM of the 8B shape except gate|up (M <= 18).
 *   The array is shared by every call from every model and thread and keeps the last call's contents; nothing has to start
 *   at zero (each launch writes every slab element its consumer reads).  Two calls that overlap on the GPU (different
 *   streams, or concurrent host threads) RACE on it: serialise them.  ev_verify and ev_op_linear never touch it. */
#define EV_STATIC_SCRATCH_BYTES (16 << 20)
int ev_op_linear_static(ev_model*, int kind, int layer, const uint8_t* dev_codes_x, const float* dev_sx,
                        int M, float* dev_out, void* stream);
/* per-token dynamic (or static, scale > 0) E4M3 quantization of fp32 rows */
int ev_op_quantize_rows(ev_model*, const float* dev_x, int M, int K, float static_scale,
                        uint8_t* dev_codes, float* dev_sx, void* stream);

/* ---- introspection ---------------------------------------------------------------------------- */
/* Device timing per kernel class with CUDA events recorded on the launching stream around each
 * launch (classes: 0..4 FP8 GEMM of QKV / O / gate-up / down / LM head, 5 tree attention, 6 attention
 * merge+quant, 7 RMSNorm+quant, 8 RoPE+KV write, 9 SwiGLU+quant, 10 other).  enable(1) starts recording; read() synchronises the
 * device, sums elapsed ms and launch counts per class into the host arrays and clears the record. */
int ev_profile_enable(ev_model*, int on);
int ev_profile_read(ev_model*, double* host_ms_by_class, long* host_count_by_class, int n_classes);
/* ev_profile_enable(m, 1): per-class CUDA-event timing (the step then runs eagerly); (m, 2): step trace; (m, 0): both off.
 * Step trace: every kernel of the layer loop of the last ev_verify (CUDA-graph replays included: this is how a kernel's
 * duration INSIDE the replayed, programmatic-dependent-launch step is measured) records, with %globaltimer, min over its CTAs of the time it
 * entered, min and max of the time it passed griddepcontrol.wait, and max of the time it left.
 * host_out[i][8] = {t_enter, t_past_wait_first, t_exit, t_past_wait_last, 4 bring-up phase marks} in ns for launch i, in launch
 * order (per layer: norm, QKV, RoPE, attention, merge, O, norm, gate/up, SwiGLU, down; then norm, LM
 * head); *n_out = launches traced.  Synchronises the device; clears the trace. */
int ev_profile_trace(ev_model*, unsigned long long* host_out, int max_entries, int* n_out);
const char* ev_last_error(void);
/* kernels launched by the calling thread's library calls since the last reset */
long ev_launch_count(int reset);
/* verify steps captured into a CUDA graph by the calling thread's ev_verify calls since the last reset: the first call with a
 * new (batch, tree size, buffer set, attention chunk-column count) captures and instantiates (host work, ~ms); every later
 * call with the same set replays.  A steady decode loop captures once per chunk-column boundary a sequence crosses. */
long ev_capture_count(int reset);
int ev_version(void);

#ifdef __cplusplus
}
#endif
#endif /* EAGLE_VERIFY_H */
