"""8B-shape parity at BASELINE.json's full sizes on sampled outputs the oracle computes one by one (DESIGN.md
section 5): the GPU runs the whole step (all 32 layers, whole batch) once EAGERLY with hidden / per-kernel taps (what the
oracle is compared with) and once in the launch configuration bench.py times (no taps: the captured CUDA graph, the fused
down-GEMM -> next-norm path), whose integer outputs must equal the eager run's; for sampled (sequence, layer) pairs the oracle recomputes that layer from the GPU's own layer
input and the GPU's exported KV of that layer (verify = f(weights, KV, tree), DESIGN.md R-kv-input) and the
outputs are compared at the north_star tolerances: hidden rel-L2 <= 1e-2 per layer, logits <= 2e-2 sigma,
argmax equal where the oracle's top-2 gap >= 1e-3, acceptance walk / compaction indices bit-exact."""
import numpy as np
import pytest

import workloads as wl
from oracle import verify_oracle as vo
from helpers import rel_l2, LAYER_KINDS

pytestmark = [pytest.mark.gpu, pytest.mark.slow8b]
torch = pytest.importorskip("torch")

TOL_HIDDEN, TOL_LOGIT_SIGMA, GAP = 1e-2, 2e-2, 1e-3


def _setup(spec, sample_layers, batch=None, ctx_override=None):
    import paper_2606_18502_b200 as ev
    from gpu_helpers import bf16_cuda_to_bits
    shape = spec.model
    B = batch or spec.batch
    ctx = wl.context_lengths(spec)[:B] if ctx_override is None else np.asarray(ctx_override, dtype=np.int32)
    model = ev.Model(shape, max_batch=B, max_tree_nodes=64, max_ctx=int(ctx.max()) + 72, page_size=spec.page_size,
                     act_scale_mode=spec.act_scale_mode)
    host = {}
    for kind, layer in [("embed", 0)] + [(k, l) for l in range(shape.n_layers) for k in LAYER_KINDS] + [("lm_head", 0)]:
        w = wl.weight_matrix_bf16(shape, spec.seed, kind, layer, device="cuda")
        model.ev_model_set_weight(kind, layer, w)
        if kind == "lm_head" or (kind != "embed" and layer in sample_layers):
            host[(kind, layer)] = bf16_cuda_to_bits(w)
        del w
    torch.cuda.synchronize()
    om = vo.OracleModel(shape, act_scale_mode=spec.act_scale_mode)
    for (kind, layer), bits in host.items():
        om.set_weight(kind, layer, bits)
    return ev, model, om, ctx


def _check_quantized_weights(model, om, layer):
    for kind in ("wq", "wdown"):
        cg, sg = model.ev_model_get_quantized(kind, layer)
        co, so = om.w[(kind, layer)]
        assert np.array_equal(sg.cpu().numpy(), so) and np.array_equal(cg.cpu().numpy(), co), (kind, layer)


def _run_config(spec, sample_layers, sample_seqs, batch=None, ctx_override=None):
    from gpu_helpers import export_kv_bits, run_verify
    ev, model, om, ctx = _setup(spec, sample_layers, batch, ctx_override)
    shape = spec.model
    B, T = len(ctx), spec.n_nodes
    parents = wl.chain_parents(T) if spec.tree_caps is None else wl.tree_parents(T, spec.tree_caps)
    for l in sample_layers[:1]:
        _check_quantized_weights(model, om, l)
    if spec.act_scale_mode == 1:
        calib = wl.calibration_hidden(spec)
        taps = model.ev_model_calibrate(torch.from_numpy(calib).cuda(), want_layer_inputs=True)
        scales = model.ev_model_get_static_scales()
        # the oracle calibrates each sampled layer from the GPU's own input of that layer (needs causal KV of the
        # calibration run itself: recomputed by the oracle layer on an empty cache, chain of 512 tokens)
        par = np.arange(-1, calib.shape[0] - 1)
        for l in sample_layers:
            rec = {}
            oc = vo.OracleKV(om, calib.shape[0] // spec.page_size + 2, spec.page_size)
            oc.add_seq(0, calib.shape[0])
            vo.layer_forward(om, l, taps[l].cpu().numpy(), oc, 0, 0, par, record=rec)
            for j, site in enumerate(vo.SITES):
                ref = np.float32(rec[(site, l)]) / np.float32(448.0)
                assert abs(float(scales[4 * l + j]) - float(ref)) <= 2e-3 * float(ref), (l, site, scales[4 * l + j], ref)
        rec = {}
        vo.lm_head(om, taps[shape.n_layers].cpu().numpy(), record=rec)
        ref = np.float32(rec[("lm_in", 0)]) / np.float32(448.0)
        assert abs(float(scales[-1]) - float(ref)) <= 2e-3 * float(ref)
        # both sides now use the GPU's calibrated constants (one model, DESIGN.md R-static)
        for l in range(shape.n_layers):
            for j, site in enumerate(vo.SITES):
                om.static[(site, l)] = np.float32(scales[4 * l + j])
        om.static[("lm_in", 0)] = np.float32(scales[-1])
    pages = sum((int(L) + 64) // spec.page_size + 2 for L in ctx)
    cache = ev.Cache(model, pages, B)
    slots = [cache.ev_cache_add_seq(int(L) + 64) for L in ctx]
    cache.ev_cache_prefill(slots, [wl.context_ids(spec, b, int(ctx[b])) for b in range(B)])
    tokens = np.stack([wl.draft_tokens_uniform(spec, parents, b) for b in range(B)])
    tap_layer = sample_layers[0]
    buf = run_verify(model, cache, slots, tokens, np.tile(parents, (B, 1)), commit=False, want_logits=True,
                     want_hidden=True, tap_layer=tap_layer)
    assert (buf.status.cpu().numpy() == 0).all()
    hid = buf.hidden.cpu().numpy().reshape(shape.n_layers + 1, B, T, shape.hidden)
    logits = buf.logits.cpu().numpy().reshape(B, T, shape.vocab)
    am = buf.argmax.cpu().numpy()
    report = []
    for b in sample_seqs:
        L = int(ctx[b])
        for l in sample_layers:
            oc = vo.OracleKV(om, (L + T) // spec.page_size + 2, spec.page_size)
            oc.add_seq(0, L + T)
            oc.import_dense(l, 0, export_kv_bits(cache, slots[b], l, l + 1, L)[0])
            oc.ctx_len[0] = L
            taps = {}
            h_ref = vo.layer_forward(om, l, hid[l, b], oc, 0, L, parents, taps=taps)
            err = rel_l2(hid[l + 1, b], h_ref)
            report.append((b, l, err))
            assert err <= TOL_HIDDEN, (b, l, err)
            # appended tree K/V (bf16): same bits except where an upstream E4M3 code differs
            g = export_kv_bits(cache, slots[b], l, l + 1, L + T)[0][:, :, L:]
            o = oc.export_dense(l, 0, L + T)[:, :, L:]
            assert np.count_nonzero(g != o) <= 2e-3 * g.size, np.count_nonzero(g != o) / g.size
            assert rel_l2(wl.bf16_bits_to_f32(g), wl.bf16_bits_to_f32(o)) <= 1e-3
            if l == tap_layer:
                t = {k: v.cpu().numpy().reshape(B, T, -1)[b] for k, v in buf.taps.items() if v.dim() == 2}
                assert np.mean(t["xq"] != taps["xq"]) <= 1e-4
                assert rel_l2(t["attn"], taps["attn"]) <= 1e-5, rel_l2(t["attn"], taps["attn"])
                assert np.mean(t["aq"] != taps["aq"]) <= 1e-3
        lg_ref = vo.lm_head(om, hid[shape.n_layers, b])
        sigma = float(lg_ref.std())
        dl = float(np.max(np.abs(logits[b] - lg_ref)))
        report.append((b, "lm", dl / sigma))
        assert dl <= TOL_LOGIT_SIGMA * sigma, (b, dl, sigma)
        srt = np.sort(lg_ref, axis=1)
        ok = (srt[:, -1] - srt[:, -2]) >= GAP
        assert np.array_equal(am[b][ok], np.argmax(lg_ref, axis=1)[ok])
    # acceptance walk + compaction indices, bit-exact on the GPU's own argmax, every sequence
    acc = buf.accept_len.cpu().numpy()
    nodes = buf.accept_nodes.cpu().numpy()
    outs = buf.out_tokens.cpu().numpy()
    newl = buf.new_ctx_len.cpu().numpy()
    for b in range(B):
        path, out = vo.accept_walk(tokens[b], parents, am[b])
        a = len(path) - 1
        assert acc[b] == a and nodes[b, :a + 1].tolist() == path and outs[b, :a + 1].tolist() == out
        assert newl[b] == int(ctx[b]) + a + 1
    # the launch configuration bench.py times (CUDA graph replay, no taps) gives the same integers as the eager tapped run
    for rep in range(2):       # first call captures, second replays
        fast = run_verify(model, cache, slots, tokens, np.tile(parents, (B, 1)), commit=False, want_logits=False, want_hidden=False)
        assert np.array_equal(fast.argmax.cpu().numpy(), am)
        assert np.array_equal(fast.accept_len.cpu().numpy(), acc) and np.array_equal(fast.accept_nodes.cpu().numpy(), nodes)
        assert np.array_equal(fast.out_tokens.cpu().numpy(), outs) and np.array_equal(fast.new_ctx_len.cpu().numpy(), newl)
    print("8B parity report (seq, layer|lm, rel-L2 | max|d|/sigma):", report)
    return report


def test_config1_b1_L2048_tree60_full_size():
    _run_config(wl.CONFIGS[1], sample_layers=[0, 17, 31], sample_seqs=[0])


def test_config2_b32_L4096_tree26_full_size():
    _run_config(wl.CONFIGS[2], sample_layers=[1, 30], sample_seqs=[0, 31])


def test_config3_b64_mixed_context_chain3_full_size():
    _run_config(wl.CONFIGS[3], sample_layers=[2], sample_seqs=[0, 63])


def test_config4_b8_L16384_tree60_static_scales_full_size():
    _run_config(wl.CONFIGS[4], sample_layers=[0, 16], sample_seqs=[7])


# ---- GPU self-consistency at 8B shape ("guaranteeing to preserve accuracy"):
# the GPU speculative loop emits exactly the tokens of GPU token-by-token greedy decoding, bit for bit.  Holds by
# construction: every contraction's reduction order is a function of the token's own data (canonical K cuts of the
# GEMMs, attention chunks at absolute key positions + per-row tail, segment-ordered RMSNorm sums).

def _rank0_chain(parents):
    """nodes whose every ancestor-or-self is the lowest-index child of its parent, by depth (root excluded)."""
    first_child = {}
    for i in range(1, len(parents)):
        first_child.setdefault(int(parents[i]), i)
    chain, cur = [], 0
    while cur in first_child:
        cur = first_child[cur]
        chain.append(cur)
    return chain


def _lossless(spec, B, ctx, n_steps=8, planted_p=0.7, kv_fp8=False):
    import paper_2606_18502_b200 as ev
    from gpu_helpers import run_verify
    shape = spec.model
    T = spec.n_nodes
    parents = wl.chain_parents(T) if spec.tree_caps is None else wl.tree_parents(T, spec.tree_caps)
    depth = int(wl.tree_depths(parents).max())
    n_greedy = n_steps * (depth + 1) + depth + 1
    model = ev.Model(shape, max_batch=2 * B, max_tree_nodes=64, max_ctx=int(max(ctx)) + n_greedy + 80, page_size=spec.page_size,
                     act_scale_mode=spec.act_scale_mode, kv_dtype=1 if kv_fp8 else 0)
    for kind, layer in [("embed", 0)] + [(k, l) for l in range(shape.n_layers) for k in LAYER_KINDS] + [("lm_head", 0)]:
        model.ev_model_set_weight(kind, layer, wl.weight_matrix_bf16(shape, spec.seed, kind, layer, device="cuda"))
    if spec.act_scale_mode == 1 or kv_fp8:
        model.ev_model_calibrate(torch.from_numpy(wl.calibration_hidden(spec, None if spec.calib_tokens else 512)).cuda())
    cap = [int(L) + n_greedy + 72 for L in ctx]
    cache = ev.Cache(model, 2 * sum(c // spec.page_size + 2 for c in cap) + cap[0] // spec.page_size + 2, 2 * B + 1)
    s_slots = [cache.ev_cache_add_seq(c) for c in cap]     # speculative decoding
    g_slots = [cache.ev_cache_add_seq(c) for c in cap]     # plain greedy decoding
    ids = [wl.context_ids(spec, b, int(ctx[b])) for b in range(B)]
    cache.ev_cache_prefill(s_slots + g_slots, ids + ids)
    rng = np.random.default_rng(spec.seed + 77)
    roots = rng.integers(0, shape.vocab, size=B).astype(np.int32)
    # --- plain greedy: one token per sequence per step (M = B rows; sequence 0 also alone, M = 1: batch invariance)
    greedy = np.zeros((B, n_greedy), dtype=np.int32)
    tok = roots.copy()
    one = np.full((B, 1), -1, dtype=np.int32)
    for s in range(n_greedy):
        buf = run_verify(model, cache, g_slots, tok[:, None], one, commit=True, want_logits=False, want_hidden=False)
        assert (buf.status.cpu().numpy() == 0).all()
        tok = buf.out_tokens.cpu().numpy()[:, 0].astype(np.int32)
        greedy[:, s] = tok
    # --- speculative loop with planted drafts
    chain = _rank0_chain(parents)
    emitted = [[] for _ in range(B)]
    root = roots.copy()
    total_acc = 0
    for s in range(n_steps):
        tokens = np.zeros((B, T), dtype=np.int32)
        for b in range(B):
            tk = rng.integers(0, shape.vocab, size=T).astype(np.int32)
            tk[0] = root[b]
            e = len(emitted[b])
            for d, node in enumerate(chain):
                if rng.random() < planted_p:
                    tk[node] = greedy[b, e + d]
            for i in range(1, T):      # siblings distinct (DESIGN.md R-tokens)
                sib = [tk[j] for j in range(1, i) if parents[j] == parents[i]]
                while tk[i] in sib:
                    tk[i] = (tk[i] + 1) % shape.vocab
            tokens[b] = tk
        buf = run_verify(model, cache, s_slots, tokens, np.tile(parents, (B, 1)), commit=True, want_logits=False, want_hidden=False)
        assert (buf.status.cpu().numpy() == 0).all()
        acc = buf.accept_len.cpu().numpy()
        outs = buf.out_tokens.cpu().numpy()
        for b in range(B):
            a = int(acc[b])
            emitted[b] += outs[b, :a + 1].tolist()
            root[b] = outs[b, a]
            total_acc += a
    for b in range(B):
        n = len(emitted[b])
        assert emitted[b] == greedy[b, :n].tolist(), (b, emitted[b], greedy[b, :n].tolist())
    # the planted drafts were accepted about as often as planted (1 + sum p^d emitted per step; loose lower bound)
    assert total_acc >= 0.5 * B * n_steps * planted_p, total_acc
    # compacted cache == cache of plain decoding, bit for bit (all layers), for sequence 0
    n0 = int(ctx[0]) + len(emitted[0])
    a = cache.ev_cache_export_seq(s_slots[0], 0, shape.n_layers, n0)
    g = cache.ev_cache_export_seq(g_slots[0], 0, shape.n_layers, n0)
    assert torch.equal(a.view(torch.int16), g.view(torch.int16))
    # sequence 0 decoded ALONE (M = 1) gives the same tokens as in the batch of B
    if B > 1:
        solo = cache.ev_cache_add_seq(cap[0])
        cache.ev_cache_prefill([solo], [ids[0]])
        tok1 = roots[:1].copy()
        for s in range(8):
            buf = run_verify(model, cache, [solo], tok1[:, None], one[:1], commit=True, want_logits=False, want_hidden=False)
            tok1 = buf.out_tokens.cpu().numpy()[:, 0].astype(np.int32)
            assert int(tok1[0]) == int(greedy[0, s]), s
    print(f"lossless {spec.name}: {sum(len(e) for e in emitted)} tokens emitted in {n_steps} steps x {B} sequences, {total_acc} drafts accepted")


def test_config1_gpu_speculative_equals_gpu_greedy():
    _lossless(wl.CONFIGS[1], 1, [2048])


def test_config2_gpu_speculative_equals_gpu_greedy():
    _lossless(wl.CONFIGS[2], 4, [4096, 4096, 4096, 4096])


def test_config3_gpu_speculative_equals_gpu_greedy():
    spec = wl.CONFIGS[3]
    ctx = wl.context_lengths(spec)
    _lossless(spec, 4, [int(ctx[0]), int(ctx[1]), int(ctx.min()), int(ctx.max())])


def test_config4_gpu_speculative_equals_gpu_greedy():
    _lossless(wl.CONFIGS[4], 2, [16384, 16384])


def test_config2_fp8_kv_cache_gpu_speculative_equals_gpu_greedy():
    """SURVEY section 8(f)-2 at 8B shape: the same bit-exact self-consistency with the FP8 (E4M3) KV cache."""
    import dataclasses
    _lossless(dataclasses.replace(wl.CONFIGS[2], name="cfg2_fp8kv"), 3, [4096, 4096, 3000], kv_fp8=True)


def test_drafter_forward_at_8b_shape_matches_oracle():
    """SURVEY section 8(f)-3 at 8B shape: FC (K = 8192) + one decoder layer + shared LM head of the draft model against
    oracle/drafter_oracle.py, lock-step from given predecessor features: predicted features rel-L2 <= 1e-2, logits <= 2e-2
    sigma, top-k equal where the oracle's gaps are >= 1e-3."""
    import dataclasses
    import paper_2606_18502_b200 as ev
    from oracle import drafter_oracle as do
    from gpu_helpers import bf16_cuda_to_bits
    shape = wl.LLAMA8B
    seed = 9
    dshape = dataclasses.replace(shape, name="llama8b_drafter", n_layers=1)
    dg = ev.Model(dshape, 1, 64, 256)
    tshape = dataclasses.replace(shape, name="llama8b_head_only", n_layers=1)     # a stand-in target: only its embedding, final norm and LM head are used
    to = vo.OracleModel(tshape)
    dm = do.DraftModel(to, shape)
    for kind in ("embed", "lm_head"):
        w = wl.weight_matrix_bf16(shape, seed, kind, 0, device="cuda")
        dg.ev_model_set_weight(kind, 0, w)
        to.set_weight(kind, 0, bf16_cuda_to_bits(w))
    for k in LAYER_KINDS:
        w = wl.weight_matrix_bf16(shape, seed, k, shape.n_layers, device="cuda")
        dg.ev_model_set_weight(k, 0, w)
        dm.set_weight(k, bf16_cuda_to_bits(w))
    w = wl.weight_matrix_bf16(shape, seed, "d_fc", 0, device="cuda")
    dg.ev_model_set_weight("d_fc", 0, w)
    dm.set_weight("d_fc", bf16_cuda_to_bits(w))
    del w
    rng = np.random.default_rng(4)
    H = shape.hidden
    ctx_tok = rng.integers(0, shape.vocab, size=48).astype(np.int32)
    ctx_feat = (rng.standard_normal((48, H)) * 2.0).astype(np.float32)
    par = wl.tree_parents(12, (3, 2, 2))
    toks = rng.integers(0, shape.vocab, size=12).astype(np.int32)
    feats = (rng.standard_normal((12, H)) * 2.0).astype(np.float32)
    odc = vo.OracleKV(dm.layer, 8, 16)
    odc.add_seq(0, 100)
    do.draft_extend(dm, odc, 0, ctx_tok, ctx_feat)
    f_o, lg_o = do.draft_forward(dm, odc, 0, toks, feats, par)
    dcache = ev.Cache(dg, 8, 1)
    slot = dcache.ev_cache_add_seq(100)
    i32 = lambda x: torch.as_tensor(np.asarray(x, dtype=np.int32)).cuda()  # noqa: E731
    tb = torch.zeros((1, 64), dtype=torch.int32, device="cuda")
    tb[0, :48] = i32(ctx_tok)
    fb = torch.zeros((1, 64, H), dtype=torch.float32, device="cuda")
    fb[0, :48] = torch.from_numpy(ctx_feat).cuda()
    ev.ev_draft_extend(dg, dcache, i32([slot]), tb, fb, i32([48]))
    buf = ev.VerifyBuffers(dg, 1, 12, want_logits=True, want_final_hidden=True, topk=4)
    buf.set_inputs([slot], toks[None], par[None])
    buf.features = torch.from_numpy(feats).cuda()
    ev.ev_verify(dg, dcache, buf, commit=False)
    torch.cuda.synchronize()
    f_g = buf.final_hidden.cpu().numpy()
    assert rel_l2(f_g, f_o) <= 1e-2, rel_l2(f_g, f_o)
    # logits lock-step from the GPU's own predicted features (one quantization site)
    lg_ref = vo.lm_head(to, f_g)
    lg = buf.logits.cpu().numpy()
    assert np.max(np.abs(lg - lg_ref)) <= 2e-2 * lg_ref.std()
    tk = buf.topk.cpu().numpy()
    for i in range(12):
        assert tk[i].tolist() == do.top_k_tokens(lg[i], 4).tolist(), i          # exactly the top-k of the GPU's own logits
        srt = np.sort(lg_ref[i])[::-1]
        if (srt[:4] - srt[1:5]).min() >= 1e-3:
            assert tk[i].tolist() == do.top_k_tokens(lg_ref[i], 4).tolist(), i


@pytest.mark.gpu
@pytest.mark.parametrize("attn_chunk", [0, 256])
def test_verify_is_repeatable_bit_for_bit_at_8b_shape(attn_chunk):
    """No compute-sanitizer on this pool: a race in the warp-specialised kernels (the attention kernel's two MMA issuers and its
    S/P hand-over, the GEMMs' pair epilogue) would show up as run-to-run differences.  The same verify step - two 8B-shaped
    layers, ragged contexts spanning one to twelve key tiles per CTA, a 26-node tree - is run forty times without commit:
    logits, final hidden states and accepted tokens must be identical bit for bit (attention chunking: the library default
    and 256-key chunks = 4 tiles per CTA, many CTAs per sequence)."""
    import dataclasses
    import paper_2606_18502_b200 as ev
    from gpu_helpers import run_verify
    spec = wl.CONFIGS[2]
    shape = dataclasses.replace(spec.model, name="llama8b_2layers", n_layers=2)
    ctx = [37, 64, 700, 1543, 3001]
    B, T = len(ctx), spec.n_nodes
    parents = wl.tree_parents(T, spec.tree_caps)
    model = ev.Model(shape, max_batch=B, max_tree_nodes=64, max_ctx=max(ctx) + 128, page_size=spec.page_size, attn_chunk=attn_chunk)
    for kind, layer in [("embed", 0)] + [(k, l) for l in range(shape.n_layers) for k in LAYER_KINDS] + [("lm_head", 0)]:
        model.ev_model_set_weight(kind, layer, wl.weight_matrix_bf16(shape, spec.seed, kind, layer, device="cuda"))
    cache = ev.Cache(model, sum(c // spec.page_size + 8 for c in ctx), B)
    slots = [cache.ev_cache_add_seq(c + 64) for c in ctx]
    cache.ev_cache_prefill(slots, [wl.context_ids(spec, b, ctx[b]) for b in range(B)])
    rng = np.random.default_rng(5)
    tokens = rng.integers(0, shape.vocab, size=(B, T)).astype(np.int32)
    ref = None
    for it in range(40):
        buf = run_verify(model, cache, slots, tokens, np.tile(parents, (B, 1)), commit=False, want_logits=True, want_hidden=True)
        assert (buf.status.cpu().numpy() == 0).all()
        cur = (buf.logits.view(torch.int32).clone(), buf.hidden.view(torch.int32).clone(), buf.out_tokens.clone(), buf.accept_len.clone())
        if ref is None:
            ref = cur
            assert torch.isfinite(buf.logits).all()
        else:
            for a, b in zip(ref, cur):
                assert torch.equal(a, b), it
