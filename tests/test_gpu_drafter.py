"""Draft side on the GPU vs oracle/drafter_oracle.py on the same seeded inputs:
the FC front end + draft layer + shared LM head (predicted features, top-k), level-by-level tree expansion, the extend step
with the target's features, and the closed loop draft -> verify -> accept -> extend, whose emitted tokens must equal the
GPU's plain greedy decode whatever the (random-weight) drafter proposes."""
import numpy as np
import pytest

import workloads as wl
from oracle import verify_oracle as vo
from oracle import drafter_oracle as do
from helpers import oracle_model, fresh_cache, rel_l2, LAYER_KINDS

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

SHAPE, SEED = wl.TINY, 0
DSHAPE = wl.ModelShape("tiny_drafter", 1, SHAPE.hidden, SHAPE.n_q_heads, SHAPE.n_kv_heads, SHAPE.head_dim, SHAPE.ffn, SHAPE.vocab,
                       SHAPE.rms_eps, SHAPE.rope_theta)


@pytest.fixture(scope="module")
def models():
    import paper_2606_18502_b200 as ev
    from gpu_helpers import gpu_model, bits_to_bf16_cuda
    tg = gpu_model(SHAPE, SEED, max_batch=4, max_tree_nodes=64, max_ctx=512)
    dg = ev.Model(DSHAPE, 4, 64, 512)
    to = oracle_model(SHAPE, SEED)
    dm = do.DraftModel(to, SHAPE)
    for k in LAYER_KINDS:
        bits = wl.weight_matrix_bf16(SHAPE, SEED, k, SHAPE.n_layers)      # the drafter layer's own stream
        dg.ev_model_set_weight(k, 0, bits_to_bf16_cuda(bits))
        dm.set_weight(k, bits)
    fc = wl.weight_matrix_bf16(SHAPE, SEED, "d_fc", 0)
    dg.ev_model_set_weight("d_fc", 0, bits_to_bf16_cuda(fc))
    dm.set_weight("d_fc", fc)
    ev.ev_model_share_head(dg, tg)
    return ev, tg, dg, to, dm


def _i32(x):
    return torch.as_tensor(np.asarray(x, dtype=np.int32)).cuda()


def test_drafter_forward_topk_and_tree_match_oracle(models):
    ev, tg, dg, to, dm = models
    H = SHAPE.hidden
    rng = np.random.default_rng(1)
    ids = rng.integers(0, SHAPE.vocab, size=40).astype(np.int32)
    # target features of the context (oracle); the drafter's cache = extend(ids, [0 ; feat[:-1]]) on both sides
    tc = fresh_cache(to, 128)
    _, hid = vo.forward_tree(to, tc, 0, ids, np.arange(-1, 39), want_hidden=True)
    feat = hid[-1]
    pre = np.concatenate([np.zeros((1, H), np.float32), feat[:-1]])
    odc = vo.OracleKV(dm.layer, 16, 16)
    odc.add_seq(0, 160)
    do.draft_extend(dm, odc, 0, ids, pre)
    dcache = ev.Cache(dg, 16, 2)
    slot = dcache.ev_cache_add_seq(160)
    slots = _i32([slot])
    tok_b = torch.zeros((1, 64), dtype=torch.int32, device="cuda")
    tok_b[0, :40] = _i32(ids)
    fe_b = torch.zeros((1, 64, H), dtype=torch.float32, device="cuda")
    fe_b[0, :40] = torch.from_numpy(pre).cuda()
    ev.ev_draft_extend(dg, dcache, slots, tok_b, fe_b, _i32([40]))
    torch.cuda.synchronize()
    assert dcache.ev_cache_get_len(slot) == 40
    from gpu_helpers import export_kv_bits
    g = export_kv_bits(dcache, slot, 0, 1, 40)[0]
    o = odc.export_dense(0, 0, 40)
    assert np.mean(g != o) <= 2e-3          # the drafter layer's K/V of the committed context (bf16 bits)
    # lock-step drafter pass over a tree with given tokens / features: predicted features, top-k
    par = wl.tree_parents(12, (3, 2, 2))
    toks = rng.integers(0, SHAPE.vocab, size=12).astype(np.int32)
    feats = rng.standard_normal((12, H)).astype(np.float32) * 0.3
    f_o, lg_o = do.draft_forward(dm, odc, 0, toks, feats, par)
    buf = ev.VerifyBuffers(dg, 1, 12, want_logits=True, want_final_hidden=True, topk=4)
    buf.set_inputs([slot], toks[None], par[None])
    buf.features = torch.from_numpy(feats).cuda()
    ev.ev_verify(dg, dcache, buf, commit=False)
    torch.cuda.synchronize()
    assert rel_l2(buf.final_hidden.cpu().numpy(), f_o) <= 1e-2
    lg = buf.logits.cpu().numpy()
    assert np.max(np.abs(lg - lg_o)) <= 2e-2 * lg_o.std()
    tk = buf.topk.cpu().numpy()
    for i in range(12):      # the GPU's top-k is exactly the top-k of the GPU's own logits, ties to the lower id
        assert tk[i].tolist() == do.top_k_tokens(lg[i], 4).tolist(), i
        srt = np.sort(lg_o[i])[::-1]
        if (srt[:4] - srt[1:5]).min() >= 1e-3:
            assert tk[i].tolist() == do.top_k_tokens(lg_o[i], 4).tolist(), i
    # level-by-level expansion against the oracle's
    root_feat = rng.standard_normal(H).astype(np.float32) * 0.3
    t_o, fh_o = do.expand_tree(dm, odc, 0, 17, root_feat, par)
    tokens_out = torch.zeros((1, 12), dtype=torch.int32, device="cuda")
    parents_out = torch.zeros((1, 12), dtype=torch.int32, device="cuda")
    ev.ev_draft_tree(dg, dcache, slots, par, _i32([17]), torch.from_numpy(root_feat[None]).cuda(), tokens_out, parents_out)
    torch.cuda.synchronize()
    assert parents_out.cpu().numpy()[0].tolist() == par.tolist()
    t_g = tokens_out.cpu().numpy()[0]
    assert t_g[0] == 17
    agree = int((t_g == t_o).sum())
    assert agree >= 10, (t_g, t_o)          # a near-tie may reorder one sibling pair; everything else is the oracle's tree
    assert dcache.ev_cache_get_len(slot) == 40      # drafting leaves the drafter's cache length alone


def test_closed_loop_draft_verify_extend_is_lossless_on_gpu(models):
    ev, tg, dg, to, dm = models
    from gpu_helpers import run_verify
    H, B = SHAPE.hidden, 3
    rng = np.random.default_rng(2)
    for par in (wl.tree_parents(16, (3, 2, 2, 1)), wl.chain_parents(4)):
        T = len(par)
        lens = [50 + 7 * b for b in range(B)]
        ids = [rng.integers(0, SHAPE.vocab, size=n).astype(np.int32) for n in lens]
        tcache = ev.Cache(tg, 2 * B * 20, 2 * B)
        s_slots = [tcache.ev_cache_add_seq(300) for _ in range(B)]
        g_slots = [tcache.ev_cache_add_seq(300) for _ in range(B)]
        dcache = ev.Cache(dg, B * 20, B)
        d_slots = [dcache.ev_cache_add_seq(300) for _ in range(B)]
        # context: target features from a non-committing chain pass, then prefill (target) and extend (drafter)
        carry = torch.zeros((B, H), dtype=torch.float32, device="cuda")
        roots = np.zeros(B, dtype=np.int32)
        for b in range(B):
            n = lens[b]
            fb = ev.VerifyBuffers(tg, 1, 64, want_final_hidden=True)
            assert n <= 64
            tk = np.zeros(64, np.int32)
            tk[:n] = ids[b]
            fb.set_inputs([s_slots[b]], tk[None], wl.chain_parents(64)[None], [n])
            ev.ev_verify(tg, tcache, fb, commit=False)
            torch.cuda.synchronize()
            feat = fb.final_hidden[:n]
            roots[b] = int(fb.argmax.cpu().numpy()[0, n - 1])
            carry[b] = feat[n - 1]
            tok_b = torch.zeros((1, 64), dtype=torch.int32, device="cuda")
            tok_b[0, :n] = _i32(ids[b])
            fe_b = torch.zeros((1, 64, H), dtype=torch.float32, device="cuda")
            fe_b[0, 1:n] = feat[:n - 1]
            ev.ev_draft_extend(dg, dcache, _i32([d_slots[b]]), tok_b, fe_b, _i32([n]))
        tcache.ev_cache_prefill(s_slots + g_slots, ids + ids)
        # plain greedy on the GPU
        n_greedy = 60
        greedy = np.zeros((B, n_greedy), dtype=np.int32)
        tok = roots.copy()
        for s in range(n_greedy):
            gb = run_verify(tg, tcache, g_slots, tok[:, None], np.full((B, 1), -1, np.int32), commit=True, want_logits=False, want_hidden=False)
            tok = gb.out_tokens.cpu().numpy()[:, 0].astype(np.int32)
            greedy[:, s] = tok
        # closed loop, everything on the device between steps
        vb = ev.VerifyBuffers(tg, B, T, want_final_hidden=True)
        vb.seq_slots.copy_(_i32(s_slots))
        dsl = _i32(d_slots)
        root_t = _i32(roots)
        ext_tok = torch.zeros((B, T), dtype=torch.int32, device="cuda")
        ext_fe = torch.zeros((B, T, H), dtype=torch.float32, device="cuda")
        ext_n = torch.zeros(B, dtype=torch.int32, device="cuda")
        emitted = [[] for _ in range(B)]
        accepted = 0
        for step in range(8):
            ev.ev_draft_tree(dg, dcache, dsl, par, root_t, carry, vb.tokens, vb.parents)
            ev.ev_verify(tg, tcache, vb, commit=True, use_n_nodes=False)
            ev.ev_gather_accepted(vb.tokens, vb.accept_len, vb.accept_nodes, vb.out_tokens, vb.final_hidden.view(B, T, H), carry,
                                  ext_tok, ext_fe, ext_n, root_t)
            ev.ev_draft_extend(dg, dcache, dsl, ext_tok, ext_fe, ext_n)
            torch.cuda.synchronize()
            acc, outs = vb.accept_len.cpu().numpy(), vb.out_tokens.cpu().numpy()
            assert (vb.status.cpu().numpy() == 0).all()
            for b in range(B):
                emitted[b] += outs[b, :acc[b] + 1].tolist()
                accepted += int(acc[b])
        for b in range(B):
            assert emitted[b] == greedy[b, :len(emitted[b])].tolist(), (b, emitted[b][:10], greedy[b, :10])
            assert dcache.ev_cache_get_len(d_slots[b]) == tcache.ev_cache_get_len(s_slots[b]) == lens[b] + len(emitted[b])
        print(f"closed loop T={T}: {sum(len(e) for e in emitted)} tokens in 8 steps x {B} sequences, {accepted} drafts accepted")
