"""Pins for oracle/drafter_oracle.py: wiring of the FC front end, feature-level
chain == incremental drafting, tree == per-path chains, top-k expansion by brute force, and the closed loop's losslessness
(the emitted tokens equal the target's greedy decode whatever the drafter predicts)."""
import numpy as np
import pytest

import workloads as wl
from oracle import verify_oracle as vo
from oracle import drafter_oracle as do
from helpers import oracle_model, fresh_cache, small_shape, LAYER_KINDS

MICRO = small_shape()


def _drafter(target, seed=7, fc_bits=None):
    dm = do.DraftModel(target, MICRO)
    for k in LAYER_KINDS:
        dm.set_weight(k, wl.weight_matrix_bf16(MICRO, seed, k, MICRO.n_layers))      # an extra layer index: its own stream
    dm.set_weight("d_fc", wl.weight_matrix_bf16(MICRO, seed, "d_fc", 0) if fc_bits is None else fc_bits)
    return dm


def _dcache(dm, n=96):
    c = vo.OracleKV(dm.layer, n // 16 + 2, 16)
    c.add_seq(0, n)
    return c


def test_child_ranks_and_top_k():
    par = np.array([-1, 0, 0, 0, 1, 1, 2, 4])
    assert do.child_ranks(par).tolist() == [0, 0, 1, 2, 0, 1, 0, 0]
    rng = np.random.default_rng(0)
    lg = rng.standard_normal(50).astype(np.float32)
    lg[7] = lg[3] = lg.max() + 1.0          # a tie at the top: lower id first
    got = do.top_k_tokens(lg, 5).tolist()
    brute = sorted(range(50), key=lambda t: (-float(lg[t]), t))[:5]
    assert got == brute and got[:2] == [3, 7]


def test_fc_wiring_selects_embedding_or_feature():
    """FC = [I | 0] passes the (quantized) token embedding, FC = [0 | I] the predecessor feature: pins the concat order."""
    target = oracle_model(MICRO, seed=3)
    H = MICRO.hidden
    eye = np.eye(H, dtype=np.float32)
    zero = np.zeros((H, H), dtype=np.float32)
    toks = np.array([5, 9, 11], dtype=np.int32)
    feats = np.random.default_rng(1).standard_normal((3, H)).astype(np.float32)
    for blocks, want in (((eye, zero), vo.embed(target, toks)), ((zero, eye), feats)):
        dm = _drafter(target, fc_bits=wl.f32_to_bf16_bits(np.concatenate(blocks, axis=1)))
        x = np.concatenate([vo.embed(target, toks), feats], axis=1)
        xq, sx = vo.quantize_rows(x)
        h0 = vo.linear(xq, sx, dm.fc[0], dm.fc[1])
        # identity weights quantize to code(448) * 1/448: h0 is the dequantized quantized input's selected half
        deq = (vo.e4m3.decode(xq) * sx[:, None].astype(np.float64)).astype(np.float32)
        half = deq[:, :H] if blocks[0] is eye else deq[:, H:]
        assert np.allclose(h0, half, rtol=1e-6, atol=1e-9)
        assert np.allclose(h0, want, rtol=0.07, atol=0.07 * np.abs(want).max())      # E4M3 step


def test_chain_drafting_equals_incremental_and_tree_equals_paths():
    target = oracle_model(MICRO, seed=3)
    dm = _drafter(target)
    rng = np.random.default_rng(2)
    ctx_tok = rng.integers(0, MICRO.vocab, size=12).astype(np.int32)
    ctx_feat = rng.standard_normal((12, MICRO.hidden)).astype(np.float32)
    toks = rng.integers(0, MICRO.vocab, size=6).astype(np.int32)
    feats = rng.standard_normal((6, MICRO.hidden)).astype(np.float32)
    ca = _dcache(dm)
    do.draft_extend(dm, ca, 0, ctx_tok, ctx_feat)
    f_all, lg_all = do.draft_forward(dm, ca, 0, toks, feats, wl.chain_parents(6))
    cb = _dcache(dm)
    do.draft_extend(dm, cb, 0, ctx_tok, ctx_feat)
    for i in range(6):
        f, lg = do.draft_extend(dm, cb, 0, toks[i:i + 1], feats[i:i + 1])
        assert np.array_equal(f, f_all[i]) and np.array_equal(lg, lg_all[i]), i
    # tree: each node == the last node of its root path run as a chain
    par = np.array([-1, 0, 0, 1, 1, 2], dtype=np.int32)
    cc = _dcache(dm)
    do.draft_extend(dm, cc, 0, ctx_tok, ctx_feat)
    f_tree, lg_tree = do.draft_forward(dm, cc, 0, toks, feats, par)
    for i in range(6):
        path = [i]
        while par[path[-1]] >= 0:
            path.append(int(par[path[-1]]))
        path = path[::-1]
        cd = _dcache(dm)
        do.draft_extend(dm, cd, 0, ctx_tok, ctx_feat)
        f, lg = do.draft_forward(dm, cd, 0, toks[path], feats[path], wl.chain_parents(len(path)))
        assert np.array_equal(f[-1], f_tree[i]) and np.array_equal(lg[-1], lg_tree[i]), i


def test_expand_tree_children_are_the_parents_top_k_and_features_chain():
    target = oracle_model(MICRO, seed=3)
    dm = _drafter(target)
    rng = np.random.default_rng(4)
    par = wl.tree_parents(12, (3, 2, 2))
    dc = _dcache(dm)
    do.draft_extend(dm, dc, 0, rng.integers(0, MICRO.vocab, size=9), rng.standard_normal((9, MICRO.hidden)).astype(np.float32))
    root_feat = rng.standard_normal(MICRO.hidden).astype(np.float32)
    tokens, f_hat = do.expand_tree(dm, dc, 0, 17, root_feat, par)
    assert tokens[0] == 17
    # re-derive every child from ONE full forward with the final tokens (rows independent): parent's logits, brute force
    feats = np.zeros((12, MICRO.hidden), dtype=np.float32)
    feats[0] = root_feat
    for i in range(1, 12):
        feats[i] = f_hat[par[i]]
    dc2 = _dcache(dm)
    dc2.pool, dc2.page_table, dc2.ctx_len = dc.pool, dc.page_table, dict(dc.ctx_len)
    f2, lg2 = do.draft_forward(dm, dc2, 0, tokens, feats, par)
    assert np.array_equal(f2, f_hat)
    rank = do.child_ranks(par)
    for i in range(1, 12):
        order = sorted(range(MICRO.vocab), key=lambda t: (-float(lg2[par[i]][t]), t))
        assert tokens[i] == order[rank[i]], i
    sib = {}
    for i in range(1, 12):
        sib.setdefault(int(par[i]), []).append(int(tokens[i]))
    assert all(len(set(v)) == len(v) for v in sib.values())       # siblings distinct by construction


@pytest.mark.parametrize("caps,T", [((3, 2, 1), 9), (None, 4)])
def test_closed_loop_is_lossless_and_a_self_drafting_target_accepts_everything(caps, T):
    target = oracle_model(MICRO, seed=3)
    dm = _drafter(target)
    par = wl.chain_parents(T) if caps is None else wl.tree_parents(T, caps)
    ids = np.random.default_rng(5).integers(0, MICRO.vocab, size=14).astype(np.int32)
    tg = fresh_cache(target, 128)
    last_logits = vo.prefill(target, tg, 0, ids)
    root = int(vo.argmax_lowest(last_logits[-1:])[0])
    greedy = vo.decode_greedy(target, tg, 0, root, 24)
    # speculative: the drafter's cache is built from the context with the target's features (hidden of the prefill)
    ts = fresh_cache(target, 128)
    _, hid = vo.forward_tree(target, ts, 0, ids, np.arange(-1, len(ids) - 1), want_hidden=True)
    ts.ctx_len[0] = len(ids)
    feat = hid[-1]
    dc = _dcache(dm, 128)
    # token p with the feature of p-1; position 0 has no predecessor: zero feature (DESIGN.md R-drafter)
    do.draft_extend(dm, dc, 0, ids, np.concatenate([np.zeros((1, MICRO.hidden), np.float32), feat[:-1]]))
    assert dc.ctx_len[0] == ts.ctx_len[0] == len(ids)
    out, acc = do.speculative_generate(target, ts, dm, dc, 0, root, feat[-1], par, 6)
    assert out == greedy[:len(out)] and len(out) >= 6
    assert ts.ctx_len[0] == len(ids) + len(out)
