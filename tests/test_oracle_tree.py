"""Pins P4-P11: the oracle's tree forward, acceptance walk and KV append against what the paper
fixes: chain == token-by-token decoding and tree attention == per-path recomputation
(PAPER.md:361), losslessness of greedy verification, zero-initialised blocks are
identity maps, plus brute force on tiny trees and paging invariances."""
import itertools

import numpy as np
import pytest

import workloads as wl
from oracle import verify_oracle as vo
from helpers import oracle_model, small_shape, fresh_cache

MICRO = small_shape()


@pytest.fixture(scope="module")
def micro():
    return oracle_model(MICRO, seed=11, random_gains=True)


def _ctx(shape, n, seed=0):
    return np.random.default_rng(seed).integers(0, shape.vocab, n).astype(np.int32)


def _run_chain_as_decode(model, ids_ctx, toks):
    """logits after each of `toks`, fed one at a time."""
    cache = fresh_cache(model, len(ids_ctx) + len(toks) + 1)
    vo.prefill(model, cache, 0, ids_ctx, chunk=7)
    outs = []
    for t in toks:
        lg, _ = vo.forward_tree(model, cache, 0, np.array([t]), np.array([-1]))
        cache.ctx_len[0] += 1
        outs.append(lg[0])
    return np.stack(outs)


def test_p4_chain_equals_token_by_token_decode(micro):
    ids = _ctx(MICRO, 21)
    toks = _ctx(MICRO, 6, seed=1)
    cache = fresh_cache(micro, 40)
    vo.prefill(micro, cache, 0, ids, chunk=64)
    lg, _ = vo.forward_tree(micro, cache, 0, toks, wl.chain_parents(6))
    ref = _run_chain_as_decode(micro, ids, toks)
    assert np.array_equal(lg, ref)            # bit-identical: rows independent, K/V bf16 either way


def test_prefill_chunking_invariance(micro):
    ids = _ctx(MICRO, 30, seed=2)
    outs = []
    for chunk in (1, 7, 64):
        cache = fresh_cache(micro, 32)
        outs.append((vo.prefill(micro, cache, 0, ids, chunk=chunk)[-1], cache.export_dense(1, 0, 30)))
    for lg, kv in outs[1:]:
        assert np.array_equal(lg, outs[0][0]) and np.array_equal(kv, outs[0][1])


def _all_parent_arrays(n):
    for tail in itertools.product(*[range(i) for i in range(1, n)]):
        yield np.array((-1,) + tail)


def _check_tree_vs_paths(model, ids, parents, toks):
    cache = fresh_cache(model, len(ids) + len(parents))
    vo.prefill(model, cache, 0, ids)
    lg, _ = vo.forward_tree(model, cache, 0, toks, parents)
    for i in range(len(parents)):
        path = []
        j = i
        while j >= 0:
            path.append(j)
            j = int(parents[j])
        path = path[::-1]
        c2 = fresh_cache(model, len(ids) + len(path))
        vo.prefill(model, c2, 0, ids)
        lp, _ = vo.forward_tree(model, c2, 0, toks[path], wl.chain_parents(len(path)))
        assert np.array_equal(lp[-1], lg[i]), (parents, i)


def test_p5_tree_mask_equals_per_path_recompute_exhaustive(micro):
    ids = _ctx(MICRO, 5, seed=3)
    for n in (1, 2, 3, 4):
        for parents in _all_parent_arrays(n):
            _check_tree_vs_paths(micro, ids, parents, _ctx(MICRO, n, seed=4 + n))
    for k, parents in enumerate(_all_parent_arrays(5)):       # 24 labelled trees of 5 nodes
        _check_tree_vs_paths(micro, ids, parents, _ctx(MICRO, 5, seed=20 + k))


def test_p5_random_trees_up_to_8_nodes(micro):
    rng = np.random.default_rng(5)
    for _ in range(4):
        n = 8
        parents = np.array([-1] + [int(rng.integers(0, i)) for i in range(1, n)])
        _check_tree_vs_paths(micro, _ctx(MICRO, 19, seed=6), parents, _ctx(MICRO, n, seed=int(rng.integers(1 << 30))))


def _spec_loop(model, ids, root, n_tokens, draft_fn, shape):
    cache = fresh_cache(model, len(ids) + n_tokens + 16)
    vo.prefill(model, cache, 0, ids)
    emitted, lens = [], []
    while len(emitted) < n_tokens:
        parents, toks = draft_fn(root, len(emitted))
        r = vo.verify(model, cache, 0, toks, parents)
        emitted += r["out_tokens"]
        lens.append(len(r["out_tokens"]))
        root = r["out_tokens"][-1]
        toks[0] = root
    return emitted[:n_tokens], lens, cache


def test_p6_losslessness_against_plain_greedy(micro):
    """speculative decoding 'guarantee[s] to preserve accuracy'."""
    ids = _ctx(MICRO, 17, seed=7)
    root, n = 3, 24
    cache = fresh_cache(micro, 17 + n + 2)
    vo.prefill(micro, cache, 0, ids)
    greedy = vo.decode_greedy(micro, cache, 0, root, n)
    rng = np.random.default_rng(8)
    tree_p = wl.tree_parents(12, (3, 2, 2))

    def random_draft(root, pos):
        toks = rng.integers(0, MICRO.vocab, len(tree_p)).astype(np.int32)
        toks[0] = root
        return tree_p, toks

    def planted_draft(root, pos):       # rank-0 chain follows the true continuation, siblings random
        toks = rng.integers(0, MICRO.vocab, len(tree_p)).astype(np.int32)
        toks[0] = root
        d = vo.node_depths(tree_p)
        first_child = {}
        for i in range(1, len(tree_p)):
            first_child.setdefault(int(tree_p[i]), i)
        cur = 0
        while cur in first_child and pos + d[first_child[cur]] - 1 < len(greedy):
            c = first_child[cur]
            toks[c] = greedy[pos + d[c] - 1]
            cur = c
        return tree_p, toks

    def adversarial_chain(root, pos):   # right, right, wrong, right...: must stop at the first wrong one
        toks = np.array([root] + [greedy[min(pos + j, n - 1)] for j in range(4)], dtype=np.int32)
        toks[3] = (toks[3] + 1) % MICRO.vocab
        return wl.chain_parents(5), toks

    for fn, min_mean in ((random_draft, 1.0), (planted_draft, 2.5), (adversarial_chain, 2.5)):
        emitted, lens, _ = _spec_loop(micro, ids, root, n, fn, MICRO)
        assert emitted == greedy, fn.__name__
        assert np.mean(lens) >= min_mean, (fn.__name__, lens)
        if fn is adversarial_chain:
            assert all(l == 3 for l in lens[:-1])


def test_p6_cache_after_speculation_equals_cache_after_decode(micro):
    ids = _ctx(MICRO, 9, seed=9)
    cache = fresh_cache(micro, 40)
    vo.prefill(micro, cache, 0, ids)
    greedy = vo.decode_greedy(micro, cache, 0, 5, 10)
    ref_kv = cache.export_dense(1, 0, 9 + 10)
    p = np.array([-1, 0, 0, 1, 2, 3])          # two branches; the right one is node 2 -> 4

    def draft(root, pos):
        toks = np.array([root, 0, 0, 0, 0, 0], dtype=np.int32)
        g = greedy + [0, 0, 0]
        toks[1], toks[3], toks[5] = (g[pos] + 1) % MICRO.vocab, g[pos + 1], g[pos + 2]
        toks[2], toks[4] = g[pos], g[pos + 1]
        return p, toks
    emitted, lens, c2 = _spec_loop(micro, ids, 5, 10, draft, MICRO)
    assert emitted == greedy and lens[0] == 3
    n = min(c2.ctx_len[0], 19)
    assert np.array_equal(c2.export_dense(1, 0, n), ref_kv[:, :, :n])      # compaction moved the right slots


def test_p7_zero_output_projections_make_the_layer_an_identity():
    """zero-initialised inserted blocks are identity maps at initialisation."""
    m = oracle_model(MICRO, seed=12)
    z = np.zeros((MICRO.hidden, MICRO.q_dim), dtype=np.uint16)
    m.set_weight("wo", 1, z)
    m.set_weight("wdown", 1, np.zeros((MICRO.hidden, MICRO.ffn), dtype=np.uint16))
    cache = fresh_cache(m, 16)
    h = np.random.default_rng(0).standard_normal((5, MICRO.hidden)).astype(np.float32)
    out = vo.layer_forward(m, 1, h, cache, 0, 0, wl.chain_parents(5))
    assert np.array_equal(out, h)
    assert not np.array_equal(vo.layer_forward(m, 0, h, cache, 0, 0, wl.chain_parents(5)), h)


def test_p8_acceptance_walk_brute_force():
    rng = np.random.default_rng(13)
    for trial in range(300):
        n = int(rng.integers(1, 9))
        parents = np.array([-1] + [int(rng.integers(0, i)) for i in range(1, n)])
        toks = np.zeros(n, dtype=np.int32)
        for i in range(1, n):                                   # sibling-distinct small alphabet
            sib = {int(toks[j]) for j in range(1, i) if parents[j] == parents[i]}
            toks[i] = next(t for t in rng.permutation(8) if t not in sib)
        am = rng.integers(0, 8, n).astype(np.int32)
        path, out = vo.accept_walk(toks, parents, am)
        # brute force: the longest root path whose every token equals the argmax at its parent
        best = [0]
        for i in range(n):
            chain = []
            j = i
            while j >= 0:
                chain.append(j)
                j = int(parents[j])
            chain = chain[::-1]
            if all(toks[c] == am[p] for p, c in zip(chain[:-1], chain[1:])) and len(chain) > len(best):
                best = chain
        assert path == best
        assert out == [int(toks[c]) for c in best[1:]] + [int(am[best[-1]])]
    # leaf => bonus from the leaf; a = 0 => bonus from the root; duplicate siblings: lowest index wins
    assert vo.accept_walk(np.array([9, 4]), np.array([-1, 0]), np.array([4, 7])) == ([0, 1], [4, 7])
    assert vo.accept_walk(np.array([9, 4]), np.array([-1, 0]), np.array([5, 7])) == ([0], [5])
    assert vo.accept_walk(np.array([9, 4, 4, 1, 2]), np.array([-1, 0, 0, 1, 2]), np.array([4, 1, 2, 0, 0]))[0] == [0, 1, 3]


def test_p9_paging_invariances(micro):
    ids = _ctx(MICRO, 21, seed=14)            # 21: not a multiple of 16; 21+6 crosses a page boundary
    parents = np.array([-1, 0, 0, 1, 2, 4])
    toks = _ctx(MICRO, 6, seed=15)
    outs = []
    for page_size, order in ((16, None), (16, [5, 2, 7, 0, 3, 1, 4, 6]), (1, None), (64, None), (4, list(range(15, -1, -1)))):
        n_pages = len(order) if order else None
        cache = fresh_cache(micro, 40, page_size=page_size, page_order=order, n_pages=n_pages)
        vo.prefill(micro, cache, 0, ids)
        r = vo.verify(micro, cache, 0, toks, parents)
        outs.append((r["logits"], r["path"], cache.export_dense(0, 0, cache.ctx_len[0])))
    for lg, path, kv in outs[1:]:
        assert np.array_equal(lg, outs[0][0]) and path == outs[0][1] and np.array_equal(kv, outs[0][2])
    # empty context (L = 0)
    cache = fresh_cache(micro, 8)
    lg, _ = vo.forward_tree(micro, cache, 0, toks, parents)
    assert np.all(np.isfinite(lg))


def test_p10_sibling_relabelling_and_padding(micro):
    ids = _ctx(MICRO, 10, seed=16)
    p1, t1 = np.array([-1, 0, 0, 1, 2]), np.array([7, 3, 4, 5, 6], dtype=np.int32)
    p2, t2 = np.array([-1, 0, 0, 2, 1]), np.array([7, 4, 3, 5, 6], dtype=np.int32)     # siblings swapped
    res = []
    for p, t in ((p1, t1), (p2, t2)):
        cache = fresh_cache(micro, 20)
        vo.prefill(micro, cache, 0, ids)
        res.append(vo.verify(micro, cache, 0, t, p, commit=False))
    assert np.array_equal(res[0]["logits"][[0, 1, 2, 3, 4]], res[1]["logits"][[0, 2, 1, 3, 4]])
    assert res[0]["out_tokens"] == res[1]["out_tokens"]
    # extra (padding) nodes appended after the real ones do not change the real nodes' logits
    cache = fresh_cache(micro, 20)
    vo.prefill(micro, cache, 0, ids)
    lg, _ = vo.forward_tree(micro, cache, 0, np.concatenate([t1, [1, 1]]).astype(np.int32), np.concatenate([p1, [0, 5]]))
    assert np.array_equal(lg[:5], res[0]["logits"])


def test_p11_planted_chain_expected_emitted_length():
    """config[3]: chain k=3, each draft equals the greedy token w.p. 0.7 independently:
    E[emitted] = 1 + 0.7 + 0.49 + 0.343 = 2.533."""
    spec = wl.CONFIGS[3]
    from workloads.gen import match_coins
    tot, n = 0, 0
    parents = wl.chain_parents(4)
    for seq in range(4000):
        coins = match_coins(spec, seq, 3)
        greedy = np.array([11, 12, 13, 14], dtype=np.int32)       # argmax at nodes 0..3
        toks = np.array([5] + [greedy[j] if coins[j] < spec.planted_p else 99 for j in range(3)], dtype=np.int32)
        path, out = vo.accept_walk(toks, parents, greedy)
        tot += len(out)
        n += 1
    assert abs(tot / n - 2.533) < 0.04


def test_p11_random_init_logit_scale():
    """logits of the random-init model ~ N(0, (0.02*sqrt(H))^2): sigma ~ 0.32 at H = 256."""
    m = oracle_model(wl.TINY, seed=0)
    cache = fresh_cache(m, 16)
    lg, hid = vo.forward_tree(m, cache, 0, _ctx(wl.TINY, 5, seed=1), wl.chain_parents(5), want_hidden=True)
    assert 0.25 < float(lg.std()) < 0.40
    assert len(hid) == 3 and hid[0].shape == (5, 256)


def test_calibration_static_scales(micro):
    m = oracle_model(MICRO, seed=11, random_gains=True, act_scale_mode=1)
    calib = np.random.default_rng(17).standard_normal((48, MICRO.hidden)).astype(np.float32)
    rec = vo.calibrate(m, calib)
    assert len(rec) == 6 * MICRO.n_layers + 1 and all(v > 0 for v in rec.values())   # 4 activation sites + K, V cache per layer; LM head input
    # with static scales from the very batch it is run on, nothing clips and the forward runs
    cache = fresh_cache(m, 64)
    ids = _ctx(MICRO, 12, seed=18)
    vo.prefill(m, cache, 0, ids)
    r = vo.verify(m, cache, 0, _ctx(MICRO, 4, seed=19), wl.chain_parents(4))
    assert np.all(np.isfinite(r["logits"]))
    assert set(k[0] for k in m.clip_counts) == {"qkv_in", "o_in", "gateup_in", "down_in", "lm_in"}
    # static and dynamic are different models (different scales) but close
    md = oracle_model(MICRO, seed=11, random_gains=True)
    cd = fresh_cache(md, 64)
    vo.prefill(md, cd, 0, ids)
    rd = vo.verify(md, cd, 0, _ctx(MICRO, 4, seed=19), wl.chain_parents(4))
    assert not np.array_equal(rd["logits"], r["logits"])
