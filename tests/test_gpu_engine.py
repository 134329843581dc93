"""Serving shell (PAPER.md:337 continuous batching): requests with different prompt lengths and budgets
are submitted over time, join and leave the running batch between steps, and every request's tokens equal its own plain
greedy decode on the GPU - whatever the batch composition was (the path is batch-invariant) and whether the steps were plain
decoding or draft-tree speculation (losslessness)."""
import numpy as np
import pytest

import workloads as wl
from helpers import LAYER_KINDS

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

SHAPE, SEED = wl.TINY, 0
DSHAPE = wl.ModelShape("tiny_drafter", 1, SHAPE.hidden, SHAPE.n_q_heads, SHAPE.n_kv_heads, SHAPE.head_dim, SHAPE.ffn, SHAPE.vocab,
                       SHAPE.rms_eps, SHAPE.rope_theta)


def _greedy_reference(ev, tg, prompt, n_new):
    from gpu_helpers import run_verify
    cache = ev.Cache(tg, 40, 1)
    slot = cache.ev_cache_add_seq(len(prompt) + n_new + 8)
    cache.ev_cache_prefill([slot], [prompt[:-1]])
    tok, out = np.array([prompt[-1]], dtype=np.int32), []
    for _ in range(n_new):
        b = run_verify(tg, cache, [slot], tok[:, None], np.full((1, 1), -1, np.int32), commit=True, want_logits=False, want_hidden=False)
        tok = b.out_tokens.cpu().numpy()[:, 0].astype(np.int32)
        out.append(int(tok[0]))
    return out


@pytest.mark.parametrize("speculate", [False, True])
def test_continuous_batching_is_exact_per_request(speculate):
    import paper_2606_18502_b200 as ev
    from gpu_helpers import gpu_model, bits_to_bf16_cuda
    tg = gpu_model(SHAPE, SEED, max_batch=4, max_tree_nodes=64, max_ctx=512)
    tcache = ev.Cache(tg, 60, 8)            # few pages: admission has to wait for finished requests to free theirs
    dg = dcache = None
    parents = None
    if speculate:
        dg = ev.Model(DSHAPE, 4, 64, 512)
        for k in LAYER_KINDS:
            dg.ev_model_set_weight(k, 0, bits_to_bf16_cuda(wl.weight_matrix_bf16(SHAPE, SEED, k, SHAPE.n_layers)))
        dg.ev_model_set_weight("d_fc", 0, bits_to_bf16_cuda(wl.weight_matrix_bf16(SHAPE, SEED, "d_fc", 0)))
        ev.ev_model_share_head(dg, tg)
        dcache = ev.Cache(dg, 60, 8)
        parents = wl.tree_parents(10, (3, 2, 1))
    eng = ev.Engine(tg, tcache, dg, dcache, max_batch=3, parents=parents)
    rng = np.random.default_rng(3)
    reqs = []
    plan = [(70, 9), (12, 20), (130, 5), (33, 14), (5, 30), (90, 11), (2, 7)]     # (prompt tokens, new tokens); 130 > one prefill chunk
    arrivals = {0: [0, 1], 2: [2, 3], 3: [4], 9: [5, 6]}                           # step -> requests submitted before it
    steps, max_active, waited = 0, 0, 0
    while True:
        for i in arrivals.get(steps, []):
            n_p, n_new = plan[i]
            prompt = rng.integers(0, SHAPE.vocab, size=n_p).astype(np.int32)
            reqs.append((eng.ev_engine_submit(prompt, n_new), prompt, n_new))
        a, f, w = eng.ev_engine_step()
        max_active, waited = max(max_active, a), max(waited, w)
        steps += 1
        assert steps < 200
        if steps > max(arrivals) and a == 0 and w == 0:
            break
    assert max_active == 3 and waited >= 1          # the batch was full and someone queued
    for rid, prompt, n_new in reqs:
        toks, fin = eng.ev_engine_poll(rid)
        assert fin and len(toks) == n_new
        assert toks.tolist() == _greedy_reference(ev, tg, prompt, n_new), rid
    # every page came back
    s1, s2 = tcache.ev_cache_add_seq(30 * 16), tcache.ev_cache_add_seq(30 * 16)      # 60 pages in all
    tcache.ev_cache_free_seq(s1)
    tcache.ev_cache_free_seq(s2)
