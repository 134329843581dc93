"""Generators: topology pins (tests/golden/tree_parents.txt) and byte/flop constants of SURVEY 8."""
import os

import numpy as np

import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold_trees():
    out = {}
    for line in open(os.path.join(GOLD, "tree_parents.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        out[k] = np.array(v, dtype=np.int32)
    return out


def test_tree_topologies_match_survey():
    g = _gold_trees()
    p60 = wl.tree_parents(60, (4, 3, 2, 2, 1, 1))
    p26 = wl.tree_parents(26, (4, 3, 2, 2, 1))
    assert np.array_equal(p60, g["T60"]) and np.array_equal(p26, g["T26"])
    d60, d26 = wl.tree_depths(p60), wl.tree_depths(p26)
    assert np.bincount(d60).tolist() == [1, 4, 11, 17, 14, 8, 5] and int((d60 + 1).sum()) == 263
    assert np.bincount(d26).tolist() == [1, 4, 7, 8, 5, 1] and int((d26 + 1).sum()) == 93
    assert all(p60[i] < i for i in range(1, 60))


def test_model_constants():
    m = wl.LLAMA8B
    assert m.weight_bytes_fp8() == 7_504_658_432          # SURVEY 8 "total 7,504,658,432 B"
    assert m.kv_bytes_per_token() == 131_072
    assert m.attn_flops_per_token_pos() == 524_288
    assert wl.TINY.weight_bytes_fp8() == 1_712_128
    assert wl.TINY.kv_bytes_per_token() == 1024


def test_bf16_roundtrip_and_determinism():
    w1 = wl.weight_matrix_bf16(wl.TINY, 0, "wq", 1)
    w2 = wl.weight_matrix_bf16(wl.TINY, 0, "wq", 1)
    assert w1.dtype == np.uint16 and np.array_equal(w1, w2)
    assert not np.array_equal(w1, wl.weight_matrix_bf16(wl.TINY, 0, "wq", 0))
    f = wl.bf16_bits_to_f32(w1)
    assert np.array_equal(wl.f32_to_bf16_bits(f), w1)
    assert abs(float(f.std()) - 0.02) < 1e-3
    # RNE: 1 + 2^-8 is a tie between 1.0 and 1+2^-7 -> even (1.0); 1 + 3*2^-8 -> 1 + 2^-6
    t = np.array([1 + 2.0 ** -8, 1 + 3 * 2.0 ** -8], dtype=np.float32)
    assert wl.bf16_bits_to_f32(wl.f32_to_bf16_bits(t)).tolist() == [1.0, 1 + 2.0 ** -6]


def test_draft_tokens_siblings_distinct():
    spec = wl.CONFIGS[2]
    p = wl.tree_parents(spec.n_nodes, spec.tree_caps)
    tok = wl.draft_tokens_uniform(spec, p, 3)
    for i in range(1, len(p)):
        for j in range(1, i):
            if p[i] == p[j]:
                assert tok[i] != tok[j]
    L = wl.context_lengths(wl.CONFIGS[3])
    assert L.min() >= 1024 and L.max() <= 8192 and len(L) == 64
