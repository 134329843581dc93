"""Seeded generators.  No method arithmetic lives here (see package docstring)."""
import itertools

import numpy as np

# matrix kinds; ids are part of the seed derivation, do not renumber
MATRIX_KINDS = {"embed": 0, "wq": 1, "wk": 2, "wv": 3, "wo": 4, "wgate": 5, "wup": 6,
                "wdown": 7, "lm_head": 8, "d_fc": 9}
_STREAM_WEIGHTS, _STREAM_INPUTS, _STREAM_CALIB = 0, 1, 2


def matrix_shape(shape, kind):
    """(rows = output channels, cols = input channels) of one weight matrix."""
    H, F, V = shape.hidden, shape.ffn, shape.vocab
    return {"embed": (V, H), "wq": (shape.q_dim, H), "wk": (shape.kv_dim, H),
            "wv": (shape.kv_dim, H), "wo": (H, shape.q_dim), "wgate": (F, H), "wup": (F, H),
            "wdown": (H, F), "lm_head": (V, H), "d_fc": (H, 2 * H)}[kind]


def f32_to_bf16_bits(x):
    """fp32 -> bf16 bit pattern (uint16), round-to-nearest-even.  Storage format
    conversion only; inputs here are finite."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    lsb = (u >> np.uint32(16)) & np.uint32(1)
    r = (u + np.uint32(0x7FFF) + lsb) >> np.uint32(16)
    return r.astype(np.uint16)


def bf16_bits_to_f32(b):
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def _rng(seed, stream, *extra):
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([seed, stream, *extra])))


def weight_matrix_bf16(shape, seed, kind, layer=0, device="cpu", std=0.02):
    """One weight matrix as bf16.  device="cpu": numpy uint16 bit patterns [rows, cols].
    device="cuda": a torch.bfloat16 CUDA tensor drawn with a torch CUDA generator (8B shapes;
    the same tensor is handed to the library and, copied to the host, to the oracle).
    The two devices give different bits; within a run both sides read the same ones."""
    rows, cols = matrix_shape(shape, kind)
    k = MATRIX_KINDS[kind]
    if device == "cpu":
        g = _rng(seed, _STREAM_WEIGHTS, k, layer)
        x = g.standard_normal((rows, cols), dtype=np.float32) * np.float32(std)
        return f32_to_bf16_bits(x)
    import torch
    g = torch.Generator(device=device)
    g.manual_seed((seed * 1000003 + k * 1009 + layer) & 0x7FFFFFFF)
    x = torch.empty((rows, cols), dtype=torch.float32, device=device)
    x.normal_(0.0, std, generator=g)
    return x.to(torch.bfloat16)


def gain_vector_bf16(shape, seed=None, which=0, layer=0):
    """RMSNorm gains: 1.0 (config recipe) or, for unit tests, random in [0.5, 1.5)."""
    if seed is None:
        return f32_to_bf16_bits(np.ones(shape.hidden, dtype=np.float32))
    g = _rng(seed, _STREAM_WEIGHTS, 100 + which, layer)
    return f32_to_bf16_bits((0.5 + g.random(shape.hidden)).astype(np.float32))


def chain_parents(n_nodes):
    return np.arange(-1, n_nodes - 1, dtype=np.int32)


_RANK_COST = (6, 16, 23, 28)  # ~ -10 ln(0.55, 0.20, 0.10, 0.06)


def tree_parents(n_nodes, caps):
    """Static draft-tree topology: all child-rank paths under per-depth caps, keep the
    n_nodes-1 cheapest (cost = sum of rank costs; ties by depth then rank path), order nodes by
    (depth, rank path); node 0 = root.  Own generator, not a third party's table."""
    cands = []
    for depth in range(1, len(caps) + 1):
        for path in itertools.product(*[range(c) for c in caps[:depth]]):
            cost = sum(_RANK_COST[r] for r in path)
            cands.append((cost, depth, path))
    cands.sort()
    kept = sorted((c[1], c[2]) for c in cands[:n_nodes - 1])
    index = {(): 0}
    parents = [-1]
    for depth, path in kept:
        index[path] = len(parents)
        parents.append(index[path[:-1]])  # parent always kept: costs are positive
    return np.asarray(parents, dtype=np.int32)


def tree_depths(parents):
    d = np.zeros(len(parents), dtype=np.int32)
    for i in range(1, len(parents)):
        d[i] = d[parents[i]] + 1
    return d


def context_lengths(spec):
    if spec.ctx_len is not None:
        return np.full(spec.batch, spec.ctx_len, dtype=np.int32)
    lo, hi = spec.ctx_range
    return _rng(spec.seed, _STREAM_INPUTS, 0).integers(lo, hi + 1, size=spec.batch).astype(np.int32)


def context_ids(spec, seq, length):
    return _rng(spec.seed, _STREAM_INPUTS, 1, seq).integers(0, spec.model.vocab, size=length).astype(np.int32)


def draft_tokens_uniform(spec, parents, seq):
    """Node tokens: uniform ids; node 0 is the root (last emitted token).  Siblings are
    forced distinct by redrawing (reading A4/A5)."""
    g = _rng(spec.seed, _STREAM_INPUTS, 2, seq)
    T = len(parents)
    tok = g.integers(0, spec.model.vocab, size=T).astype(np.int32)
    for i in range(1, T):
        sib = [tok[j] for j in range(1, i) if parents[j] == parents[i]]
        while tok[i] in sib:
            tok[i] = g.integers(0, spec.model.vocab)
    return tok


def match_coins(spec, seq, n):
    """config[3]: per-position coins; coin < planted_p means 'draft = greedy token'."""
    return _rng(spec.seed, _STREAM_INPUTS, 3, seq).random(n)


def calibration_hidden(spec, n_tokens=None):
    """config[4]: N(0,1) hidden states [calib_tokens, hidden], fp32.  n_tokens overrides the count for configs that state no
    calibration batch (FP8 KV cache scales, DESIGN.md R-kv8: config[4]'s recipe, 512 tokens)."""
    return _rng(spec.seed, _STREAM_CALIB).standard_normal(
        (n_tokens or spec.calib_tokens, spec.model.hidden), dtype=np.float32)
