"""Test-side glue: builds the oracle's model from the seeded generators.  (The CUDA library is
fed the same arrays by tests/gpu_helpers.py; neither side imports the other.)"""
import numpy as np

import workloads as wl
from oracle import verify_oracle as vo

LAYER_KINDS = ("wq", "wk", "wv", "wo", "wgate", "wup", "wdown")


def oracle_model(shape, seed, random_gains=False, act_scale_mode=0, accum="exact", layers=None,
                 with_lm_head=True, device="cpu", weight_fn=None, weight_scale_mode=0):
    """weight_fn(kind, layer) -> uint16 bits overrides the generator (8B shapes: tensors drawn on
    the GPU and copied to the host)."""
    get = weight_fn or (lambda kind, layer: wl.weight_matrix_bf16(shape, seed, kind, layer))
    m = vo.OracleModel(shape, act_scale_mode=act_scale_mode, accum=accum, weight_scale_mode=weight_scale_mode)
    m.set_weight("embed", 0, get("embed", 0))
    for layer in (range(shape.n_layers) if layers is None else layers):
        for kind in LAYER_KINDS:
            m.set_weight(kind, layer, get(kind, layer))
        if random_gains:
            m.set_weight("norm1", layer, wl.gain_vector_bf16(shape, seed, 0, layer))
            m.set_weight("norm2", layer, wl.gain_vector_bf16(shape, seed, 1, layer))
    if with_lm_head:
        m.set_weight("lm_head", 0, get("lm_head", 0))
    if random_gains:
        m.set_weight("normf", 0, wl.gain_vector_bf16(shape, seed, 2, 0))
    return m


def small_shape(**kw):
    """A shape even smaller than config[0] for brute-force pins."""
    base = dict(name="micro", n_layers=2, hidden=64, n_q_heads=4, n_kv_heads=2, head_dim=16,
                ffn=96, vocab=50, rms_eps=1e-5, rope_theta=1e4)
    base.update(kw)
    return wl.ModelShape(**base)


def fresh_cache(model, capacity, page_size=16, page_order=None, n_pages=None):
    n = n_pages or (-(-capacity // page_size) + 2)
    c = vo.OracleKV(model, n, page_size, page_order)
    c.add_seq(0, capacity)
    return c


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-30))
