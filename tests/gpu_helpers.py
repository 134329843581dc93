"""GPU-side test glue: feeds the CUDA library the same seeded arrays the oracle gets."""
import numpy as np
import torch

import workloads as wl
import paper_2606_18502_b200 as ev
from helpers import LAYER_KINDS


def bits_to_bf16_cuda(bits_u16):
    return torch.from_numpy(np.ascontiguousarray(bits_u16).view(np.int16)).cuda().view(torch.bfloat16)


def bf16_cuda_to_bits(t):
    return t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def gpu_model(shape, seed, max_batch, max_tree_nodes, max_ctx, random_gains=False, act_scale_mode=0,
              page_size=16, device_weights=False, keep=None, weight_scale_mode=0, kv_dtype=0, attn_chunk=0):
    """device_weights=True draws the matrices on the GPU (8B shapes); `keep` (dict) then receives
    host copies (uint16 bits) of the (kind, layer) pairs listed in keep['want'] for the oracle."""
    m = ev.Model(shape, max_batch, max_tree_nodes, max_ctx, page_size=page_size, act_scale_mode=act_scale_mode,
                 weight_scale_mode=weight_scale_mode, kv_dtype=kv_dtype, attn_chunk=attn_chunk)

    def put(kind, layer):
        if device_weights:
            w = wl.weight_matrix_bf16(shape, seed, kind, layer, device="cuda")
            if keep is not None and (kind, layer) in keep.get("want", ()):
                keep[(kind, layer)] = bf16_cuda_to_bits(w)
        else:
            w = bits_to_bf16_cuda(wl.weight_matrix_bf16(shape, seed, kind, layer))
        m.ev_model_set_weight(kind, layer, w)

    put("embed", 0)
    for layer in range(shape.n_layers):
        for kind in LAYER_KINDS:
            put(kind, layer)
        if random_gains:
            m.ev_model_set_weight("norm1", layer, bits_to_bf16_cuda(wl.gain_vector_bf16(shape, seed, 0, layer)))
            m.ev_model_set_weight("norm2", layer, bits_to_bf16_cuda(wl.gain_vector_bf16(shape, seed, 1, layer)))
    put("lm_head", 0)
    if random_gains:
        m.ev_model_set_weight("normf", 0, bits_to_bf16_cuda(wl.gain_vector_bf16(shape, seed, 2, 0)))
    torch.cuda.synchronize()
    return m


def import_oracle_kv(cache, slot, ocache, oseq, n_tokens, n_layers):
    dense = np.stack([ocache.export_dense(l, oseq, n_tokens) for l in range(n_layers)])
    cache.ev_cache_import_seq(slot, 0, n_layers, bits_to_bf16_cuda(dense), set_len=True)


def export_kv_bits(cache, slot, layer_begin, layer_end, n_tokens):
    return bf16_cuda_to_bits(cache.ev_cache_export_seq(slot, layer_begin, layer_end, n_tokens))


def run_verify(model, cache, slots, tokens, parents, n_nodes=None, commit=False, want_logits=True,
               want_hidden=True, tap_layer=-1, hidden_override=None, buf=None):
    tokens = np.asarray(tokens, dtype=np.int32)
    B, T = tokens.shape
    buf = buf or ev.VerifyBuffers(model, B, T, want_logits=want_logits, want_hidden=want_hidden, tap_layer=tap_layer)
    buf.set_inputs(slots, tokens, parents, n_nodes)
    if hidden_override is not None:
        buf.hidden_override = torch.from_numpy(np.ascontiguousarray(hidden_override, dtype=np.float32)).cuda()
    ev.ev_verify(model, cache, buf, commit=commit)
    torch.cuda.synchronize()
    return buf
