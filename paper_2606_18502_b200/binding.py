"""Thin ctypes binding of include/eagle_verify.h: same names, argument marshalling only.

Every step of the hot path runs inside libeagle_verify.so; torch is used here for device memory
and streams.  There is no CPU fallback: if the library is missing or a call fails, an exception
is raised.
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libeagle_verify.so")

EV_OK, EV_EINVAL, EV_ENOMEM, EV_ECAPACITY, EV_ECUDA, EV_ESTATE = 0, -1, -2, -3, -4, -5
EV_W = dict(embed=0, wq=1, wk=2, wv=3, wo=4, wgate=5, wup=6, wdown=7, lm_head=8, norm1=9, norm2=10, normf=11, d_fc=12)
EV_SEQ_BAD_TREE, EV_SEQ_BAD_TOKEN, EV_SEQ_OVER_CAPACITY = 1, 2, 4


class EvError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"eagle_verify error {code}: {msg}")
        self.code = code


class ev_config(C.Structure):
    _fields_ = [("n_layers", C.c_int), ("hidden", C.c_int), ("n_q_heads", C.c_int), ("n_kv_heads", C.c_int),
                ("head_dim", C.c_int), ("ffn", C.c_int), ("vocab", C.c_int), ("rms_eps", C.c_float),
                ("rope_theta", C.c_float), ("page_size", C.c_int), ("act_scale_mode", C.c_int),
                ("max_batch", C.c_int), ("max_tree_nodes", C.c_int), ("max_ctx", C.c_int), ("weight_scale_mode", C.c_int),
                ("attn_chunk", C.c_int), ("kv_dtype", C.c_int)]


class ev_verify_in(C.Structure):
    _fields_ = [("n_seqs", C.c_int), ("n_nodes_max", C.c_int), ("dev_seq_slots", C.c_void_p),
                ("dev_tokens", C.c_void_p), ("dev_parents", C.c_void_p), ("dev_n_nodes", C.c_void_p),
                ("commit", C.c_int), ("force_accept_all", C.c_int), ("dev_hidden_override", C.c_void_p),
                ("override_first_only", C.c_int), ("dev_features", C.c_void_p)]


class ev_verify_out(C.Structure):
    _fields_ = [("dev_accept_len", C.c_void_p), ("dev_accept_nodes", C.c_void_p), ("dev_out_tokens", C.c_void_p),
                ("dev_new_ctx_len", C.c_void_p), ("dev_status", C.c_void_p), ("dev_argmax", C.c_void_p),
                ("dev_logits", C.c_void_p), ("dev_hidden", C.c_void_p), ("tap_layer", C.c_int),
                ("dev_tap_xq", C.c_void_p), ("dev_tap_sx", C.c_void_p), ("dev_tap_qkv", C.c_void_p),
                ("dev_tap_attn", C.c_void_p), ("dev_tap_aq", C.c_void_p), ("dev_tap_sa", C.c_void_p),
                ("dev_tap_hmid", C.c_void_p), ("dev_tap_gu", C.c_void_p), ("dev_tap_tq", C.c_void_p),
                ("dev_tap_st", C.c_void_p), ("dev_final_hidden", C.c_void_p), ("dev_topk", C.c_void_p), ("topk", C.c_int)]


class ev_engine_config(C.Structure):
    _fields_ = [("max_batch", C.c_int), ("n_nodes", C.c_int), ("host_parents", C.c_void_p)]


class ev_draft_args(C.Structure):
    _fields_ = [("n_seqs", C.c_int), ("n_nodes", C.c_int), ("dev_seq_slots", C.c_void_p), ("host_parents", C.c_void_p),
                ("dev_root_tokens", C.c_void_p), ("dev_root_feats", C.c_void_p), ("dev_tokens", C.c_void_p),
                ("dev_parents", C.c_void_p)]


# every symbol include/eagle_verify.h declares: name -> (restype, argtypes)
_P = C.c_void_p
SIGNATURES = {
    "ev_model_create": (C.c_int, [C.POINTER(ev_config), C.POINTER(_P)]),
    "ev_model_set_weight": (C.c_int, [_P, C.c_int, C.c_int, _P, C.c_long, C.c_long, _P]),
    "ev_model_get_quantized": (C.c_int, [_P, C.c_int, C.c_int, _P, _P, C.c_long, C.c_long, _P]),
    "ev_model_calibrate": (C.c_int, [_P, _P, C.c_int, _P, _P]),
    "ev_model_get_static_scales": (C.c_int, [_P, _P]),
    "ev_model_set_static_scales": (C.c_int, [_P, _P]),
    "ev_model_get_kv_scales": (C.c_int, [_P, _P]),
    "ev_model_set_kv_scales": (C.c_int, [_P, _P]),
    "ev_model_get_clip_counts": (C.c_int, [_P, _P, C.c_int]),
    "ev_model_destroy": (C.c_int, [_P]),
    "ev_cache_create": (C.c_int, [_P, C.c_long, C.c_int, C.POINTER(_P)]),
    "ev_cache_add_seq": (C.c_int, [_P, C.c_int, _P, C.POINTER(C.c_int)]),
    "ev_cache_free_seq": (C.c_int, [_P, C.c_int]),
    "ev_cache_prefill": (C.c_int, [_P, _P, C.c_int, _P, _P, _P, _P]),
    "ev_cache_export_seq": (C.c_int, [_P, C.c_int, C.c_int, C.c_int, C.c_int, _P, _P]),
    "ev_cache_import_seq": (C.c_int, [_P, C.c_int, C.c_int, C.c_int, C.c_int, _P, C.c_int, _P]),
    "ev_cache_set_len": (C.c_int, [_P, C.c_int, C.c_int, _P]),
    "ev_cache_set_lens": (C.c_int, [_P, C.c_int, _P, _P, _P]),
    "ev_cache_get_len": (C.c_int, [_P, C.c_int, C.POINTER(C.c_int), _P]),
    "ev_cache_destroy": (C.c_int, [_P]),
    "ev_verify": (C.c_int, [_P, _P, C.POINTER(ev_verify_in), C.POINTER(ev_verify_out), _P]),
    "ev_verify_host": (C.c_int, [_P, _P, C.c_int, C.c_int, _P, _P, _P, _P, C.c_int, _P, _P, _P, _P, _P, _P]),
    "ev_profile_enable": (C.c_int, [_P, C.c_int]),
    "ev_profile_read": (C.c_int, [_P, _P, _P, C.c_int]),
    "ev_profile_trace": (C.c_int, [_P, _P, C.c_int, _P]),
    "ev_op_linear": (C.c_int, [_P, C.c_int, C.c_int, _P, _P, C.c_int, _P, _P]),
    "ev_op_linear_static": (C.c_int, [_P, C.c_int, C.c_int, _P, _P, C.c_int, _P, _P]),
    "ev_op_quantize_rows": (C.c_int, [_P, _P, C.c_int, C.c_int, C.c_float, _P, _P, _P]),
    "ev_last_error": (C.c_char_p, []),
    "ev_model_share_head": (C.c_int, [_P, _P]),
    "ev_draft_tree": (C.c_int, [_P, _P, C.POINTER(ev_draft_args), _P]),
    "ev_draft_extend": (C.c_int, [_P, _P, C.c_int, C.c_int, _P, _P, _P, _P, _P]),
    "ev_gather_accepted": (C.c_int, [C.c_int, C.c_int, C.c_int, _P, _P, _P, _P, _P, _P, _P, _P, _P, _P, _P]),
    "ev_engine_create": (C.c_int, [_P, _P, _P, _P, C.POINTER(ev_engine_config), C.POINTER(_P)]),
    "ev_engine_submit": (C.c_int, [_P, _P, C.c_int, C.c_int, C.POINTER(C.c_int)]),
    "ev_engine_step": (C.c_int, [_P, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int), _P]),
    "ev_engine_poll": (C.c_int, [_P, C.c_int, _P, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int)]),
    "ev_engine_destroy": (C.c_int, [_P]),
    "ev_launch_count": (C.c_long, [C.c_int]),
    "ev_capture_count": (C.c_long, [C.c_int]),
    "ev_version": (C.c_int, []),
}

_lib = None


def load_library():
    """Loads libeagle_verify.so (built by paper_2606_18502_b200.build).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise EvError(EV_ESTATE, f"{LIB_PATH} not built; run `python -m paper_2606_18502_b200.build` "
                                     "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def _check(rc):
    if rc != EV_OK:
        raise EvError(rc, load_library().ev_last_error().decode())


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def ev_last_error():
    return load_library().ev_last_error().decode()


def ev_capture_count(reset=False):
    return int(load_library().ev_capture_count(1 if reset else 0))


def ev_launch_count(reset=False):
    return load_library().ev_launch_count(1 if reset else 0)


class Model:
    """ev_model handle."""

    def __init__(self, shape, max_batch, max_tree_nodes, max_ctx, page_size=16, act_scale_mode=0, weight_scale_mode=0,
                 attn_chunk=0, kv_dtype=0):
        self.lib = load_library()
        self.cfg = ev_config(shape.n_layers, shape.hidden, shape.n_q_heads, shape.n_kv_heads, shape.head_dim,
                             shape.ffn, shape.vocab, shape.rms_eps, shape.rope_theta, page_size, act_scale_mode,
                             max_batch, max_tree_nodes, max_ctx, weight_scale_mode, attn_chunk, kv_dtype)
        self.shape = shape
        h = C.c_void_p()
        _check(self.lib.ev_model_create(C.byref(self.cfg), C.byref(h)))
        self.h = h

    def ev_model_set_weight(self, kind, layer, w_bf16):
        """w_bf16: torch.bfloat16 CUDA tensor [rows, cols] (gains: [hidden])."""
        import torch
        assert w_bf16.is_cuda and w_bf16.dtype == torch.bfloat16 and w_bf16.is_contiguous()
        rows, cols = (1, w_bf16.shape[0]) if w_bf16.dim() == 1 else w_bf16.shape
        _check(self.lib.ev_model_set_weight(self.h, EV_W[kind] if isinstance(kind, str) else kind, layer, _ptr(w_bf16),
                                            rows, cols, _stream()))

    def ev_model_get_quantized(self, kind, layer):
        """-> (codes uint8 [rows, cols] row-major, scales float32 [rows]) as torch CUDA tensors."""
        import torch
        sh, H, F = self.shape, self.shape.hidden, self.shape.ffn
        rows, cols = {"wq": (sh.q_dim, H), "wk": (sh.kv_dim, H), "wv": (sh.kv_dim, H), "wo": (H, sh.q_dim), "wgate": (F, H),
                      "wup": (F, H), "wdown": (H, F), "lm_head": (sh.vocab, H)}[kind]
        out_c = torch.empty((rows, cols), dtype=torch.uint8, device="cuda")
        out_s = torch.empty((rows,), dtype=torch.float32, device="cuda")
        _check(self.lib.ev_model_get_quantized(self.h, EV_W[kind], layer, _ptr(out_c), _ptr(out_s), rows, cols, _stream()))
        return out_c, out_s

    def ev_model_calibrate(self, hidden_f32, want_layer_inputs=False):
        import torch
        assert hidden_f32.is_cuda and hidden_f32.dtype == torch.float32 and hidden_f32.is_contiguous()
        n = hidden_f32.shape[0]
        taps = torch.empty((self.cfg.n_layers + 1, n, self.cfg.hidden), dtype=torch.float32, device="cuda") \
            if want_layer_inputs else None
        _check(self.lib.ev_model_calibrate(self.h, _ptr(hidden_f32), n, _ptr(taps), _stream()))
        return taps

    def ev_model_get_static_scales(self):
        import numpy as np
        out = np.empty(4 * self.cfg.n_layers + 1, dtype=np.float32)
        _check(self.lib.ev_model_get_static_scales(self.h, out.ctypes.data_as(C.c_void_p)))
        return out

    def ev_model_get_kv_scales(self):
        import numpy as np
        out = np.zeros(2 * self.cfg.n_layers, dtype=np.float32)
        _check(self.lib.ev_model_get_kv_scales(self.h, out.ctypes.data_as(C.c_void_p)))
        return out

    def ev_model_set_kv_scales(self, scales):
        import numpy as np
        s = np.ascontiguousarray(scales, dtype=np.float32)
        assert s.shape == (2 * self.cfg.n_layers,)
        _check(self.lib.ev_model_set_kv_scales(self.h, s.ctypes.data_as(C.c_void_p)))

    def ev_model_get_clip_counts(self, reset=False):
        import numpy as np
        out = np.zeros(4 * self.cfg.n_layers + 1, dtype=np.uint64)
        _check(self.lib.ev_model_get_clip_counts(self.h, out.ctypes.data_as(C.c_void_p), 1 if reset else 0))
        return out

    def ev_model_set_static_scales(self, scales):
        import numpy as np
        s = np.ascontiguousarray(scales, dtype=np.float32)
        assert s.shape == (4 * self.cfg.n_layers + 1,)
        _check(self.lib.ev_model_set_static_scales(self.h, s.ctypes.data_as(C.c_void_p)))

    def ev_op_linear(self, kind, layer, codes_x, sx):
        import torch
        M = codes_x.shape[0]
        n_out = {"wq": self.shape.q_dim + 2 * self.shape.kv_dim, "wo": self.shape.hidden, "wgate": 2 * self.shape.ffn,
                 "wdown": self.shape.hidden, "lm_head": self.shape.vocab}[kind]
        out = torch.empty((M, n_out), dtype=torch.float32, device="cuda")
        _check(self.lib.ev_op_linear(self.h, EV_W[kind], layer, _ptr(codes_x.contiguous()), _ptr(sx.contiguous()), M,
                                     _ptr(out), _stream()))
        return out

    def ev_op_linear_static(self, kind, layer, codes_x, sx, out):
        """no-allocation variant: the caller passes the output tensor [M, N] too (include/eagle_verify.h)"""
        _check(self.lib.ev_op_linear_static(self.h, EV_W[kind], layer, _ptr(codes_x), _ptr(sx), codes_x.shape[0], _ptr(out), _stream()))
        return out

    def ev_op_quantize_rows(self, x, static_scale=0.0):
        import torch
        M, K = x.shape
        codes = torch.empty((M, K), dtype=torch.uint8, device="cuda")
        sx = torch.empty((M,), dtype=torch.float32, device="cuda")
        _check(self.lib.ev_op_quantize_rows(self.h, _ptr(x.contiguous()), M, K, float(static_scale), _ptr(codes), _ptr(sx),
                                            _stream()))
        return codes, sx

    PROFILE_CLASSES = ("gemm_qkv", "gemm_o", "gemm_gateup", "gemm_down", "gemm_lm_head", "tree_attention", "attn_merge_quant",
                       "rmsnorm_quant", "rope_kvwrite", "swiglu_quant", "other")

    def ev_profile_enable(self, on=True):
        """True / 1: per-class CUDA-event timing; 2: in-graph step trace (ev_profile_trace); False / 0: off"""
        _check(self.lib.ev_profile_enable(self.h, int(on)))

    def ev_profile_read(self):
        """-> {class: (total_ms, launches)} since enable / the last read."""
        n = len(self.PROFILE_CLASSES)
        ms = (C.c_double * n)()
        cnt = (C.c_long * n)()
        _check(self.lib.ev_profile_read(self.h, ms, cnt, n))
        return {k: (ms[i], cnt[i]) for i, k in enumerate(self.PROFILE_CLASSES)}

    def ev_profile_trace(self, max_entries=1024):
        """-> list of (t_enter, t_past_wait_first, t_exit, t_past_wait_last, 4 phase marks) in ns per traced launch of the
        last verify step (after ev_profile_enable(2))."""
        buf = (C.c_ulonglong * (8 * max_entries))()
        n = C.c_int(0)
        _check(self.lib.ev_profile_trace(self.h, buf, max_entries, C.byref(n)))
        return [tuple(buf[8 * i + j] for j in range(8)) for i in range(n.value)]

    def ev_model_destroy(self):
        if self.h:
            self.lib.ev_model_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.ev_model_destroy()
        except Exception:
            pass


class Cache:
    """ev_cache handle."""

    def __init__(self, model, n_pages, max_seqs):
        self.lib, self.model = model.lib, model
        h = C.c_void_p()
        _check(self.lib.ev_cache_create(model.h, n_pages, max_seqs, C.byref(h)))
        self.h = h

    def ev_cache_add_seq(self, capacity_tokens, pages=None):
        slot = C.c_int(-1)
        arr = None
        if pages is not None:
            arr = (C.c_int * len(pages))(*pages)
        _check(self.lib.ev_cache_add_seq(self.h, capacity_tokens, arr, C.byref(slot)))
        return slot.value

    def ev_cache_free_seq(self, slot):
        _check(self.lib.ev_cache_free_seq(self.h, slot))

    def ev_cache_prefill(self, slots, ids_list):
        """ids_list: one host int32 array per sequence."""
        import numpy as np
        n = len(slots)
        sl = (C.c_int * n)(*slots)
        lens = (C.c_int * n)(*[len(x) for x in ids_list])
        cat = np.ascontiguousarray(np.concatenate([np.asarray(x, dtype=np.int32) for x in ids_list]), dtype=np.int32)
        _check(self.lib.ev_cache_prefill(self.model.h, self.h, n, sl, cat.ctypes.data_as(C.c_void_p), lens, _stream()))

    def _dense_shape(self, lb, le, n_tokens):
        c = self.model.cfg
        return (le - lb, 2, c.n_kv_heads, n_tokens, c.head_dim)

    def ev_cache_export_seq(self, slot, layer_begin, layer_end, n_tokens):
        import torch
        dt = torch.uint8 if self.model.cfg.kv_dtype == 1 else torch.bfloat16      # kv_dtype 1: the E4M3 codes themselves
        out = torch.empty(self._dense_shape(layer_begin, layer_end, n_tokens), dtype=dt, device="cuda")
        _check(self.lib.ev_cache_export_seq(self.h, slot, layer_begin, layer_end, n_tokens, _ptr(out), _stream()))
        return out

    def ev_cache_import_seq(self, slot, layer_begin, layer_end, dense_bf16, set_len=True):
        n_tokens = dense_bf16.shape[3]
        assert tuple(dense_bf16.shape) == self._dense_shape(layer_begin, layer_end, n_tokens) and dense_bf16.is_contiguous()
        _check(self.lib.ev_cache_import_seq(self.h, slot, layer_begin, layer_end, n_tokens, _ptr(dense_bf16),
                                            1 if set_len else 0, _stream()))

    def ev_cache_set_len(self, slot, n):
        _check(self.lib.ev_cache_set_len(self.h, slot, n, _stream()))

    def ev_cache_set_lens(self, slots, lens):
        n = len(slots)
        _check(self.lib.ev_cache_set_lens(self.h, n, (C.c_int * n)(*slots), (C.c_int * n)(*lens), _stream()))

    def ev_cache_get_len(self, slot):
        v = C.c_int(0)
        _check(self.lib.ev_cache_get_len(self.h, slot, C.byref(v), _stream()))
        return v.value

    def ev_cache_destroy(self):
        if self.h:
            self.lib.ev_cache_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.ev_cache_destroy()
        except Exception:
            pass


class VerifyBuffers:
    """Device buffers of one ev_verify call, allocated once and reused (no allocation per step)."""

    def __init__(self, model, B, T, want_logits=False, want_hidden=False, want_argmax=True, tap_layer=-1,
                 want_final_hidden=False, topk=0):
        import torch
        c = model.cfg
        i32 = dict(dtype=torch.int32, device="cuda")
        self.B, self.T, self.model = B, T, model
        self.seq_slots = torch.zeros(B, **i32)
        self.tokens = torch.zeros((B, T), **i32)
        self.parents = torch.zeros((B, T), **i32)
        self.n_nodes = torch.full((B,), T, **i32)
        self.accept_len = torch.zeros(B, **i32)
        self.accept_nodes = torch.zeros((B, T), **i32)
        self.out_tokens = torch.zeros((B, T), **i32)
        self.new_ctx_len = torch.zeros(B, **i32)
        self.status = torch.zeros(B, **i32)
        self.argmax = torch.zeros((B, T), **i32) if want_argmax else None
        self.logits = torch.empty((B * T, c.vocab), dtype=torch.float32, device="cuda") if want_logits else None
        self.hidden = torch.empty((c.n_layers + 1, B * T, c.hidden), dtype=torch.float32, device="cuda") if want_hidden else None
        self.hidden_override = None
        self.features = None           # draft models: [B*T, hidden] fp32 predecessor features
        self.final_hidden = torch.empty((B * T, c.hidden), dtype=torch.float32, device="cuda") if want_final_hidden else None
        self.topk = torch.zeros((B * T, topk), **i32) if topk else None
        self.tap_layer = tap_layer
        self.taps = {}
        if tap_layer >= 0:
            M, H, F = B * T, c.hidden, c.ffn
            qd = c.n_q_heads * c.head_dim
            qkvd = qd + 2 * c.n_kv_heads * c.head_dim
            f32 = dict(dtype=torch.float32, device="cuda")
            u8 = dict(dtype=torch.uint8, device="cuda")
            self.taps = dict(xq=torch.empty((M, H), **u8), sx=torch.empty(M, **f32), qkv=torch.empty((M, qkvd), **f32),
                             attn=torch.empty((M, qd), **f32), aq=torch.empty((M, qd), **u8), sa=torch.empty(M, **f32),
                             hmid=torch.empty((M, H), **f32), gu=torch.empty((M, 2 * F), **f32),
                             tq=torch.empty((M, F), **u8), st=torch.empty(M, **f32))

    def set_inputs(self, seq_slots, tokens, parents, n_nodes=None):
        import numpy as np
        import torch
        self.seq_slots.copy_(torch.as_tensor(np.asarray(seq_slots, dtype=np.int32)))
        self.tokens.copy_(torch.as_tensor(np.asarray(tokens, dtype=np.int32).reshape(self.B, self.T)))
        self.parents.copy_(torch.as_tensor(np.asarray(parents, dtype=np.int32).reshape(self.B, self.T)))
        if n_nodes is not None:
            self.n_nodes.copy_(torch.as_tensor(np.asarray(n_nodes, dtype=np.int32)))


def ev_verify(model, cache, buf, commit=True, use_n_nodes=True, override_first_only=False):
    """One verify step on the current torch CUDA stream; asynchronous (outputs valid after a sync)."""
    vin = ev_verify_in(buf.B, buf.T, buf.seq_slots.data_ptr(), buf.tokens.data_ptr(), buf.parents.data_ptr(),
                       buf.n_nodes.data_ptr() if use_n_nodes else None, 1 if commit else 0, 0,
                       buf.hidden_override.data_ptr() if buf.hidden_override is not None else None,
                       1 if override_first_only else 0, buf.features.data_ptr() if buf.features is not None else None)
    t = buf.taps
    g = lambda k: t[k].data_ptr() if k in t else None  # noqa: E731
    vout = ev_verify_out(buf.accept_len.data_ptr(), buf.accept_nodes.data_ptr(), buf.out_tokens.data_ptr(),
                         buf.new_ctx_len.data_ptr(), buf.status.data_ptr(),
                         buf.argmax.data_ptr() if buf.argmax is not None else None,
                         buf.logits.data_ptr() if buf.logits is not None else None,
                         buf.hidden.data_ptr() if buf.hidden is not None else None, buf.tap_layer,
                         g("xq"), g("sx"), g("qkv"), g("attn"), g("aq"), g("sa"), g("hmid"), g("gu"), g("tq"), g("st"),
                         buf.final_hidden.data_ptr() if buf.final_hidden is not None else None,
                         buf.topk.data_ptr() if buf.topk is not None else None, buf.topk.shape[1] if buf.topk is not None else 0)
    _check(model.lib.ev_verify(model.h, cache.h, C.byref(vin), C.byref(vout), _stream()))


def ev_verify_host(model, cache, host, commit=True):
    """End-to-end step with HOST (pinned) int32 tensors: host = dict(seq_slots[B], tokens[B,T], parents[B,T],
    n_nodes[B] or None, accept_len[B], accept_nodes[B,T], out_tokens[B,T], new_ctx_len[B], status[B]).
    Copies in, verifies, copies out, synchronises."""
    B, T = host["tokens"].shape
    p = lambda k: C.c_void_p(host[k].data_ptr()) if host.get(k) is not None else None  # noqa: E731
    _check(model.lib.ev_verify_host(model.h, cache.h, B, T, p("seq_slots"), p("tokens"), p("parents"), p("n_nodes"),
                                    1 if commit else 0, p("accept_len"), p("accept_nodes"), p("out_tokens"),
                                    p("new_ctx_len"), p("status"), _stream()))


# ---- draft side (include/eagle_verify.h "draft side") ------------------------------------------------------------

def ev_model_share_head(drafter, target):
    _check(drafter.lib.ev_model_share_head(drafter.h, target.h))
    drafter._target = target          # the target must outlive the drafter


def ev_draft_tree(drafter, dcache, seq_slots, parents, root_tokens, root_feats, tokens_out, parents_out):
    """seq_slots [B] int32 cuda, parents: host int32 numpy [T], root_tokens [B] int32 cuda, root_feats [B, H] f32 cuda,
    tokens_out / parents_out [B, T] int32 cuda (filled)."""
    import numpy as np
    par = np.ascontiguousarray(parents, dtype=np.int32)
    B, T = tokens_out.shape
    a = ev_draft_args(B, T, seq_slots.data_ptr(), par.ctypes.data_as(C.c_void_p), root_tokens.data_ptr(), root_feats.data_ptr(),
                      tokens_out.data_ptr(), parents_out.data_ptr())
    _check(drafter.lib.ev_draft_tree(drafter.h, dcache.h, C.byref(a), _stream()))


def ev_draft_extend(drafter, dcache, seq_slots, tokens, feats, n):
    """tokens [B, T] int32, feats [B, T, H] f32, n [B] int32, seq_slots [B] int32: all cuda."""
    B, T = tokens.shape
    _check(drafter.lib.ev_draft_extend(drafter.h, dcache.h, B, T, seq_slots.data_ptr(), tokens.data_ptr(), feats.data_ptr(), n.data_ptr(), _stream()))


def ev_gather_accepted(tokens, accept_len, accept_nodes, out_tokens, feat, carry, ext_tokens, ext_feats, ext_n, next_root):
    B, T = tokens.shape
    H = carry.shape[1]
    _check(load_library().ev_gather_accepted(B, T, H, tokens.data_ptr(), accept_len.data_ptr(), accept_nodes.data_ptr(), out_tokens.data_ptr(),
                                             feat.data_ptr(), carry.data_ptr(), ext_tokens.data_ptr(), ext_feats.data_ptr(), ext_n.data_ptr(),
                                             next_root.data_ptr(), _stream()))


class Engine:
    """ev_engine handle: continuous batching around verify (include/eagle_verify.h "serving shell")."""

    def __init__(self, target, tcache, drafter=None, dcache=None, max_batch=1, parents=None):
        import numpy as np
        self.lib = load_library()
        self._keep = (target, tcache, drafter, dcache)
        par = np.ascontiguousarray(parents if parents is not None else [-1], dtype=np.int32)
        cfg = ev_engine_config(max_batch, len(par), par.ctypes.data_as(C.c_void_p))
        h = C.c_void_p()
        _check(self.lib.ev_engine_create(target.h, tcache.h, drafter.h if drafter else None, dcache.h if dcache else None, C.byref(cfg), C.byref(h)))
        self.h = h

    def ev_engine_submit(self, prompt, max_new_tokens):
        import numpy as np
        p = np.ascontiguousarray(prompt, dtype=np.int32)
        rid = C.c_int(-1)
        _check(self.lib.ev_engine_submit(self.h, p.ctypes.data_as(C.c_void_p), len(p), max_new_tokens, C.byref(rid)))
        return rid.value

    def ev_engine_step(self):
        a, f, w = C.c_int(0), C.c_int(0), C.c_int(0)
        _check(self.lib.ev_engine_step(self.h, C.byref(a), C.byref(f), C.byref(w), _stream()))
        return a.value, f.value, w.value

    def ev_engine_poll(self, rid, cap=4096):
        import numpy as np
        out = np.zeros(cap, dtype=np.int32)
        n, fin = C.c_int(0), C.c_int(0)
        _check(self.lib.ev_engine_poll(self.h, rid, out.ctypes.data_as(C.c_void_p), cap, C.byref(n), C.byref(fin)))
        return out[:min(n.value, cap)].copy(), bool(fin.value)

    def ev_engine_destroy(self):
        if self.h:
            self.lib.ev_engine_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.ev_engine_destroy()
        except Exception:
            pass
