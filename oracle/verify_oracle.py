"""ORACLE (test infrastructure, not product code): the FP8 EAGLE tree-verification step on the CPU.

A plain, slow, by-the-definition numpy implementation of what the hot path computes:
the target model's forward pass over all nodes of a draft-token tree against a paged KV
cache, with FP8 (E4M3) W8A8 linear layers, followed by greedy acceptance and the KV append.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import it; it shares no code with paper_2606_18502_b200/ and imports nothing from it.

What the paper fixes (PAPER.md = /root/reference/PAPER.md):
  * PAPER.md:92 (section 3.1): speculative decoding verifies draft tokens in parallel with the
    target model "while guaranteeing to preserve accuracy" -> greedy acceptance is lossless.
  * PAPER.md:98 (section 3.2): "FP8 (E4M3) weight-and-activation quantization (W8A8) ...
    min-max ... post-training quantization"; static scales come from calibration data.
  * PAPER.md:361 (App. E): a tree of candidate continuations is "verified in a single forward
    pass of the target model via tree attention"; greedy drafting = "a single candidate chain".
Everything below that level (decoder architecture, scale granularity, where fp32 roundings sit)
is BASELINE.json:north_star/configs plus the readings listed in DESIGN.md section 3 (R-*),
cited at each function.

Precision convention (DESIGN.md R-accum): element-wise operations are single IEEE fp32
operations in the order written; every reduction (dot products, mean of squares, softmax sums)
is accumulated in fp64 and rounded once to fp32.  For the E4M3 dot products fp64 accumulation
is *exact* (products are multiples of 2^-18 below 2^18; 2^14 of them stay below 2^53), so
"rounded once" is the correctly rounded value of the true sum, the value every fp32-accumulating
implementation approximates.

Pins: tests/test_oracle_*.py.  End-to-end logits of the 8B-shape
random model have no external truth: "parity unpinned" for that single item, everything it is
composed of is pinned on small shapes.
"""
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

from . import e4m3

try:  # a library matmul is allowed as a step; torch's CPU dgemm is ~2.5x numpy's here
    import torch as _torch
except Exception:  # pragma: no cover
    _torch = None

F32 = np.float32
_N_THREADS = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
_LUT64 = e4m3.decode_table()


# ----------------------------------------------------------------------------- helpers

def bf16_bits_to_f32(bits):
    return (np.ascontiguousarray(bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(F32)


def round_to_bf16(x):
    """fp32 -> nearest bf16 (ties to even), returned as fp32 holding the bf16 value.
    This is the KV-cache storage format (BASELINE.json: "paged bf16 KV cache")."""
    u = np.ascontiguousarray(x, dtype=F32).view(np.uint32)
    lsb = (u >> np.uint32(16)) & np.uint32(1)
    r = (u + np.uint32(0x7FFF) + lsb) & np.uint32(0xFFFF0000)
    return r.view(F32)


def f32_to_bf16_bits(x):
    return (round_to_bf16(x).view(np.uint32) >> np.uint32(16)).astype(np.uint16)


def _matmul64(a, bt):
    """a[M,K] @ bt[N,K]^T in fp64 (library dgemm)."""
    if _torch is not None:
        return (_torch.from_numpy(np.ascontiguousarray(a)) @ _torch.from_numpy(np.ascontiguousarray(bt)).T).numpy()
    return a @ bt.T


# ----------------------------------------------------------------------------- quantization

def quantize_weight(w_bf16_bits, per_tensor=False):
    """Absmax E4M3 quantization of a [N_out, K] bf16 matrix.
    Per output channel (default; BASELINE.json:configs[0] "E4M3 per-output-channel absmax scales";
    PAPER.md:98 "min-max"): s_w[n] = max_k |W[n,k]| / 448 (fp32 IEEE division; 1 for an all-zero row);
    Wq[n,k] = encode(W[n,k] / s_w[n]) (fp32 IEEE division).  DESIGN.md R-quant.
    per_tensor=True ("per-tensor"; DESIGN.md R-pertensor): ONE scale per
    matrix, s_w = max_{n,k} |W[n,k]| / 448, returned replicated over the N_out channels."""
    w_bf16_bits = np.asarray(w_bf16_bits)
    t_amax = None
    if per_tensor:
        t_amax = F32(0.0)
        for r0 in range(0, w_bf16_bits.shape[0], 4096):
            t_amax = max(t_amax, F32(np.max(np.abs(bf16_bits_to_f32(w_bf16_bits[r0:r0 + 4096])))))

    def rows(block):
        w = bf16_bits_to_f32(block)
        amax = np.max(np.abs(w), axis=1).astype(F32)
        if t_amax is not None:
            amax = np.full_like(amax, t_amax)
        s = (amax / F32(448.0)).astype(F32)
        s = np.where(amax == 0, F32(1.0), s).astype(F32)
        return e4m3.encode((w / s[:, None]).astype(F32)), s

    n = w_bf16_bits.shape[0]
    if w_bf16_bits.size < (1 << 22):
        return rows(w_bf16_bits)
    # rows are independent: big matrices go through a thread pool in row blocks (same arithmetic)
    step = max(1, (1 << 21) // w_bf16_bits.shape[1])
    with ThreadPoolExecutor(max_workers=_N_THREADS) as ex:
        parts = list(ex.map(lambda r0: rows(w_bf16_bits[r0:r0 + step]), range(0, n, step)))
    return np.concatenate([p[0] for p in parts]), np.concatenate([p[1] for p in parts])


def quantize_rows(x, static_scale=None):
    """Per-token activation quantization.  Dynamic (BASELINE.json:north_star (1) "per-token
    dynamic activation scales"): s_x[m] = max_k |x[m,k]| / 448 (1 for a zero row).
    Static (config[4], DESIGN.md R-static): s_x[m] = the calibrated constant of this site;
    values beyond 448*s saturate (that is the clipping PAPER.md:140 counts).
    Returns (codes uint8 [M,K], s_x fp32 [M])."""
    x = np.asarray(x, dtype=F32)
    if static_scale is None:
        amax = np.max(np.abs(x), axis=1).astype(F32)
        s = (amax / F32(448.0)).astype(F32)
        s = np.where(amax == 0, F32(1.0), s).astype(F32)
    else:
        s = np.full(x.shape[0], static_scale, dtype=F32)
    codes = e4m3.encode((x / s[:, None]).astype(F32))
    return codes, s


ACCUM_MODES = ("exact", "f32", "f32perm", "f32seq")


def _perm_k(K):
    """The fixed permutation of the K axis used by accum="f32perm" (seeded by K only)."""
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([0x5EED, K]))).permutation(K)


def linear(xq, s_x, wq, s_w, accum="exact", n_block=8192):
    """W8A8 linear, DESIGN.md R-accum:
    y[m,n] = fp32( sum_k decode(xq[m,k]) * decode(wq[n,k]) ) * s_x[m] * s_w[n],
    the sum exact (fp64) and rounded once, the two scales applied left to right in fp32.
    The other accumulation modes exist for the noise-floor study only (SURVEY section 8(c)-6 item 1, 8(c)-7 `--accum`;
    DESIGN.md R-noise): they are what an honest fp32-accumulating implementation may compute instead of the exact sum:
      "f32"     a library fp32 GEMM (its own blocked summation order);
      "f32perm" the same library GEMM with the K axis of both operands permuted by one fixed permutation (a second,
                unrelated fp32 summation order);
      "f32seq"  strictly sequential fp32 accumulation over k ascending (slow: small cases and pins).
    The loop over n_block output channels bounds memory; it splits no reduction."""
    assert accum in ACCUM_MODES, accum
    M, K = xq.shape
    N = wq.shape[0]
    x64 = _LUT64[xq]
    y = np.empty((M, N), dtype=F32)
    perm = _perm_k(K) if accum == "f32perm" else None
    for n0 in range(0, N, n_block):
        w64 = _LUT64[wq[n0:n0 + n_block]]
        if accum == "exact":
            acc = _matmul64(x64, w64).astype(F32)
        elif accum == "f32":
            acc = (x64.astype(F32) @ w64.astype(F32).T).astype(F32)
        elif accum == "f32perm":
            acc = (np.ascontiguousarray(x64[:, perm].astype(F32)) @ np.ascontiguousarray(w64[:, perm].astype(F32)).T).astype(F32)
        else:
            x32, w32 = x64.astype(F32), w64.astype(F32)
            acc = np.zeros((M, w32.shape[0]), dtype=F32)
            for k in range(K):    # every product is exact in fp32; one rounded fp32 addition per k
                acc = (acc + x32[:, k, None] * w32[None, :, k]).astype(F32)
        y[:, n0:n0 + n_block] = (acc * s_x[:, None].astype(F32)) * s_w[None, n0:n0 + n_block].astype(F32)
    return y


# ----------------------------------------------------------------------------- perturbation injection

ROUND_MODES = {"bf16": 8, "tf32": 11, "split16": 16}   # significand bits kept (implicit one included)
ROUND_SITES = ("resid", "prequant", "qp")


def round_sig(x, bits):
    """fp32 -> nearest value with `bits` significand bits (round to nearest, ties to even), as fp32.  bits = 8 is bf16,
    11 is tf32's operand precision, 16 is what a hi+lo pair of bf16 holds.  Used ONLY by the perturbation-injection
    switches (SURVEY section 8(c)-6/7 `--round <site>:bf16|tf32|split16`; DESIGN.md R-noise); the default oracle never
    rounds anywhere but at the E4M3 quantizers and the bf16 K/V."""
    drop = 24 - bits
    u = np.ascontiguousarray(x, dtype=F32).view(np.uint32)
    if drop <= 0:
        return u.view(F32).copy()
    lsb = (u >> np.uint32(drop)) & np.uint32(1)
    r = (u + np.uint32((1 << (drop - 1)) - 1) + lsb) & np.uint32((0xFFFFFFFF << drop) & 0xFFFFFFFF)
    return r.view(F32)


# ----------------------------------------------------------------------------- element ops

def rmsnorm(h, gain, eps):
    """y = (h * r) * g with r = 1/sqrtf(mean_k h_k^2 + eps); the mean in fp64 rounded once.
    BASELINE.json:configs[0] "RMSNorm eps 1e-5"."""
    h = np.asarray(h, dtype=F32)
    ms = (np.sum(h.astype(np.float64) ** 2, axis=1) / h.shape[1]).astype(F32)
    r = (F32(1.0) / np.sqrt((ms + F32(eps)).astype(F32))).astype(F32)
    return ((h * r[:, None]).astype(F32) * gain[None, :].astype(F32)).astype(F32)


def rope_cos_sin(positions, head_dim, theta):
    """angle[p, j] = p * theta^(-2j/d), j < d/2; computed in fp64, cos/sin rounded to fp32.
    BASELINE.json:north_star (3) "positions = context length + tree depth"."""
    j = np.arange(head_dim // 2, dtype=np.float64)
    inv_freq = np.float64(theta) ** (-(2.0 * j) / head_dim)
    ang = np.asarray(positions, dtype=np.float64)[:, None] * inv_freq[None, :]
    return np.cos(ang).astype(F32), np.sin(ang).astype(F32)


def apply_rope(x, cos, sin):
    """Half-split pairing (DESIGN.md R-rope): for j < d/2
    (x_j, x_{j+d/2}) -> (x_j cos - x_{j+d/2} sin,  x_{j+d/2} cos + x_j sin); x is [M, heads, d]."""
    d2 = x.shape[-1] // 2
    a, b = x[..., :d2].astype(F32), x[..., d2:].astype(F32)
    c, s = cos[:, None, :], sin[:, None, :]
    lo = ((a * c).astype(F32) - (b * s).astype(F32)).astype(F32)
    hi = ((b * c).astype(F32) + (a * s).astype(F32)).astype(F32)
    return np.concatenate([lo, hi], axis=-1)


def swiglu(g, u):
    """t = (g / (1 + exp(-g))) * u; exp evaluated in fp64 and rounded to fp32, the rest fp32."""
    g = np.asarray(g, dtype=F32)
    e = np.exp(-g.astype(np.float64)).astype(F32)
    sig = (g / (F32(1.0) + e).astype(F32)).astype(F32)
    return (sig * np.asarray(u, dtype=F32)).astype(F32)


def ancestor_mask(parents):
    """anc[i, j] = True iff j is i or an ancestor of i (node 0 = root, parents[i] < i)."""
    T = len(parents)
    anc = np.zeros((T, T), dtype=bool)
    for i in range(T):
        j = i
        while j >= 0:
            anc[i, j] = True
            j = int(parents[j])
    return anc


def node_depths(parents):
    d = np.zeros(len(parents), dtype=np.int64)
    for i in range(1, len(parents)):
        d[i] = d[parents[i]] + 1
    return d


def tree_attention(q, k_ctx, v_ctx, k_tree, v_tree, parents, qp_bits=None):
    """Tree attention: node i attends to the L committed context positions and to
    its own ancestors-or-self among the tree nodes; GQA: q-head h uses kv-head h // (Hq/Hkv).
    q [T,Hq,d] fp32; k_*/v_* hold bf16 values (as fp32): ctx [L,Hkv,d], tree [T,Hkv,d].
    s = fp32(q.k) * fp32(1/sqrt(d)); m = max s; p = fp32(exp(s - m)); out = fp32(sum p v) / fp32(sum p);
    the three sums in fp64 rounded once (DESIGN.md R-accum).  Returns [T, Hq*d] fp32."""
    T, Hq, d = q.shape
    Hkv = k_tree.shape[1]
    G = Hq // Hkv
    if qp_bits is not None:      # perturbation injection "qp": Q and P rounded as a tensor-core attention would hold them
        q = round_sig(q, qp_bits)
    scale = (F32(1.0) / np.sqrt(F32(d))).astype(F32)
    anc = ancestor_mask(parents)
    out = np.empty((T, Hq, d), dtype=F32)
    for g in range(Hkv):
        keys = np.concatenate([k_ctx[:, g, :], k_tree[:, g, :]], axis=0).astype(np.float64)   # [L+T, d]
        vals = np.concatenate([v_ctx[:, g, :], v_tree[:, g, :]], axis=0).astype(np.float64)
        L = k_ctx.shape[0]
        for hh in range(G):
            h = g * G + hh
            s = (_matmul64(q[:, h, :].astype(np.float64), keys).astype(F32) * scale).astype(F32)  # [T, L+T]
            s[:, L:][~anc] = -np.inf
            m = np.max(s, axis=1, keepdims=True)
            p = np.exp((s - m).astype(F32).astype(np.float64)).astype(F32)
            l = np.sum(p.astype(np.float64), axis=1).astype(F32)
            if qp_bits is not None:
                p = round_sig(p, qp_bits)
            o = (p.astype(np.float64) @ vals).astype(F32)
            out[:, h, :] = (o / l[:, None]).astype(F32)
    return out.reshape(T, Hq * d)


# ----------------------------------------------------------------------------- model + cache

SITES = ("qkv_in", "o_in", "gateup_in", "down_in")   # per layer; plus "lm_in" once


class OracleModel:
    """Quantized target model.  set_weight() quantizes bf16 matrices on arrival; q,k,v share the
    input quantization and are three independent per-output-channel matrices, likewise gate/up
    (DESIGN.md R-quant).  Embedding and RMSNorm gains stay bf16 (R-embed)."""

    def __init__(self, shape, act_scale_mode=0, accum="exact", weight_scale_mode=0):
        for f in ("n_layers", "hidden", "n_q_heads", "n_kv_heads", "head_dim", "ffn", "vocab",
                  "rms_eps", "rope_theta"):
            setattr(self, f, getattr(shape, f))
        self.act_scale_mode = act_scale_mode
        self.weight_scale_mode = weight_scale_mode   # 0 per output channel, 1 per tensor (each matrix its own scale)
        self.accum = accum
        self.inject = {}     # perturbation injection: site in ROUND_SITES -> significand bits (empty = none, the default)
        self.w = {}          # (kind, layer) -> (codes, scales)
        self.embed = None    # bf16 bits [V, H]
        self.gain = {}       # ("norm1"|"norm2", layer) / ("normf", 0) -> fp32 [H]
        self.static = {}     # (site, layer) -> fp32 scale, when act_scale_mode == 1
        self.clip_counts = {}

    def set_weight(self, kind, layer, bf16_bits):
        if kind == "embed":
            self.embed = np.ascontiguousarray(bf16_bits, dtype=np.uint16)
        elif kind in ("norm1", "norm2", "normf"):
            self.gain[(kind, layer)] = bf16_bits_to_f32(bf16_bits)
        else:
            self.w[(kind, layer)] = quantize_weight(bf16_bits, per_tensor=self.weight_scale_mode == 1)

    def set_quantized(self, kind, layer, codes, scales):
        self.w[(kind, layer)] = (np.ascontiguousarray(codes, dtype=np.uint8), np.ascontiguousarray(scales, dtype=F32))

    def _gain(self, kind, layer):
        g = self.gain.get((kind, layer))
        return g if g is not None else np.ones(self.hidden, dtype=F32)

    def set_round(self, spec):
        """spec: "" or "<site>:<mode>[,<site>:<mode>...]" with site in ROUND_SITES, mode in ROUND_MODES."""
        self.inject = {}
        for item in filter(None, (spec or "").split(",")):
            site, mode = item.split(":")
            assert site in ROUND_SITES and mode in ROUND_MODES, item
            self.inject[site] = ROUND_MODES[mode]

    def _inj(self, x, site):
        b = self.inject.get(site)
        return x if b is None else round_sig(x, b)

    def _quant(self, x, site, layer, record=None):
        x = self._inj(x, "prequant")
        if record is not None:   # calibration pass: dynamic scales, remember per-site absmax
            record[(site, layer)] = max(record.get((site, layer), 0.0), float(np.max(np.abs(x))))
            return quantize_rows(x)
        if self.act_scale_mode == 1:
            s = self.static[(site, layer)]
            codes, sx = quantize_rows(x, static_scale=s)
            self.clip_counts[(site, layer)] = self.clip_counts.get((site, layer), 0) + \
                int(np.count_nonzero(np.abs(x) > F32(448.0) * s))
            return codes, sx
        return quantize_rows(x)

    def _lin(self, xq, sx, kind, layer):
        wq, sw = self.w[(kind, layer)]
        return linear(xq, sx, wq, sw, accum=self.accum)


class OracleKV:
    """Paged bf16 KV cache (BASELINE.json:configs[2] "bf16 paged KV cache with 16-token pages").
    pool[layer] is uint16 [n_pages, 2(K|V), Hkv, page_size, d]; a sequence owns a list of physical
    pages; token slot t lives in page_table[seq][t // page_size] at offset t % page_size.
    Layers are allocated on first touch so sampled-layer checks at 8B shape stay small.
    kv_dtype="e4m3" ("quantizing the KV cache to FP8 halves the storage compared to FP16/BF16"; SURVEY section
    8(f)-2; DESIGN.md R-kv8): the pool holds E4M3 codes (one byte per element) and K, V are quantized with STATIC per-tensor
    scales - one for the K cache and one for the V cache of each layer, set by calibrate() as absmax / 448 over the
    calibration tokens (the paper's static min-max PTQ): code = E4M3_sat(x / s) on write (values beyond 448 s saturate),
    value = fp32(decode(code) * s) on read.  The scales live in model.static under ("k_cache", layer), ("v_cache", layer)."""

    def __init__(self, model, n_pages, page_size=16, page_order=None, kv_dtype="bf16"):
        assert kv_dtype in ("bf16", "e4m3")
        self.kv_dtype, self.model = kv_dtype, model
        self.Hkv, self.d, self.page_size, self.n_pages = model.n_kv_heads, model.head_dim, page_size, n_pages
        self.pool = {}
        self.free = list(range(n_pages)) if page_order is None else list(page_order)
        self.page_table = {}
        self.ctx_len = {}

    def _layer(self, layer):
        if layer not in self.pool:
            self.pool[layer] = np.zeros((self.n_pages, 2, self.Hkv, self.page_size, self.d),
                                        dtype=np.uint16 if self.kv_dtype == "bf16" else np.uint8)
        return self.pool[layer]

    def bytes_per_token(self):
        """cache storage per token per layer"""
        return 2 * self.Hkv * self.d * (2 if self.kv_dtype == "bf16" else 1)

    def _scales(self, layer):
        return F32(self.model.static[("k_cache", layer)]), F32(self.model.static[("v_cache", layer)])

    def _encode(self, layer, k, v):
        """fp32 K, V -> the pool's storage bits"""
        if self.kv_dtype == "bf16":
            return f32_to_bf16_bits(k), f32_to_bf16_bits(v)
        sk, sv = self._scales(layer)
        return e4m3.encode((np.asarray(k, dtype=F32) / sk).astype(F32)), e4m3.encode((np.asarray(v, dtype=F32) / sv).astype(F32))

    def _decode(self, layer, kb, vb):
        if self.kv_dtype == "bf16":
            return bf16_bits_to_f32(kb), bf16_bits_to_f32(vb)
        sk, sv = self._scales(layer)
        return (e4m3.decode(kb).astype(F32) * sk).astype(F32), (e4m3.decode(vb).astype(F32) * sv).astype(F32)

    def add_seq(self, seq, capacity_tokens):
        n = -(-capacity_tokens // self.page_size)
        assert len(self.free) >= n, "out of pages"
        self.page_table[seq] = [self.free.pop(0) for _ in range(n)]
        self.ctx_len[seq] = 0

    def capacity(self, seq):
        return len(self.page_table[seq]) * self.page_size

    def write(self, layer, seq, slots, k, v):
        """k, v: fp32 [n, Hkv, d]; stored rounded to bf16 (or quantized to E4M3, kv_dtype)."""
        pool = self._layer(layer)
        kb, vb = self._encode(layer, k, v)
        for i, t in enumerate(slots):
            pg, off = self.page_table[seq][t // self.page_size], t % self.page_size
            pool[pg, 0, :, off, :] = kb[i]
            pool[pg, 1, :, off, :] = vb[i]

    def read(self, layer, seq, start, stop):
        """-> K, V as fp32 [stop-start, Hkv, d] (the stored values: bf16, or dequantized E4M3)."""
        pool = self._layer(layer)
        slots = np.arange(start, stop)
        pages = np.asarray(self.page_table[seq], dtype=np.int64)[slots // self.page_size]
        offs = slots % self.page_size
        blk = pool[pages, :, :, offs, :]            # [n, 2, Hkv, d]
        return self._decode(layer, blk[:, 0], blk[:, 1])

    def read_bits(self, layer, seq, start, stop):
        """-> the stored bits of K, V: [stop-start, Hkv, d] uint16 (bf16) or uint8 (E4M3 codes)"""
        pool = self._layer(layer)
        slots = np.arange(start, stop)
        pages = np.asarray(self.page_table[seq], dtype=np.int64)[slots // self.page_size]
        blk = pool[pages, :, :, slots % self.page_size, :]
        return blk[:, 0], blk[:, 1]

    def move(self, seq, src_slot, dst_slot):
        for pool in self.pool.values():
            ps, os_ = self.page_table[seq][src_slot // self.page_size], src_slot % self.page_size
            pd, od = self.page_table[seq][dst_slot // self.page_size], dst_slot % self.page_size
            pool[pd, :, :, od, :] = pool[ps, :, :, os_, :]

    def export_dense(self, layer, seq, n_tokens):
        """-> stored bits [2, Hkv, n_tokens, d] (the layout of the library's export, per layer)."""
        kb, vb = self.read_bits(layer, seq, 0, n_tokens)
        return np.ascontiguousarray(np.stack([kb.transpose(1, 0, 2), vb.transpose(1, 0, 2)]))

    def import_dense(self, layer, seq, dense_bits):
        """dense_bits (stored bits) [2, Hkv, n, d] -> slots 0..n-1 of seq (DESIGN.md R-kv-input)."""
        n = dense_bits.shape[2]
        pool = self._layer(layer)
        kb, vb = dense_bits[0].transpose(1, 0, 2), dense_bits[1].transpose(1, 0, 2)
        for t in range(n):
            pg, off = self.page_table[seq][t // self.page_size], t % self.page_size
            pool[pg, 0, :, off, :] = kb[t]
            pool[pg, 1, :, off, :] = vb[t]


# ----------------------------------------------------------------------------- forward

def layer_forward(model, layer, h, cache, seq, L, parents, record=None, taps=None):
    """One decoder layer over the T tree nodes of sequence `seq` whose cache holds L tokens.
    Writes node i's K/V at slot L+i (BASELINE.json:north_star "the KV append") and returns the
    new residual stream [T, H].  `taps` (dict) collects intermediates for per-kernel checks."""
    T = h.shape[0]
    Hq, Hkv, d = model.n_q_heads, model.n_kv_heads, model.head_dim
    depth = node_depths(parents)
    x = rmsnorm(h, model._gain("norm1", layer), model.rms_eps)
    xq, sx = model._quant(x, "qkv_in", layer, record)
    q = model._lin(xq, sx, "wq", layer).reshape(T, Hq, d)
    k = model._lin(xq, sx, "wk", layer).reshape(T, Hkv, d)
    v = model._lin(xq, sx, "wv", layer).reshape(T, Hkv, d)
    cos, sin = rope_cos_sin(L + depth, d, model.rope_theta)
    q, k = apply_rope(q, cos, sin), apply_rope(k, cos, sin)
    if record is not None:   # calibration pass: per-tensor absmax of what the cache stores (FP8 KV scales, DESIGN.md R-kv8)
        record[("k_cache", layer)] = max(record.get(("k_cache", layer), 0.0), float(np.max(np.abs(k))))
        record[("v_cache", layer)] = max(record.get(("v_cache", layer), 0.0), float(np.max(np.abs(v))))
    cache.write(layer, seq, [L + i for i in range(T)], k, v)          # rounds to bf16 (or quantizes to E4M3)
    k_ctx, v_ctx = cache.read(layer, seq, 0, L)
    k_tree, v_tree = cache.read(layer, seq, L, L + T)
    attn = tree_attention(q, k_ctx, v_ctx, k_tree, v_tree, parents, qp_bits=model.inject.get("qp"))
    aq, sa = model._quant(attn, "o_in", layer, record)
    h = model._inj((h + model._lin(aq, sa, "wo", layer)).astype(F32), "resid")
    x2 = rmsnorm(h, model._gain("norm2", layer), model.rms_eps)
    x2q, s2 = model._quant(x2, "gateup_in", layer, record)
    g = model._lin(x2q, s2, "wgate", layer)
    u = model._lin(x2q, s2, "wup", layer)
    t = swiglu(g, u)
    tq, st = model._quant(t, "down_in", layer, record)
    h_out = model._inj((h + model._lin(tq, st, "wdown", layer)).astype(F32), "resid")
    if taps is not None:
        taps.update(dict(x=x, xq=xq, sx=sx, q=q, k=k, v=v, attn=attn, aq=aq, sa=sa, h_mid=h,
                         x2q=x2q, s2=s2, g=g, u=u, t=t, tq=tq, st=st))
    return h_out


def lm_head(model, h, record=None):
    x = rmsnorm(h, model._gain("normf", 0), model.rms_eps)
    xq, sx = model._quant(x, "lm_in", 0, record)
    return model._lin(xq, sx, "lm_head", 0)


def embed(model, tokens):
    return bf16_bits_to_f32(model.embed[np.asarray(tokens, dtype=np.int64)])


def forward_tree(model, cache, seq, tokens, parents, record=None, want_hidden=False):
    """Full forward over one sequence's tree.  -> (logits [T,V] fp32, hidden list or None)."""
    L = cache.ctx_len[seq]
    assert L + len(tokens) <= cache.capacity(seq), "capacity"
    h = embed(model, tokens)
    hidden = [h] if want_hidden else None
    for layer in range(model.n_layers):
        h = layer_forward(model, layer, h, cache, seq, L, parents, record)
        if want_hidden:
            hidden.append(h)
    return lm_head(model, h, record), hidden


# ----------------------------------------------------------------------------- acceptance

def argmax_lowest(logits):
    """Row argmax, lowest token id on exact ties (DESIGN.md R-ties)."""
    return np.argmax(logits, axis=1).astype(np.int32)


def accept_walk(tokens, parents, am):
    """Greedy acceptance (BASELINE.json:north_star (4)): from the root, move to
    the lowest-index child whose token equals the target argmax at the current node; stop when
    none does.  Returns (path, out_tokens): path[0] = 0 (root), a = len(path)-1 accepted drafts,
    out_tokens = accepted draft tokens then the bonus token argmax[path[-1]] (a+1 tokens)."""
    cur, path = 0, [0]
    T = len(tokens)
    while True:
        nxt = -1
        for c in range(cur + 1, T):
            if parents[c] == cur and tokens[c] == am[cur]:
                nxt = c
                break
        if nxt < 0:
            break
        path.append(nxt)
        cur = nxt
    out = [int(tokens[c]) for c in path[1:]] + [int(am[cur])]
    return path, out


def kv_compact(cache, seq, path):
    """KV append after acceptance: slot L+path[j] -> slot L+j for j = 0..a (path[j] >= j so the
    forward in-place copy is safe); ctx_len = L + a + 1.  The bonus token is the next root."""
    L = cache.ctx_len[seq]
    for j, node in enumerate(path):
        if node != j:
            cache.move(seq, L + node, L + j)
    cache.ctx_len[seq] = L + len(path)


def verify(model, cache, seq, tokens, parents, commit=True, want_hidden=False):
    """verify(tree, cache) -> accepted tokens plus the KV append, for one sequence."""
    logits, hidden = forward_tree(model, cache, seq, tokens, parents, want_hidden=want_hidden)
    am = argmax_lowest(logits)
    path, out = accept_walk(tokens, parents, am)
    if commit:
        kv_compact(cache, seq, path)
    return dict(logits=logits, hidden=hidden, argmax=am, path=path, out_tokens=out,
                accept_len=len(path) - 1, new_ctx_len=cache.ctx_len[seq])


def prefill(model, cache, seq, ids, chunk=64, record=None):
    """Context KV by definition: the K/V the quantized model yields for `ids` under causal
    attention = a chain tree with every node force-accepted (DESIGN.md R-kv-input)."""
    last = None
    for c0 in range(0, len(ids), chunk):
        part = np.asarray(ids[c0:c0 + chunk])
        par = np.arange(-1, len(part) - 1)
        last, _ = forward_tree(model, cache, seq, part, par, record)
        cache.ctx_len[seq] += len(part)
    return last


def decode_greedy(model, cache, seq, root, n_steps):
    """Plain token-by-token greedy decoding (the sequence speculative decoding must reproduce)."""
    out, tok = [], int(root)
    for _ in range(n_steps):
        logits, _ = forward_tree(model, cache, seq, np.array([tok]), np.array([-1]))
        cache.ctx_len[seq] += 1
        tok = int(argmax_lowest(logits)[0])
        out.append(tok)
    return out


def calibrate(model, calib_hidden, n_pages=None, page_size=16):
    """Static activation scales ("Static quantization sets scales offline from
    activation statistics collected on calibration data"; config[4]; DESIGN.md R-static):
    feed calib_hidden [n, H] as the layer-0 residual stream of n causal tokens at positions
    0..n-1 of an empty cache, run with dynamic scales, record per site the absmax over all
    tokens and channels; s_site = absmax / 448."""
    n = calib_hidden.shape[0]
    cache = OracleKV(model, n_pages or -(-n // page_size), page_size)
    cache.add_seq(0, n)
    record = {}
    h = np.asarray(calib_hidden, dtype=F32)
    par = np.arange(-1, n - 1)
    for layer in range(model.n_layers):
        h = layer_forward(model, layer, h, cache, 0, 0, par, record)
    lm_head(model, h, record)
    model.static = {k: (F32(v) / F32(448.0)).astype(F32) if v > 0 else F32(1.0) for k, v in record.items()}
    return record
