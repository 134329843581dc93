"""Pins P2/P3/P12: the oracle's quantizer and element ops against closed forms, invariants and
library routines (never against a retyped copy of the oracle's own formula)."""
import numpy as np
import pytest

import workloads as wl
from oracle import e4m3
from oracle import verify_oracle as vo
from helpers import rel_l2

torch = pytest.importorskip("torch")


def _grid_matrix(rng, n, k, row_pow2=True):
    """values exactly on the E4M3 grid times a power-of-two row scale, each row containing 448."""
    t = e4m3.decode_table()
    finite = t[~np.isnan(t)]
    w = rng.choice(finite, size=(n, k))
    w[:, 0] = 448.0
    sc = 2.0 ** rng.integers(-12, -4, size=n) if row_pow2 else np.ones(n)
    return (w * sc[:, None]).astype(np.float32), sc.astype(np.float32)


def test_p2_grid_weights_quantize_losslessly_and_linear_is_exact():
    rng = np.random.default_rng(0)
    w, sc = _grid_matrix(rng, 24, 96)
    bits = wl.f32_to_bf16_bits(w)
    assert np.array_equal(wl.bf16_bits_to_f32(bits), w)            # 4 significant bits fit bf16
    codes, s = vo.quantize_weight(bits)
    assert np.array_equal(s, sc)                                    # 448*2^k / 448 exactly
    assert np.array_equal(e4m3.decode(codes) * s[:, None].astype(np.float64), w.astype(np.float64))
    x, sx_true = _grid_matrix(rng, 7, 96)
    xq, sx = vo.quantize_rows(x)
    assert np.array_equal(sx, sx_true)
    y = vo.linear(xq, sx, codes, s)
    exact = x.astype(np.float64) @ w.astype(np.float64).T          # power-of-two scales commute
    assert np.array_equal(y, exact.astype(np.float32))


def test_p2_row_scaling_by_power_of_two():
    w = wl.weight_matrix_bf16(wl.TINY, 5, "wq", 0)
    f = wl.bf16_bits_to_f32(w)
    c1, s1 = vo.quantize_weight(w)
    c2, s2 = vo.quantize_weight(wl.f32_to_bf16_bits(f * np.float32(4.0)))
    assert np.array_equal(c1, c2) and np.array_equal(s2, s1 * np.float32(4.0))
    assert np.all(np.max(c1 & 0x7F, axis=1) == 0x7E)               # every row reaches +-448
    # dequantized weights are within half an E4M3 step (2^-4 relative) of the originals
    deq = e4m3.decode(c1) * s1[:, None]
    assert np.max(np.abs(deq - f) / np.maximum(np.abs(f), s1[:, None] * 2.0 ** -6)) <= 2.0 ** -4 + 1e-6


def test_zero_row_scale_is_one():
    w = np.zeros((3, 16), dtype=np.uint16)
    codes, s = vo.quantize_weight(w)
    assert np.all(codes == 0) and np.all(s == 1.0)
    xq, sx = vo.quantize_rows(np.zeros((2, 16), dtype=np.float32))
    assert np.all(xq == 0) and np.all(sx == 1.0)


def test_linear_matches_fp64_matmul_of_dequantized():
    rng = np.random.default_rng(3)
    x = rng.standard_normal((5, 256)).astype(np.float32)
    w = wl.weight_matrix_bf16(wl.TINY, 1, "wk", 0)
    xq, sx = vo.quantize_rows(x)
    wq, sw = vo.quantize_weight(w)
    y = vo.linear(xq, sx, wq, sw)
    # library route: torch fp64 matmul of the torch-fp8-decoded codes
    xd = torch.from_numpy(xq).view(torch.float8_e4m3fn).double() * torch.from_numpy(sx).double()[:, None]
    wd = torch.from_numpy(wq).view(torch.float8_e4m3fn).double() * torch.from_numpy(sw).double()[:, None]
    assert rel_l2(y, (xd @ wd.T).numpy()) < 2e-7
    # quantization error of the whole W8A8 product vs the unquantized fp64 product: a few percent
    full = x.astype(np.float64) @ wl.bf16_bits_to_f32(w).astype(np.float64).T
    assert 5e-3 < rel_l2(y, full) < 6e-2
    assert rel_l2(vo.linear(xq, sx, wq, sw, accum="f32"), y) < 1e-6


def test_rmsnorm_invariants():
    rng = np.random.default_rng(4)
    h = rng.standard_normal((6, 256)).astype(np.float32) * 3
    y = vo.rmsnorm(h, np.ones(256, np.float32), 0.0)
    assert np.allclose(np.sqrt(np.mean(y.astype(np.float64) ** 2, axis=1)), 1.0, atol=1e-6)
    assert rel_l2(vo.rmsnorm(h * np.float32(8), np.ones(256, np.float32), 0.0), y) < 1e-6
    g = rng.uniform(0.5, 1.5, 256).astype(np.float32)
    ref = torch.nn.functional.rms_norm(torch.from_numpy(h).double(), (256,), torch.from_numpy(g).double(), 1e-5)
    assert rel_l2(vo.rmsnorm(h, g, 1e-5), ref.numpy()) < 2e-7
    c = np.full((1, 256), 2.0, np.float32)                 # constant row: y = 2/sqrt(4+eps)
    assert np.allclose(vo.rmsnorm(c, np.ones(256, np.float32), 1e-5), 2 / np.sqrt(4 + 1e-5), rtol=1e-7)


def test_rope_properties():
    rng = np.random.default_rng(5)
    d = 64
    x = rng.standard_normal((3, 2, d)).astype(np.float32)
    c0, s0 = vo.rope_cos_sin([0, 0, 0], d, 1e4)
    assert np.array_equal(vo.apply_rope(x, c0, s0), x)                         # position 0 = identity
    c, s = vo.rope_cos_sin([5, 77, 16390], d, 5e5)
    y = vo.apply_rope(x, c, s)
    assert np.allclose(np.linalg.norm(y, axis=-1), np.linalg.norm(x, axis=-1), rtol=1e-6)   # rotation
    # relative-position property: <R_p q, R_p' k> depends on p - p' only
    q = rng.standard_normal((1, 1, d)).astype(np.float32)
    k = rng.standard_normal((1, 1, d)).astype(np.float32)
    dots = []
    for p, pp in ((10, 3), (107, 100), (2055, 2048)):
        cq, sq = vo.rope_cos_sin([p], d, 1e4)
        ck, sk = vo.rope_cos_sin([pp], d, 1e4)
        dots.append(float(np.sum(vo.apply_rope(q, cq, sq).astype(np.float64) * vo.apply_rope(k, ck, sk))))
    assert np.allclose(dots, dots[0], rtol=0, atol=2e-4)
    # d = 2: one plain 2-D rotation by angle p (frequency theta^0 = 1)
    c2, s2 = vo.rope_cos_sin([2], 2, 1e4)
    v = vo.apply_rope(np.array([[[1.0, 0.0]]], np.float32), c2, s2)
    assert np.allclose(v[0, 0], [np.cos(2.0), np.sin(2.0)], atol=1e-7)
    # half-split pairing: element j pairs with j + d/2, frequency theta^(-2j/d)
    e = np.zeros((1, 1, d), np.float32)
    e[0, 0, 3] = 1.0
    c3, s3 = vo.rope_cos_sin([7], d, 1e4)
    r = vo.apply_rope(e, c3, s3)[0, 0]
    ang = 7 * 1e4 ** (-6.0 / d)
    assert np.allclose(r[3], np.cos(ang), atol=1e-7) and np.allclose(r[3 + d // 2], np.sin(ang), atol=1e-7)
    assert np.count_nonzero(r) == 2


def test_swiglu_vs_library():
    rng = np.random.default_rng(6)
    g = (rng.standard_normal((4, 688)) * 4).astype(np.float32)
    u = rng.standard_normal((4, 688)).astype(np.float32)
    ref = torch.nn.functional.silu(torch.from_numpy(g).double()) * torch.from_numpy(u).double()
    assert np.max(np.abs(vo.swiglu(g, u) - ref.numpy()) / (np.abs(ref.numpy()) + 1e-3)) < 3e-7
    assert vo.swiglu(np.zeros((1, 2), np.float32), np.ones((1, 2), np.float32)).tolist() == [[0.0, 0.0]]


def _mk_attn(rng, T, L, Hq=4, Hkv=2, d=16):
    q = rng.standard_normal((T, Hq, d)).astype(np.float32)
    kc = vo.round_to_bf16(rng.standard_normal((L, Hkv, d)).astype(np.float32))
    vc = vo.round_to_bf16(rng.standard_normal((L, Hkv, d)).astype(np.float32))
    kt = vo.round_to_bf16(rng.standard_normal((T, Hkv, d)).astype(np.float32))
    vt = vo.round_to_bf16(rng.standard_normal((T, Hkv, d)).astype(np.float32))
    return q, kc, vc, kt, vt


def test_attention_vs_library_sdpa_with_tree_mask():
    rng = np.random.default_rng(7)
    parents = np.array([-1, 0, 0, 1, 1, 2, 3])
    T, L, Hq, Hkv, d = len(parents), 37, 4, 2, 16
    q, kc, vc, kt, vt = _mk_attn(rng, T, L, Hq, Hkv, d)
    out = vo.tree_attention(q, kc, vc, kt, vt, parents).reshape(T, Hq, d)
    anc = vo.ancestor_mask(parents)
    mask = torch.from_numpy(np.concatenate([np.ones((T, L), bool), anc], axis=1))
    K = torch.from_numpy(np.concatenate([kc, kt])).double().repeat_interleave(Hq // Hkv, dim=1)
    V = torch.from_numpy(np.concatenate([vc, vt])).double().repeat_interleave(Hq // Hkv, dim=1)
    ref = torch.nn.functional.scaled_dot_product_attention(
        torch.from_numpy(q).double().permute(1, 0, 2), K.permute(1, 0, 2), V.permute(1, 0, 2), attn_mask=mask)
    assert rel_l2(out, ref.permute(1, 0, 2).numpy()) < 3e-7


def test_attention_special_cases():
    rng = np.random.default_rng(8)
    parents = np.array([-1, 0, 1, 1])
    q, kc, vc, kt, vt = _mk_attn(rng, 4, 9)
    # constant V => output = V (softmax rows sum to one)
    vconst = np.full_like(vc, 0.75)
    vtc = np.full_like(vt, 0.75)
    out = vo.tree_attention(q, kc, vconst, kt, vtc, parents)
    assert np.allclose(out, 0.75, atol=1e-7)
    # no context, root only: the single key is itself => output = its own V (GQA: head h -> kv h//2)
    out = vo.tree_attention(q[:1], kc[:0], vc[:0], kt[:1], vt[:1], np.array([-1])).reshape(4, 16)
    assert np.array_equal(out, vt[0][[0, 0, 1, 1]])
    # all keys identical => uniform weights => output = mean of visible V
    ksame = np.broadcast_to(kc[:1], kc.shape).copy()
    ktsame = np.broadcast_to(kc[:1], kt.shape).copy()
    out = vo.tree_attention(q, ksame, vc, ktsame, vt, parents).reshape(4, 4, 16)
    vis = np.concatenate([vc, vt[[0, 1, 3]]])                          # node 3: root, 1, itself
    assert np.allclose(out[3, 2], vis[:, 1, :].astype(np.float64).mean(axis=0), atol=1e-6)


def test_ancestor_mask_and_depths():
    p = wl.tree_parents(26, (4, 3, 2, 2, 1))
    anc = vo.ancestor_mask(p)
    d = vo.node_depths(p)
    assert np.array_equal(anc.sum(axis=1), d + 1) and int(anc.sum()) == 93
    assert np.all(np.triu(anc, 1) == 0) and np.all(anc[:, 0])


def test_p12_static_mode_clip_count_equals_saturated_codes():
    """clip rate = fraction of activations beyond the calibrated bounds."""
    rng = np.random.default_rng(9)
    x = rng.standard_normal((32, 256)).astype(np.float32)
    s = np.float32(2.0 ** -8)                       # calibrated absmax 1.75 -> several percent clipped
    codes, sx = vo.quantize_rows(x, static_scale=s)
    assert np.all(sx == s)
    n_clip = int(np.count_nonzero(np.abs(x) > np.float32(1.75)))
    sat = (codes & 0x7F) == 0x7E
    assert 100 < n_clip and np.count_nonzero(sat & (np.abs(x) > np.float32(1.75))) == n_clip
    deq = e4m3.decode(codes) * float(s)
    assert np.max(np.abs(deq)) == 1.75


def test_per_tensor_weight_quantizer_pins():
    """SURVEY 8(f)-1 / PAPER.md:98, 140: per-tensor min-max weight scales.  Pinned without retyping the formula:
    (i) a matrix on the E4M3 grid times ONE power of two quantizes losslessly with s = 2^k on every channel;
    (ii) the row that holds the matrix absmax gets the same codes as under per-channel scales, every other row's
    per-channel scale is <= the tensor scale; (iii) every code is the E4M3 value nearest to w / s, found by
    exhaustive search over the 256 codes (ties to the even code); (iv) an all-zero matrix has scale 1."""
    rng = np.random.default_rng(5)
    t = e4m3.decode_table()
    finite = t[~np.isnan(t)]
    w = (rng.choice(finite, size=(16, 64)) * 2.0 ** -7).astype(np.float32)
    w[3, 5] = np.float32(448.0 * 2.0 ** -7)
    bits = wl.f32_to_bf16_bits(w)
    codes, s = vo.quantize_weight(bits, per_tensor=True)
    assert np.all(s == np.float32(2.0 ** -7))
    assert np.array_equal(e4m3.decode(codes) * 2.0 ** -7, w.astype(np.float64))

    bits = wl.weight_matrix_bf16(wl.TINY, 0, "wq", 0)
    wf = wl.bf16_bits_to_f32(bits)
    codes_t, s_t = vo.quantize_weight(bits, per_tensor=True)
    codes_c, s_c = vo.quantize_weight(bits)
    r, _ = np.unravel_index(np.argmax(np.abs(wf)), wf.shape)
    assert np.all(s_t == s_t[0]) and s_t[0] == s_c[r] and np.all(s_c <= s_t[0])
    assert np.array_equal(codes_t[r], codes_c[r])
    # exhaustive nearest-code search on a sample of elements (fp64 distances; ties -> even code)
    vals = t.astype(np.float64)
    idx = rng.choice(wf.size, size=400, replace=False)
    x = (wf.reshape(-1)[idx] / s_t[0]).astype(np.float32).astype(np.float64)
    for xi, ci in zip(x, codes_t.reshape(-1)[idx]):
        d = np.abs(vals - xi)
        d[np.isnan(d)] = np.inf
        best = np.flatnonzero(d == d.min())
        assert ci in best and (len(best) == 1 or ci % 2 == 0 or vals[ci] == xi), (xi, ci, best)
    z, sz = vo.quantize_weight(np.zeros((4, 16), dtype=np.uint16), per_tensor=True)
    assert np.all(sz == 1.0) and np.all(z == 0)
