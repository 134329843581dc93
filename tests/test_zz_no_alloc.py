"""ev_op_linear_static (include/eagle_verify.h): the linear operator for callers that may not allocate - the GEMM kernel's
scratch (K-piece slabs) lives in a file-scope static __device__ array whose address the library resolves per device with
cudaGetSymbolAddress.  Checked against the existing path (ev_op_linear: same kernel, the model's cudaMalloc'ed workspace) on
calls in a row that share the static array: equal bit for bit (the tolerance the GEMM tests use, 1e-5 relative, is the
fallback bar stated below), stale contents of the array do not matter, sizes beyond the stated maximum are rejected.
Collected last (file name) so that a failure here hides no other test under `pytest -x`; needs no state from other tests."""
import dataclasses

import pytest

import workloads as wl

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

K_OF = {"wq": "hidden", "wo": "hidden", "wgate": "hidden", "wdown": "ffn"}
N_OF = {"wq": lambda s: s.q_dim + 2 * s.kv_dim, "wo": lambda s: s.hidden, "wgate": lambda s: 2 * s.ffn, "wdown": lambda s: s.hidden}


def _inputs(shape, kind, M, seed):
    g = torch.Generator(device="cpu").manual_seed(seed)
    K = getattr(shape, K_OF[kind])
    codes = torch.randint(0, 256, (M, K), dtype=torch.uint8, generator=g)
    codes[(codes & 0x7F) == 0x7F] = 0x38          # no NaN codes (E4M3 0x7F / 0xFF)
    sx = torch.rand(M, generator=g, dtype=torch.float32) * 0.05 + 0.001
    return codes.cuda(), sx.cuda()


def _both(model, shape, kind, M, seed):
    codes, sx = _inputs(shape, kind, M, seed)
    ref = model.ev_op_linear(kind, 0, codes, sx).clone()
    out = torch.full((M, N_OF[kind](shape)), float("nan"), dtype=torch.float32, device="cuda")
    model.ev_op_linear_static(kind, 0, codes, sx, out)
    torch.cuda.synchronize()
    assert torch.isfinite(ref).all() and ref.abs().max() > 0
    rel = float((out - ref).norm() / ref.norm())
    assert rel <= 1e-5, (kind, M, rel)             # the GEMM tests' bar (tests/test_gpu_kernels.py)
    assert torch.equal(out, ref), (kind, M, rel)   # same kernel, same K cuts: identical bits
    return out


def test_static_scratch_linear_matches_existing_path_on_calls_in_a_row():
    from gpu_helpers import gpu_model
    import paper_2606_18502_b200 as ev
    shape = wl.TINY
    model = gpu_model(shape, 0, max_batch=8, max_tree_nodes=64, max_ctx=256)
    # two calls in a row on the shared array, then more shapes: stream-K slabs (M <= 256, several K pieces per tile, ragged K = 688
    # and ragged N = 1376), the CTA-pair form (M = 300), a tiny M after a large one (the array keeps the last call's contents)
    first = _both(model, shape, "wgate", 60, 1)
    second = _both(model, shape, "wgate", 60, 1)
    assert torch.equal(first, second)
    for kind, M, seed in (("wdown", 17, 2), ("wq", 256, 3), ("wgate", 300, 4), ("wo", 1, 5), ("wdown", 60, 6), ("wq", 33, 7)):
        _both(model, shape, kind, M, seed)
    # LM head (argmax epilogue, no slabs) is not offered by this entry point
    codes, sx = _inputs(shape, "wq", 4, 8)
    with pytest.raises(ev.EvError):
        model.ev_op_linear_static("lm_head", 0, codes, sx, torch.empty((4, shape.vocab), device="cuda"))


def test_static_scratch_linear_rejects_sizes_beyond_its_maximum():
    """(M <= 256 ? 8 : 1) * M * N floats must fit 16 MiB: a wide FFN (gate|up N = 16,384) passes at M = 16, is refused at M = 64
    with EV_ECAPACITY and a message naming the limit; the refused call launches nothing and the next call is still right."""
    from gpu_helpers import gpu_model
    import paper_2606_18502_b200 as ev
    shape = dataclasses.replace(wl.TINY, name="tiny_wide_ffn", n_layers=1, ffn=8192)
    model = gpu_model(shape, 0, max_batch=2, max_tree_nodes=64, max_ctx=128)
    _both(model, shape, "wgate", 16, 11)
    codes, sx = _inputs(shape, "wgate", 64, 12)
    out = torch.zeros((64, 2 * shape.ffn), dtype=torch.float32, device="cuda")
    n0 = ev.ev_launch_count()
    with pytest.raises(ev.EvError) as e:
        model.ev_op_linear_static("wgate", 0, codes, sx, out)
    assert e.value.code == -3 and "static scratch" in str(e.value), str(e.value)   # EV_ECAPACITY
    assert "16 MiB" in str(e.value)
    assert ev.ev_launch_count() == n0
    assert float(out.abs().max()) == 0.0
    _both(model, shape, "wgate", 16, 13)
    _both(model, shape, "wdown", 64, 14)     # N = 256: 8 * 64 * 256 floats fit
