#!/usr/bin/env python
"""Benchmark of the FP8 EAGLE verify step (BASELINE.json metric) on one B200, or N replicas.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--impl ours|reference]

A "step" is one pass of the whole hot path (every row of SURVEY.md section 8(a): embedding gather,
32 x {RMSNorm+quant, QKV GEMM, RoPE+KV write, tree attention, merge+quant, O GEMM, RMSNorm+quant,
gate/up GEMM, SwiGLU+quant, down GEMM}, final norm, LM head + argmax, acceptance walk, KV compaction)
over one batch of synthetic draft trees, plus one tiny launch that rewinds ctx_len so every step
sees the same context.  Default workload = BASELINE.json configs[1] (8B shape, batch 1, context 2048,
60-node tree).  Prints ONE JSON line (rank 0).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

LAYER_KINDS = ("wq", "wk", "wv", "wo", "wgate", "wup", "wdown")
METRIC = "verified tree-tokens/s (FP8 EAGLE verify step)"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), bf16_tflops=float(d["bf16_tflops"]), source="measured")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, source="fallback")  # B200_PROFILING.md fallback


def fp8_peak_probe(torch):
    """Dense E4M3 tensor peak of THIS GPU, measured the way MEASURED_PEAKS.json measures its bf16 figure:
    an 8192^3 E4M3 matmul through torch._scaled_mm, best of 10 (burst).  A probe outside the product path: it only sets
    the FLOP roofline's denominator.  Falls back to 2 x the measured bf16 burst when the probe is unavailable."""
    try:
        a = torch.randn(8192, 8192, device="cuda").to(torch.float8_e4m3fn)
        b = torch.randn(8192, 8192, device="cuda").to(torch.float8_e4m3fn).t()
        one = torch.tensor(1.0, device="cuda")
        for _ in range(3):
            torch._scaled_mm(a, b, scale_a=one, scale_b=one, out_dtype=torch.bfloat16)
        best = 1e9
        for _ in range(10):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            torch._scaled_mm(a, b, scale_a=one, scale_b=one, out_dtype=torch.bfloat16)
            e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        del a, b
        torch.cuda.empty_cache()
        return 2 * 8192 ** 3 / (best * 1e-3), "measured: torch._scaled_mm 8192^3 E4M3, best of 10 (probe outside the product path)"
    except Exception as e:  # pragma: no cover
        return 2 * peaks()["bf16_tflops"] * 1e12, f"2 x bf16 burst (E4M3 probe unavailable: {type(e).__name__})"


# ------------------------------------------------------------------------------------------ workload

def tree_of(spec):
    return wl.chain_parents(spec.n_nodes) if spec.tree_caps is None else wl.tree_parents(spec.n_nodes, spec.tree_caps)


def algorithmic_work(spec, ctx_lens, parents, kv_fp8=False):
    """bytes = FP8 weight bytes + KV bytes of the context; FLOPs = linear + attention."""
    m = spec.model
    depth = wl.tree_depths(parents)
    B, T = len(ctx_lens), len(parents)
    kv_bytes = m.kv_bytes_per_token() * int(np.sum(ctx_lens)) // (2 if kv_fp8 else 1)
    w_bytes = m.weight_bytes_fp8()
    lin = B * T * m.linear_flops_per_token()
    attn = m.attn_flops_per_token_pos() * int(sum(int(L) * T + int((depth + 1).sum()) for L in ctx_lens))
    return dict(weight_bytes=w_bytes, kv_bytes=kv_bytes, flops=lin + attn)


class ClockSampler(threading.Thread):
    Q = "index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown," \
        "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, gpu_index):
        super().__init__(daemon=True)
        self.idx, self.rows, self._stop_evt = gpu_index, [], threading.Event()

    def run(self):
        while not self._stop_evt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                f = [x.strip() for x in out.strip().split(",")]
                if len(f) >= 8:
                    self.rows.append(f)
            except Exception:
                pass
            self._stop_evt.wait(0.2)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=6)
        if not self.rows:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["unavailable"])
        sm = sorted(float(r[1]) for r in self.rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[4 + i].lower().startswith("active") for r in self.rows)]
        return dict(sm_mhz=sm[len(sm) // 2], sm_max_mhz=float(self.rows[0][2]), reasons=reasons, samples=len(self.rows))


def rank0_chain(parents):
    """the nodes reached from the root by always taking the lowest-index child, by depth"""
    first_child = {}
    for i in range(1, len(parents)):
        first_child.setdefault(int(parents[i]), i)
    chain, cur = [], 0
    while cur in first_child:
        cur = first_child[cur]
        chain.append(cur)
    return chain


def plant(spec, parents, b, root, greedy_next, coins, base=None):
    """Draft tokens of one tree (DESIGN.md R-tokens): uniform ids with distinct siblings, the root given, and on the rank-0
    chain the GPU's own greedy continuation with probability 0.7 per depth (config[3]'s rule): coins[d] < 0.7 plants."""
    tk = wl.draft_tokens_uniform(spec, parents, b) if base is None else base.copy()
    tk[0] = root
    for d, node in enumerate(rank0_chain(parents)):
        if coins[d] < 0.7:
            tk[node] = greedy_next[d]
    for i in range(1, len(tk)):        # planting may have collided with a sibling
        sib = [tk[j] for j in range(1, i) if parents[j] == parents[i]]
        while tk[i] in sib:
            tk[i] = (tk[i] + 1) % spec.model.vocab
    return tk


def build_gpu_workload(spec, steps_total, torch, ev, log, loop_steps=0, kv_fp8=False, attn_chunk=0):
    shape = spec.model
    B, T = spec.batch, spec.n_nodes
    parents = tree_of(spec)
    ctx = wl.context_lengths(spec)
    D0 = int(wl.tree_depths(parents).max())
    grow = loop_steps * (D0 + 1) + D0 + 1 if loop_steps else 0     # tokens a sustained loop may append
    max_ctx = int(ctx.max()) + 64 + 8 + grow
    t0 = time.time()
    model = ev.Model(shape, max_batch=B, max_tree_nodes=64, max_ctx=max_ctx, page_size=spec.page_size,
                     act_scale_mode=spec.act_scale_mode, kv_dtype=1 if kv_fp8 else 0, attn_chunk=attn_chunk)
    for kind, layer in [("embed", 0)] + [(k, l) for l in range(shape.n_layers) for k in LAYER_KINDS] + [("lm_head", 0)]:
        model.ev_model_set_weight(kind, layer, wl.weight_matrix_bf16(shape, spec.seed, kind, layer, device="cuda"))
    torch.cuda.synchronize()
    log(f"weights quantized in {time.time() - t0:.1f}s")
    if spec.act_scale_mode == 1 or kv_fp8:
        calib = torch.from_numpy(wl.calibration_hidden(spec, None if spec.calib_tokens else 512)).cuda()
        model.ev_model_calibrate(calib)
        log("calibrated static scales (activations: config[4] only; K/V cache: --kv fp8)")
    pages = sum((int(L) + 64 + grow + spec.page_size - 1) // spec.page_size + 1 for L in ctx)
    cache = ev.Cache(model, pages, B)
    slots = [cache.ev_cache_add_seq(int(L) + 64 + grow) for L in ctx]
    t0 = time.time()
    cache.ev_cache_prefill(slots, [wl.context_ids(spec, b, int(ctx[b])) for b in range(B)])
    torch.cuda.synchronize()
    log(f"prefilled {int(ctx.sum())} context tokens in {time.time() - t0:.1f}s")
    # drafts: GPU greedy continuation planted on the rank-0 chain w.p. 0.7 (config[3]'s rule), else uniform ids
    depth = wl.tree_depths(parents)
    D = int(depth.max())
    n_greedy = max(D, grow)
    root = np.array([wl.draft_tokens_uniform(spec, parents, b)[0] for b in range(B)], dtype=np.int32)
    greedy = np.zeros((B, n_greedy), dtype=np.int32)
    one = ev.VerifyBuffers(model, B, 1, want_argmax=True)
    cur = root.copy()
    for d in range(n_greedy):
        one.set_inputs(slots, cur[:, None], np.full((B, 1), -1, np.int32))
        ev.ev_verify(model, cache, one, commit=True)
        torch.cuda.synchronize()
        cur = one.argmax.cpu().numpy()[:, 0].astype(np.int32)
        greedy[:, d] = cur
    cache.ev_cache_set_lens(slots, [int(L) for L in ctx])
    tokens = np.zeros((B, T), dtype=np.int32)
    planted = np.zeros(B, dtype=np.int64)     # drafts that verification must accept if it reproduces greedy decoding
    for b in range(B):
        coins = wl.gen.match_coins(spec, b, D)
        tokens[b] = plant(spec, parents, b, root[b], greedy[b], coins)
        hit = coins[:len(rank0_chain(parents))] < 0.7
        planted[b] = int(np.argmin(hit)) if not hit.all() else len(hit)
    return dict(model=model, cache=cache, slots=slots, ctx=ctx, parents=parents, tokens=tokens, greedy=greedy, root=root,
                planted=planted)


# ------------------------------------------------------------------------------------------ oracle arm

def oracle_sample(spec, steps, warmup, log):
    """Times the oracle (as it stands) on a bounded sample of the workload: one decoder layer over the
    full tree of sequence 0 per step (x n_layers), LM head once; weights from the CPU generator and a
    random bf16 KV block (values do not change the oracle's work)."""
    from oracle import verify_oracle as vo
    shape = spec.model
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else os.cpu_count()
    L = int(wl.context_lengths(spec)[0])
    parents = tree_of(spec)
    T = len(parents)
    om = vo.OracleModel(shape, act_scale_mode=0)
    t0 = time.time()
    for k in LAYER_KINDS:
        om.set_weight(k, 0, wl.weight_matrix_bf16(shape, spec.seed, k, 0))
    om.set_weight("lm_head", 0, wl.weight_matrix_bf16(shape, spec.seed, "lm_head", 0))
    log(f"oracle: quantized 1 layer + LM head in {time.time() - t0:.1f}s on {cores} cores")
    rng = np.random.default_rng(spec.seed)
    oc = vo.OracleKV(om, (L + T) // spec.page_size + 2, spec.page_size)
    oc.add_seq(0, L + T)
    dense = wl.f32_to_bf16_bits(rng.standard_normal((2, shape.n_kv_heads, L, shape.head_dim)).astype(np.float32))
    oc.import_dense(0, 0, dense)
    oc.ctx_len[0] = L
    h = (rng.standard_normal((T, shape.hidden)) * 0.02).astype(np.float32)
    t0 = time.time()
    vo.lm_head(om, h)
    t_lm = time.time() - t0
    times = []
    for i in range(warmup + steps):
        t0 = time.time()
        vo.layer_forward(om, 0, h, oc, 0, L, parents)
        if i >= warmup:
            times.append(time.time() - t0)
    t_layer = float(np.mean(times))
    # a whole step for the whole batch: every sequence runs n_layers layers + LM head
    t_step = spec.batch * (t_layer * shape.n_layers + t_lm)
    return dict(value=spec.batch * T / t_step, ms_per_step=1e3 * t_step, cores=cores,
                sample=f"1 of {shape.n_layers} decoder layers (x{shape.n_layers}) + LM head, full {T}-node tree of "
                       f"sequence 0 (x{spec.batch} sequences), context {L}; {steps} timed layer passes, "
                       f"{t_layer:.2f}s/layer, LM head {t_lm:.2f}s")


# ------------------------------------------------------------------------------------------ multi-rank host logic

def max_over_ranks(x, dist, device):
    """Replicas only: the one cross-rank exchange is the MAX of a timing."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank, world, ms_per_step):
    """Aggregate throughput of `world` independent replicas that each process units_per_rank per step."""
    return world * units_per_rank / (ms_per_step * 1e-3)


# ------------------------------------------------------------------------------------------ main

def measure(spec, args, torch, ev, dist, rank, world, local_rank, log, warmup, steps, with_cpu, fp8_peak):
    """Builds the workload of one config, times `steps` verify steps (device events), the per-class pass, the end-to-end
    leg through ev_verify_host and - with --loop - the sustained closed loop.  Returns the JSON line as a dict."""
    kv_fp8 = args.kv == "fp8"
    wk = build_gpu_workload(spec, warmup + steps, torch, ev, log, loop_steps=args.loop, kv_fp8=kv_fp8, attn_chunk=args.attn_chunk)
    model, cache, slots, ctx, parents, tokens = (wk[k] for k in ("model", "cache", "slots", "ctx", "parents", "tokens"))
    B, T = tokens.shape
    L0 = [int(x) for x in ctx]
    buf = ev.VerifyBuffers(model, B, T, want_argmax=False)
    buf.set_inputs(slots, tokens, np.tile(parents, (B, 1)))

    def step():
        cache.ev_cache_set_lens(slots, L0)
        ev.ev_verify(model, cache, buf, commit=True, use_n_nodes=False)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(warmup):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev.ev_launch_count(reset=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.profiler.start()          # no-op unless run under ncu --profile-from-start off
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    torch.cuda.profiler.stop()
    barrier()
    launches = ev.ev_launch_count()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    ms = max_over_ranks(ms, dist, "cuda")
    ms_step = ms / steps
    acc = buf.accept_len.cpu().numpy()
    assert (buf.status.cpu().numpy() == 0).all(), "a sequence was rejected during the timed steps"
    # losslessness inside the bench: the drafts planted from the GPU's own greedy decode must be accepted
    assert (acc >= wk["planted"]).all(), ("tree verification did not reproduce the GPU's greedy decode", acc.tolist(), wk["planted"].tolist())

    # per-kernel-class device time over a second pass of the same K steps (CUDA events on the launch stream)
    model.ev_profile_enable(True)
    for _ in range(steps):
        step()
    prof = model.ev_profile_read()
    model.ev_profile_enable(False)
    # duration of every kernel INSIDE the graph-replayed step (the library's step trace: %globaltimer when a kernel's first CTA
    # passes griddepcontrol.wait and when its last CTA leaves); the CUDA-event class times above come from an eager pass
    # whose launches are CPU-paced
    ingraph = None
    layer_timeline = None
    try:
        model.ev_profile_enable(2)
        step(); step()
        torch.cuda.synchronize()
        model.ev_profile_trace()
        step()
        torch.cuda.synchronize()
        tr = np.asarray(model.ev_profile_trace(), dtype=np.float64)
        names = ["rmsnorm_quant", "gemm_qkv", "rope_kvwrite", "tree_attention", "attn_merge_quant", "gemm_o", "rmsnorm_quant", "gemm_gateup",
                 "swiglu_quant", "gemm_down"]
        nl = spec.model.n_layers
        if tr.shape[0] >= 10 * nl + 2:
            ex = (tr[:, 2] - tr[:, 1]) / 1e3      # us: last exit - first past-wait
            ingraph = {}
            for i in range(10 * nl):
                ingraph[names[i % 10]] = ingraph.get(names[i % 10], 0.0) + ex[i]
            ingraph["gemm_lm_head"] = ex[10 * nl + 1]
            ingraph["step_us"] = (tr[10 * nl + 1, 2] - tr[0, 0]) / 1e3
            # the ten kernels of a layer against their predecessor's last exit, averaged over the inner layers: when the first CTA
            # enters (how early programmatic dependent launch makes it resident), when the first / the last CTA passes
            # griddepcontrol.wait (a late last CTA = it could not be co-resident with the predecessor), when the last CTA leaves
            lo, hi = (2, nl - 2) if nl > 6 else (1, nl)
            tl = np.zeros((10, 4))
            for l in range(lo, hi):
                for k in range(10):
                    r, prev = tr[10 * l + k], tr[10 * l + k - 1][2]
                    tl[k] += [r[0] - prev, r[1] - prev, r[3] - prev, r[2] - prev]
            tl /= max(hi - lo, 1) * 1e3
            ph = np.zeros((10, 4))      # phase marks (only a bring-up build of the library records them: -DEV_GEMM_PROBE)
            for l in range(lo, hi):
                for k in range(10):
                    ph[k] += tr[10 * l + k][4:8] - tr[10 * l + k - 1][2]
            ph /= max(hi - lo, 1) * 1e3
            layer_timeline = {"kernels": ["rmsnorm1_quant", "gemm_qkv", "rope_kvwrite", "tree_attention", "attn_merge_quant", "gemm_o",
                                          "rmsnorm2_quant", "gemm_gateup", "swiglu_quant", "gemm_down"],
                              "us_after_predecessor_exit": {key: [round(float(v), 2) if abs(v) < 1e6 else None for v in tl[:, col]]   # None: the kernel does not record that mark
                                                            for col, key in enumerate(("first_cta_enters", "first_cta_past_wait", "last_cta_past_wait", "last_cta_exits"))},
                              "layer_us": round(float(tl[:, 3].sum()), 2), "layers_averaged": [lo, hi]}
            if (np.abs(ph) < 1e6).any():
                layer_timeline["gemm_phase_marks_last_cta"] = {
                    "def": "activations requested, first stage complete, first accumulator complete, epilogue holds it (us after the predecessor's last exit)",
                    **{layer_timeline["kernels"][k]: [round(float(v), 2) for v in ph[k]] for k in range(10) if (np.abs(ph[k]) < 1e6).all()}}
    except Exception as e:  # pragma: no cover
        log(f"step trace unavailable: {e}")
    model.ev_profile_enable(0)
    work = algorithmic_work(spec, ctx, parents, kv_fp8)
    pk = peaks()
    gemm_ms = sum(v[0] for k, v in prof.items() if k.startswith("gemm_"))
    gemm_n = sum(v[1] for k, v in prof.items() if k.startswith("gemm_"))
    per_launch_us = {k: round(1e3 * v[0] / max(v[1], 1), 2) for k, v in prof.items()}
    attn_ms, attn_n = prof["tree_attention"]
    share = {k: round(v[0] / max(sum(x[0] for x in prof.values()), 1e-9), 4) for k, v in prof.items()}
    gemm_gbs = work["weight_bytes"] * steps / (gemm_ms * 1e-3) / 1e9
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        traffic = json.load(open(tpath)).get(spec.name, {}).get("gemm_dram_bytes_per_launch")
    peak_src = pk["source"] + " (MEASURED_PEAKS.json hbm_gbs)" if pk["source"] == "measured" else "fallback (B200_PROFILING.md)"
    lin_flops = B * T * spec.model.linear_flops_per_token()
    hbm_bound = work["weight_bytes"] / (pk["hbm_gbs"] * 1e9) >= lin_flops / fp8_peak[0]
    if hbm_bound:     # few rows: the GEMMs stream the weights once per step
        roofline = {"bound": "hbm", "kernel": "gemm_e4m3_kernel (tcgen05 FP8 W8A8 linears)", "achieved": round(gemm_gbs, 1),
                    "peak": pk["hbm_gbs"], "peak_source": peak_src, "unit": "GB/s", "frac": round(gemm_gbs / pk["hbm_gbs"], 4),
                    "bytes_per_launch": work["weight_bytes"] / (gemm_n / steps)}
    else:             # many rows: the same kernels are bound by the FP8 tensor pipe
        tf = lin_flops * steps / (gemm_ms * 1e-3) / 1e12
        roofline = {"bound": "tensor", "kernel": "gemm_e4m3_kernel (tcgen05 FP8 W8A8 linears)", "achieved": round(tf, 1),
                    "peak": round(fp8_peak[0] / 1e12, 1), "peak_source": fp8_peak[1], "unit": "TFLOP/s", "frac": round(tf * 1e12 / fp8_peak[0], 4),
                    "flops_per_launch": lin_flops / (gemm_n / steps)}
    if attn_ms > gemm_ms:   # long contexts: the attention kernel, not the GEMMs, is the dominant kernel - bound by the KV stream
        kv_gbs = work["kv_bytes"] * steps / (attn_ms * 1e-3) / 1e9
        roofline = {"bound": "hbm", "kernel": "tree_attn_tc_kernel (tcgen05 tree attention over the paged KV cache)", "achieved": round(kv_gbs, 1),
                    "peak": pk["hbm_gbs"], "peak_source": peak_src, "unit": "GB/s", "frac": round(kv_gbs / pk["hbm_gbs"], 4),
                    "bytes_per_launch": work["kv_bytes"] / (attn_n / steps), "gemm_frac_of_its_own_bound": roofline["frac"]}
        gemm_n, gemm_ms = attn_n, attn_ms
    if ingraph is not None:
        g_us = sum(v for k, v in ingraph.items() if k.startswith("gemm_"))
        roofline["in_graph"] = {"us_per_step_by_class": {k: round(v, 1) for k, v in ingraph.items()},
                                "gemm_gbs": round(work["weight_bytes"] / (g_us * 1e-6) / 1e9, 1),
                                "gemm_frac_of_hbm": round(work["weight_bytes"] / (g_us * 1e-6) / 1e9 / pk["hbm_gbs"], 4),
                                "gemm_tflops": round(lin_flops / (g_us * 1e-6) / 1e12, 1),
                                "layer_timeline": layer_timeline,
                                "def": "per-kernel durations inside the CUDA-graph replay (step trace: first CTA past griddepcontrol.wait -> last CTA exit, "
                                       "%globaltimer), summed per class over one step; the event-timed `achieved` above is from an eager, CPU-paced pass"}
    roofline.update({"launches_per_step": gemm_n // steps, "avg_launch_us": round(1e3 * gemm_ms / gemm_n, 2), "traffic": traffic,
                     "time_share_by_class": share, "avg_launch_us_by_class": per_launch_us})
    t_roof = max((work["weight_bytes"] + work["kv_bytes"]) / (pk["hbm_gbs"] * 1e9), work["flops"] / fp8_peak[0])

    # end to end: host (pinned) buffers through the C ABI, copies inside the timed region
    host = {k: torch.empty(s, dtype=torch.int32).pin_memory() for k, s in
            dict(seq_slots=(B,), tokens=(B, T), parents=(B, T), accept_len=(B,), accept_nodes=(B, T), out_tokens=(B, T),
                 new_ctx_len=(B,), status=(B,)).items()}
    host["seq_slots"].copy_(torch.tensor(slots, dtype=torch.int32))
    host["tokens"].copy_(torch.from_numpy(tokens))
    host["parents"].copy_(torch.from_numpy(np.tile(parents, (B, 1)).astype(np.int32)))
    for _ in range(3):
        cache.ev_cache_set_lens(slots, L0)
        ev.ev_verify_host(model, cache, host)
    barrier()
    t0 = time.perf_counter()
    for _ in range(steps):
        cache.ev_cache_set_lens(slots, L0)
        ev.ev_verify_host(model, cache, host)      # synchronises internally
    e2e_ms = 1e3 * (time.perf_counter() - t0)
    e2e_ms = max_over_ranks(e2e_ms, dist, "cuda")
    assert np.array_equal(host["accept_len"].numpy(), acc)
    emitted = int((acc + 1).sum())

    # sustained closed loop (--loop K): commit = 1, no rewind, every sequence advances by its own a + 1 per step; the drafts
    # of the next step are planted (p = 0.7 per depth) from the greedy stream at the position the sequence has reached -
    # the role a drafter plays - on the host, between steps, inside the timed region; results come back through
    # ev_verify_host, which also tells the library the true new lengths.
    loop = None
    if args.loop > 0:
        greedy, D = wk["greedy"], int(wl.tree_depths(parents).max())
        rng = np.random.default_rng(spec.seed + 991)
        base = [wl.draft_tokens_uniform(spec, parents, b) for b in range(B)]      # the uniform part of the drafts, drawn once
        # the "drafter" of this loop: for every position a sequence can reach, the tree it would be handed there (greedy
        # continuation planted with p = 0.7 per depth) - built before the timed region, looked up inside it
        n_pos = args.loop * (D + 1) + 1
        table = [[plant(spec, parents, b, 0, greedy[b, p:p + D], rng.random(D), base[b]) for p in range(n_pos)] for b in range(B)]
        cache.ev_cache_set_lens(slots, L0)
        pos = np.zeros(B, dtype=np.int64)           # tokens emitted so far
        root = wk["root"].copy()
        tot_emit = tot_acc = 0
        caps_at = []
        barrier()
        ev.ev_capture_count(reset=True)
        t0 = time.perf_counter()
        for s in range(args.loop):
            tk = np.stack([table[b][pos[b]] for b in range(B)])
            tk[:, 0] = root
            host["tokens"].copy_(torch.from_numpy(tk))
            ev.ev_verify_host(model, cache, host)
            a = host["accept_len"].numpy().astype(np.int64)
            out = host["out_tokens"].numpy()
            assert (host["status"].numpy() == 0).all()
            for b in range(B):
                assert out[b, :a[b] + 1].tolist() == greedy[b, pos[b]:pos[b] + a[b] + 1].tolist(), "sustained loop left the greedy sequence"
                root[b] = out[b, a[b]]
            pos += a + 1
            tot_emit += int((a + 1).sum())
            tot_acc += int(a.sum())
            if ev.ev_capture_count(reset=True):
                caps_at.append(s)
        loop_ms = 1e3 * (time.perf_counter() - t0)
        loop_ms = max_over_ranks(loop_ms, dist, "cuda")
        loop = {"steps": args.loop, "ms_per_step": round(loop_ms / args.loop, 4),
                "tree_tokens_per_s": round(whole_job_rate(B * T, world, loop_ms / args.loop), 1),
                "emitted_tokens_per_s": round(world * tot_emit / (loop_ms * 1e-3), 1),
                "accepted_tokens_per_s": round(world * tot_acc / (loop_ms * 1e-3), 1),
                "mean_emitted_per_step": round(tot_emit / (B * args.loop), 3), "graph_captures_at_steps": caps_at,
                "vs_rewound_e2e": round((e2e_ms / steps) / (loop_ms / args.loop), 4),
                "def": "commit=1, no rewind, ctx advances by a+1; the next step's drafts (greedy continuation planted with p = 0.7, precomputed per "
                       "position) are looked up on the host between steps, inside the timed region; every emitted token checked against the greedy stream"}
    if rank != 0:
        return None
    # static scales (config[4]): the clip rate PAPER.md:140 reports, from the quantizers' own counters over one step
    clip = None
    if spec.act_scale_mode == 1:
        model.ev_model_get_clip_counts(reset=True)
        step()
        torch.cuda.synchronize()
        cc = model.ev_model_get_clip_counts(reset=True)
        sh = spec.model
        per_layer = B * T * (2 * sh.hidden + sh.n_q_heads * sh.head_dim + sh.ffn)   # qkv_in, gateup_in, o_in, down_in
        n_el = sh.n_layers * per_layer + B * T * sh.hidden
        clip = {"clipped": int(cc.sum()), "quantized_elements": int(n_el), "rate": float(cc.sum()) / n_el,
                "def": "activation elements with |x| > 448 * s_site over one verify step (PAPER.md:140)"}
    cpu = None
    if with_cpu and world == 1:
        r = oracle_sample(spec, 4, 1, log)
        cpu = {"value": round(r["value"], 3), "unit": "tree-tokens/s", "cores": r["cores"], "kind": "oracle", "sample": r["sample"]}
    line = {
        "metric": METRIC, "value": round(whole_job_rate(B * T, world, ms_step), 1), "unit": "tree-tokens/s", "n_gpus": world,
        "steps": steps, "warmup": warmup, "ms_per_step": round(ms_step, 4), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": f"e4m3 x e4m3 -> f32 ({'E4M3' if kv_fp8 else 'bf16'} KV, f32 residual)", "data": "synthetic",
        "config": {"workload": spec.name, "batch_per_gpu": B, "tree_nodes": T, "context": L0 if B <= 4 else [min(L0), max(L0)],
                   "cache_state": "cold: 7.5 GB of weights + KV exceed the 126 MB L2 every step", "replicas": world,
                   "attn_chunk": args.attn_chunk or "library default for this max_batch (ev_config.attn_chunk = 0: 256 keys for <= 2 sequences, 2048 below 16, else 4096)",
                   "kv_cache": "E4M3, static per-tensor scales (PAPER.md:98; ev_config.kv_dtype = 1)" if kv_fp8 else "bf16 (BASELINE.json configs)"},
        "accepted_tokens_per_s": round(world * int(acc.sum()) / (ms_step * 1e-3), 1),
        "emitted_tokens_per_s": round(world * emitted / (ms_step * 1e-3), 1),
        "mean_emitted_per_step": round(emitted / B, 3),
        "planted_emitted_per_step": round(float((wk["planted"] + 1).mean()), 3),
        "step_roofline": {"ideal_ms": round(1e3 * t_roof, 4), "frac": round(1e3 * t_roof / ms_step, 4),
                          "def": "max((weight+KV bytes)/HBM, FLOPs/FP8 peak)", "fp8_peak_tflops": round(fp8_peak[0] / 1e12, 1),
                          "fp8_peak_source": fp8_peak[1], "hbm_gbs": pk["hbm_gbs"],
                          "weight_bytes": work["weight_bytes"], "kv_bytes": work["kv_bytes"], "flops": work["flops"]},
        "roofline": roofline,
        "cpu_baseline": cpu,
        "e2e": {"value": round(whole_job_rate(B * T, world, e2e_ms / steps), 1), "unit": "tree-tokens/s",
                "ms_per_step": round(e2e_ms / steps, 4), "h2d_bytes_per_step": (2 * B * T + B) * 4,
                "d2h_bytes_per_step": (2 * B * T + 3 * B) * 4},
        "gpu_launches": int(launches), "clocks": clocks,
        "attention": {"ms_per_step": round(attn_ms / steps, 4), "kv_gbs": round(work["kv_bytes"] * steps / max(attn_ms, 1e-9) / 1e6, 1)},
    }
    if loop is not None:
        line["sustained_loop"] = loop
    if clip is not None:
        line["clip_rate"] = clip
    del buf, cache, model
    torch.cuda.empty_cache()
    return line


def engine_leg(spec, args, torch, ev, log):
    """Serving shell with the draft side (8(f)-3): B requests with the config's prompts run
    through ev_engine - continuous batching around verify - as plain decoding (one node per sequence), with the EAGLE-style
    drafter proposing a chain of k = 3, and with it proposing the config's tree (the chain-vs-tree trade-off is
    drafting + verification overhead against accepted length; the drafter here has random weights, so its acceptance is ~0 and
    the figures are the overhead side of that trade-off)."""
    shape = spec.model
    B = min(spec.batch, args.engine_batch)
    ctx = wl.context_lengths(spec)[:B]
    new_tokens = args.engine_steps * 8
    max_ctx = int(ctx.max()) + new_tokens + 80
    target = ev.Model(shape, max_batch=B, max_tree_nodes=64, max_ctx=max_ctx, page_size=spec.page_size)
    for kind, layer in [("embed", 0)] + [(k, l) for l in range(shape.n_layers) for k in LAYER_KINDS] + [("lm_head", 0)]:
        target.ev_model_set_weight(kind, layer, wl.weight_matrix_bf16(shape, spec.seed, kind, layer, device="cuda"))
    import dataclasses
    dshape = dataclasses.replace(shape, name=shape.name + "_drafter", n_layers=1)
    drafter = ev.Model(dshape, max_batch=B, max_tree_nodes=64, max_ctx=max_ctx, page_size=spec.page_size)
    for k in LAYER_KINDS:
        drafter.ev_model_set_weight(k, 0, wl.weight_matrix_bf16(shape, spec.seed, k, shape.n_layers, device="cuda"))
    drafter.ev_model_set_weight("d_fc", 0, wl.weight_matrix_bf16(shape, spec.seed, "d_fc", 0, device="cuda"))
    ev.ev_model_share_head(drafter, target)
    pages = sum((int(L) + new_tokens + 80) // spec.page_size + 2 for L in ctx)
    out = {"batch": B, "context": [int(ctx.min()), int(ctx.max())], "steps": args.engine_steps,
           "def": "ev_engine_step wall time after all requests are admitted (host sync per step); drafter = 1 decoder layer + FC of the "
                  "target's shape, random weights (acceptance ~ 0: overhead side of the chain-vs-tree trade-off, PAPER.md:361-363)"}
    prompts = [wl.context_ids(spec, b, int(ctx[b])) for b in range(B)]
    for mode, parents in (("plain_decode", None), ("draft_chain_k3", wl.chain_parents(4)), ("draft_tree", tree_of(spec))):
        tcache = ev.Cache(target, pages, B)
        dcache = ev.Cache(drafter, pages, B) if parents is not None else None
        eng = ev.Engine(target, tcache, drafter if parents is not None else None, dcache, max_batch=B, parents=parents)
        rids = [eng.ev_engine_submit(p, new_tokens) for p in prompts]
        t0 = time.time()
        eng.ev_engine_step()                      # admits (prefills) every request and runs the first step
        torch.cuda.synchronize()
        t_admit = time.time() - t0
        for _ in range(3):
            eng.ev_engine_step()
        torch.cuda.synchronize()
        n0 = sum(len(eng.ev_engine_poll(r)[0]) for r in rids)
        t0 = time.perf_counter()
        for _ in range(args.engine_steps):
            eng.ev_engine_step()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        n1 = sum(len(eng.ev_engine_poll(r)[0]) for r in rids)
        T = 1 if parents is None else len(parents)
        out[mode] = {"tree_nodes": T, "ms_per_step": round(1e3 * dt / args.engine_steps, 3),
                     "emitted_tokens_per_s": round((n1 - n0) / dt, 1), "mean_emitted_per_step": round((n1 - n0) / (B * args.engine_steps), 3),
                     "admission_s": round(t_admit, 2)}
        log(f"engine {mode}: {out[mode]}")
        eng.ev_engine_destroy()
        del eng, tcache, dcache
        torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--loop", type=int, default=0, help="also run a sustained closed loop of this many committed steps")
    ap.add_argument("--kv", default="bf16", choices=["bf16", "fp8"], help="KV cache: bf16 (the configs' format) or fp8 = E4M3 (PAPER.md:98, SURVEY 8(f)-2)")
    ap.add_argument("--layers", type=int, default=0, help="override the number of decoder layers (40 = the paper's ~10B block-expanded "
                                                           "student shape, PAPER.md:76/102; SURVEY 8(f)-4)")
    ap.add_argument("--engine", action="store_true", help="also run the serving shell + draft side leg (ev_engine: plain decode, chain, tree)")
    ap.add_argument("--engine-steps", type=int, default=16)
    ap.add_argument("--engine-batch", type=int, default=32)
    ap.add_argument("--attn-chunk", type=int, default=0, help="ev_config.attn_chunk (0 = the library's default for the model's max_batch)")
    ap.add_argument("--also", default="auto", help="configs whose short line is added under 'also' (default: 2 = batch 32 "
                                                   "when the headline config 1 runs on one GPU; 'none' to skip)")
    args = ap.parse_args()
    spec = wl.CONFIGS[args.config]
    if args.layers:
        import dataclasses
        spec = dataclasses.replace(spec, name=f"{spec.name}_{args.layers}layers", model=dataclasses.replace(spec.model, name=f"{spec.model.name}_{args.layers}l", n_layers=args.layers))
    if args.impl != "reference" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # N independent replicas, one process per GPU: start them the way the driver would
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    log = lambda s: print(f"[bench r{rank}] {s}", file=sys.stderr, flush=True)  # noqa: E731
    warmup = max(args.warmup, 3)

    if args.impl == "reference":
        if rank != 0:
            return
        r = oracle_sample(spec, min(args.steps, 10), min(warmup, 2), log)
        line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": "tree-tokens/s", "n_gpus": args.gpus,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64 accumulate / f32 elementwise (E4M3 W8A8 emulated)",
                "data": "synthetic", "config": {"workload": spec.name, "batch_per_gpu": spec.batch, "tree_nodes": spec.n_nodes},
                "cpu_baseline": {"value": r["value"], "unit": "tree-tokens/s", "cores": r["cores"], "kind": "oracle",
                                 "sample": r["sample"]},
                "e2e": {"value": r["value"], "unit": "tree-tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
        print(json.dumps(line), flush=True)
        return

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback for the product path)")
    torch.cuda.set_device(local_rank)
    import paper_2606_18502_b200 as ev
    from paper_2606_18502_b200 import build
    build.build()
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    fp8_peak = fp8_peak_probe(torch)
    log(f"FP8 tensor peak: {fp8_peak[0] / 1e12:.0f} TFLOP/s ({fp8_peak[1]})")
    line = measure(spec, args, torch, ev, dist, rank, world, local_rank, log, warmup, args.steps, not args.no_cpu_baseline, fp8_peak)
    also = [2] if (args.also == "auto" and args.config == 1 and world == 1) else \
        [int(x) for x in args.also.split(",") if x.strip().isdigit()] if args.also not in ("auto", "none") else []
    if also:   # north_star names batch 1 AND batch 32: the batch-32 config rides along as a short line
        args.loop = 0
        extra = {}
        for c in also:
            try:
                l2 = measure(wl.CONFIGS[c], args, torch, ev, dist, rank, world, local_rank, log, 3, min(args.steps, 8), False, fp8_peak)
            except Exception as e:   # the headline line must survive a failure of the ride-along config (it is reported, not hidden)
                extra[wl.CONFIGS[c].name] = {"error": f"{type(e).__name__}: {e}"[:300]}
                continue
            if l2 is not None:
                extra[wl.CONFIGS[c].name] = {k: l2[k] for k in ("value", "unit", "ms_per_step", "steps", "config", "mean_emitted_per_step",
                                                                   "planted_emitted_per_step", "emitted_tokens_per_s", "step_roofline", "roofline", "e2e", "clocks", "attention")}
        if line is not None:
            line["also"] = extra
    if args.engine and rank == 0 and line is not None:
        try:
            line["engine"] = engine_leg(spec, args, torch, ev, log)
        except Exception as e:
            line["engine"] = {"error": f"{type(e).__name__}: {e}"[:300]}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
