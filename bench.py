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


# ------------------------------------------------------------------------------------------ workload

def tree_of(spec):
    return wl.chain_parents(spec.n_nodes) if spec.tree_caps is None else wl.tree_parents(spec.n_nodes, spec.tree_caps)


def algorithmic_work(spec, ctx_lens, parents):
    """bytes = FP8 weight bytes + KV bytes of the context; FLOPs = linear + attention."""
    m = spec.model
    depth = wl.tree_depths(parents)
    B, T = len(ctx_lens), len(parents)
    kv_bytes = m.kv_bytes_per_token() * int(np.sum(ctx_lens))
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


def build_gpu_workload(spec, steps_total, torch, ev, log):
    shape = spec.model
    B, T = spec.batch, spec.n_nodes
    parents = tree_of(spec)
    ctx = wl.context_lengths(spec)
    max_ctx = int(ctx.max()) + 64 + 8
    t0 = time.time()
    model = ev.Model(shape, max_batch=B, max_tree_nodes=64, max_ctx=max_ctx, page_size=spec.page_size,
                     act_scale_mode=spec.act_scale_mode)
    for kind, layer in [("embed", 0)] + [(k, l) for l in range(shape.n_layers) for k in LAYER_KINDS] + [("lm_head", 0)]:
        model.ev_model_set_weight(kind, layer, wl.weight_matrix_bf16(shape, spec.seed, kind, layer, device="cuda"))
    torch.cuda.synchronize()
    log(f"weights quantized in {time.time() - t0:.1f}s")
    if spec.act_scale_mode == 1:
        calib = torch.from_numpy(wl.calibration_hidden(spec)).cuda()
        model.ev_model_calibrate(calib)
        log("calibrated static activation scales")
    pages = sum((int(L) + 64 + spec.page_size - 1) // spec.page_size + 1 for L in ctx)
    cache = ev.Cache(model, pages, B)
    slots = [cache.ev_cache_add_seq(int(L) + 64) for L in ctx]
    t0 = time.time()
    cache.ev_cache_prefill(slots, [wl.context_ids(spec, b, int(ctx[b])) for b in range(B)])
    torch.cuda.synchronize()
    log(f"prefilled {int(ctx.sum())} context tokens in {time.time() - t0:.1f}s")
    # drafts: GPU greedy continuation planted on the rank-0 chain w.p. 0.7 (config[3]'s rule), else uniform ids
    depth = wl.tree_depths(parents)
    D = int(depth.max())
    root = np.array([wl.draft_tokens_uniform(spec, parents, b)[0] for b in range(B)], dtype=np.int32)
    greedy = np.zeros((B, D), dtype=np.int32)
    one = ev.VerifyBuffers(model, B, 1, want_argmax=True)
    cur = root.copy()
    for d in range(D):
        one.set_inputs(slots, cur[:, None], np.full((B, 1), -1, np.int32))
        ev.ev_verify(model, cache, one, commit=True)
        torch.cuda.synchronize()
        cur = one.argmax.cpu().numpy()[:, 0].astype(np.int32)
        greedy[:, d] = cur
    cache.ev_cache_set_lens(slots, [int(L) for L in ctx])
    tokens = np.zeros((B, T), dtype=np.int32)
    first_child = {}
    for i in range(1, T):
        first_child.setdefault(int(parents[i]), i)
    for b in range(B):
        tk = wl.draft_tokens_uniform(spec, parents, b)
        coins = wl.gen.match_coins(spec, b, D)
        node = 0
        while node in first_child:
            c = first_child[node]
            if coins[depth[c] - 1] < 0.7:
                tk[c] = greedy[b, depth[c] - 1]
            node = c
        tokens[b] = tk
    return dict(model=model, cache=cache, slots=slots, ctx=ctx, parents=parents, tokens=tokens)


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

def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    spec = wl.CONFIGS[args.config]
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
                "data": "synthetic", "config": {"workload": spec.name, "batch": spec.batch, "tree_nodes": spec.n_nodes},
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

    wk = build_gpu_workload(spec, warmup + args.steps, torch, ev, log)
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
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    torch.cuda.profiler.stop()
    barrier()
    launches = ev.ev_launch_count()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    ms = max_over_ranks(ms, dist, "cuda")
    ms_step = ms / args.steps
    acc = buf.accept_len.cpu().numpy()
    assert (buf.status.cpu().numpy() == 0).all(), "a sequence was rejected during the timed steps"

    # per-kernel-class device time over a second pass of the same K steps (CUDA events on the launch stream)
    model.ev_profile_enable(True)
    for _ in range(args.steps):
        step()
    prof = model.ev_profile_read()
    model.ev_profile_enable(False)
    work = algorithmic_work(spec, ctx, parents)
    pk = peaks()
    gemm_ms = sum(v[0] for k, v in prof.items() if k.startswith("gemm_"))
    gemm_n = sum(v[1] for k, v in prof.items() if k.startswith("gemm_"))
    per_launch_us = {k: round(1e3 * v[0] / max(v[1], 1), 2) for k, v in prof.items()}
    attn_ms, attn_n = prof["tree_attention"]
    share = {k: round(v[0] / max(sum(x[0] for x in prof.values()), 1e-9), 4) for k, v in prof.items()}
    gemm_gbs = work["weight_bytes"] * args.steps / (gemm_ms * 1e-3) / 1e9
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        traffic = json.load(open(tpath)).get(spec.name, {}).get("gemm_dram_bytes_per_launch")
    roofline = {"bound": "hbm", "kernel": "gemm_e4m3_kernel (tcgen05 FP8 W8A8 linears)", "achieved": round(gemm_gbs, 1),
                "peak": pk["hbm_gbs"], "peak_source": pk["source"] + " (MEASURED_PEAKS.json hbm_gbs)" if pk["source"] == "measured" else "fallback (B200_PROFILING.md)",
                "unit": "GB/s", "frac": round(gemm_gbs / pk["hbm_gbs"], 4),
                "bytes_per_launch": work["weight_bytes"] / (gemm_n / args.steps), "launches_per_step": gemm_n // args.steps,
                "avg_launch_us": round(1e3 * gemm_ms / gemm_n, 2), "traffic": traffic, "time_share_by_class": share,
                "avg_launch_us_by_class": per_launch_us}
    fp8_peak = 2 * pk["bf16_tflops"] * 1e12
    t_roof = max((work["weight_bytes"] + work["kv_bytes"]) / (pk["hbm_gbs"] * 1e9), work["flops"] / fp8_peak)

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
    for _ in range(args.steps):
        cache.ev_cache_set_lens(slots, L0)
        ev.ev_verify_host(model, cache, host)      # synchronises internally
    e2e_ms = 1e3 * (time.perf_counter() - t0)
    e2e_ms = max_over_ranks(e2e_ms, dist, "cuda")
    assert np.array_equal(host["accept_len"].numpy(), acc)
    emitted = int((acc + 1).sum())
    if rank != 0:
        return
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
    if not args.no_cpu_baseline and world == 1:
        r = oracle_sample(spec, 4, 1, log)
        cpu = {"value": round(r["value"], 3), "unit": "tree-tokens/s", "cores": r["cores"], "kind": "oracle", "sample": r["sample"]}
    line = {
        "metric": METRIC, "value": round(whole_job_rate(B * T, world, ms_step), 1), "unit": "tree-tokens/s", "n_gpus": world,
        "steps": args.steps, "warmup": warmup, "ms_per_step": round(ms_step, 4), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "e4m3 x e4m3 -> f32 (bf16 KV, f32 residual)", "data": "synthetic",
        "config": {"workload": spec.name, "batch_per_gpu": B, "tree_nodes": T, "context": L0 if B <= 4 else [min(L0), max(L0)],
                   "cache_state": "cold: 7.5 GB of weights + KV exceed the 126 MB L2 every step", "replicas": world},
        "accepted_tokens_per_s": round(world * int(acc.sum()) / (ms_step * 1e-3), 1),
        "emitted_tokens_per_s": round(world * emitted / (ms_step * 1e-3), 1),
        "mean_emitted_per_step": round(emitted / B, 3),
        "step_roofline": {"ideal_ms": round(1e3 * t_roof, 4), "frac": round(1e3 * t_roof / ms_step, 4),
                          "def": "max((weight+KV bytes)/HBM, FLOPs/FP8 peak); FP8 peak = 2 x measured bf16 burst",
                          "weight_bytes": work["weight_bytes"], "kv_bytes": work["kv_bytes"], "flops": work["flops"]},
        "roofline": roofline,
        "cpu_baseline": cpu,
        "e2e": {"value": round(whole_job_rate(B * T, world, e2e_ms / args.steps), 1), "unit": "tree-tokens/s",
                "ms_per_step": round(e2e_ms / args.steps, 4), "h2d_bytes_per_step": (2 * B * T + B) * 4,
                "d2h_bytes_per_step": (2 * B * T + 3 * B) * 4},
        "gpu_launches": int(launches), "clocks": clocks,
        "attention": {"ms_per_step": round(attn_ms / args.steps, 4), "kv_gbs": round(work["kv_bytes"] * args.steps / max(attn_ms, 1e-9) / 1e6, 1)},
    }
    if clip is not None:
        line["clip_rate"] = clip
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
