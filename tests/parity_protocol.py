#!/usr/bin/env python
"""The parity protocol of SURVEY.md section 8(c)-6, run end to end for one config (needs a B200):

    python tests/parity_protocol.py --config N [--seqs 0,31] [--out gpurun_out/parity_cfgN.json]

1. NOISE FLOOR (item 1): the oracle against itself - exact accumulation (the default) vs a library fp32 GEMM
   (accum="f32") vs the same GEMM over a permuted K axis (accum="f32perm"): free-running hidden rel-L2 per layer,
   logits max|d| / sigma, argmax agreement.  This is what two honest fp32-accumulating implementations differ by.
2. FREE-RUNNING GPU vs oracle (item 4) on the same inputs, at the literal north_star tolerances (hidden rel-L2 <= 1e-2
   per layer, logits <= 2e-2 sigma, accepted tokens / compaction indices equal outside sub-1e-3 top-2 gaps): pass / fail
   per line, printed beside the noise floor.
3. The criterion SURVEY gives where the literal one is unattainable: GPU divergence <= 2 x the noise floor per layer.
config[0] additionally runs the perturbation-injection modes (`round=<site>:bf16|tf32|split16`) and both KV forms
(imported from the oracle's prefill / prefilled by the GPU).  8B configs run a stated subset of sequences (the GPU
path is batch-invariant, tests/test_gpu_8b.py, so the subset's rows are the full batch's rows); context KV is the
GPU's prefill, exported (DESIGN.md R-kv-input).  Test infrastructure: imports oracle/."""
import argparse
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, HERE)

import workloads as wl  # noqa: E402
from oracle import verify_oracle as vo  # noqa: E402
from helpers import rel_l2, LAYER_KINDS, fresh_cache, oracle_model  # noqa: E402

TOL_HIDDEN, TOL_LOGIT_SIGMA, GAP = 1e-2, 2e-2, 1e-3


def log(s):
    print(f"[protocol {time.strftime('%H:%M:%S')}] {s}", file=sys.stderr, flush=True)


def compare(ref, other):
    """ref / other: dicts with hidden (list of [T,H]), logits [T,V]."""
    sigma = float(ref["logits"].std())
    srt = np.sort(ref["logits"], axis=1)
    gap_ok = (srt[:, -1] - srt[:, -2]) >= GAP
    am_r, am_o = np.argmax(ref["logits"], axis=1), np.argmax(other["logits"], axis=1)
    return dict(hidden=[rel_l2(o, r) for o, r in zip(other["hidden"], ref["hidden"])],
                logits_maxabs_over_sigma=float(np.max(np.abs(other["logits"] - ref["logits"])) / sigma),
                argmax_agree=int((am_r == am_o).sum()), argmax_agree_outside_gaps=int((am_r == am_o)[gap_ok].sum()),
                n_outside_gaps=int(gap_ok.sum()), n_nodes=int(len(am_r)), sigma=sigma)


def oracle_run(om, oc, tokens, parents, accum="exact", rnd=""):
    om.accum = accum
    om.set_round(rnd)
    t0 = time.time()
    logits, hidden = vo.forward_tree(om, oc, 0, tokens, parents, want_hidden=True)
    om.accum = "exact"
    om.set_round("")
    log(f"  oracle accum={accum} round={rnd or '-'}: {time.time() - t0:.1f}s")
    return dict(hidden=hidden, logits=logits)


def walk_ok(ref_logits, gpu_path, gpu_out, tokens, parents):
    """accepted tokens / compaction indices vs the oracle's walk; positions after a sub-1e-3 gap are void (R-tol)."""
    am = vo.argmax_lowest(ref_logits)
    path, out = vo.accept_walk(tokens, parents, am)
    srt = np.sort(ref_logits, axis=1)
    gap_ok = (srt[:, -1] - srt[:, -2]) >= GAP
    for j in range(max(len(path), len(gpu_path))):
        node = path[j] if j < len(path) else None
        prev = path[j - 1] if j > 0 and j - 1 < len(path) else 0
        if j > 0 and not gap_ok[prev]:
            return True, "void after a sub-1e-3 gap"
        if j >= len(path) or j >= len(gpu_path) or gpu_path[j] != node:
            return False, f"path differs at {j}: oracle {path} gpu {list(gpu_path)}"
    if not gap_ok[path[-1]]:
        return True, "bonus void (gap)"
    return (list(gpu_out) == out), f"oracle out {out} gpu {list(gpu_out)}"


def run_tiny(args):
    import torch
    import paper_2606_18502_b200 as ev
    from gpu_helpers import gpu_model, import_oracle_kv, run_verify
    spec = wl.CONFIGS[0]
    om = oracle_model(spec.model, spec.seed)
    ids = wl.context_ids(spec, 0, spec.ctx_len)
    parents = wl.chain_parents(spec.n_nodes)
    toks = wl.draft_tokens_uniform(spec, parents, 0)
    oc = fresh_cache(om, 160)
    vo.prefill(om, oc, 0, ids)
    ref = oracle_run(om, oc, toks, parents)
    res = {"config": 0, "workload": spec.name, "noise_floor": {}, "injection": {}, "gpu": {}}
    for mode in ("f32", "f32perm", "f32seq"):
        # a different accumulation also changes the prefill: (i) verify only on the exact model's KV, (ii) whole pipeline
        res["noise_floor"][mode] = compare(ref, oracle_run(om, oc, toks, parents, accum=mode))
        om2 = oracle_model(spec.model, spec.seed, accum=mode)
        oc2 = fresh_cache(om2, 160)
        vo.prefill(om2, oc2, 0, ids)
        res["noise_floor"][mode + "+prefill"] = compare(ref, oracle_run(om2, oc2, toks, parents, accum=mode))
    for rnd in ("resid:bf16", "prequant:bf16", "qp:bf16", "qp:tf32", "qp:split16"):
        res["injection"][rnd] = compare(ref, oracle_run(om, oc, toks, parents, rnd=rnd))
    gm = gpu_model(spec.model, spec.seed, max_batch=1, max_tree_nodes=8, max_ctx=256)
    for form in ("imported_kv", "gpu_prefill"):
        cache = ev.Cache(gm, 16, 1)
        slot = cache.ev_cache_add_seq(160)
        if form == "imported_kv":
            import_oracle_kv(cache, slot, oc, 0, spec.ctx_len, spec.model.n_layers)
        else:
            cache.ev_cache_prefill([slot], [ids])
        buf = run_verify(gm, cache, [slot], toks[None], parents[None], commit=False)
        T = len(toks)
        gpu = dict(hidden=list(buf.hidden.cpu().numpy().reshape(spec.model.n_layers + 1, T, -1)), logits=buf.logits.cpu().numpy())
        c = compare(ref, gpu)
        a = int(buf.accept_len.cpu()[0])
        ok, why = walk_ok(ref["logits"], buf.accept_nodes.cpu().numpy()[0, :a + 1], buf.out_tokens.cpu().numpy()[0, :a + 1], toks, parents)
        c["accept_ok"], c["accept_note"] = bool(ok), why
        res["gpu"][form] = c
    return res


def run_8b(args):
    import torch
    import paper_2606_18502_b200 as ev
    from gpu_helpers import bf16_cuda_to_bits, export_kv_bits, run_verify
    spec = wl.CONFIGS[args.config]
    shape = spec.model
    ctx_all = wl.context_lengths(spec)
    seqs = [int(x) for x in args.seqs.split(",")] if args.seqs else [0]
    ctx = [int(ctx_all[b]) for b in seqs]
    B, T = len(seqs), spec.n_nodes
    parents = wl.chain_parents(T) if spec.tree_caps is None else wl.tree_parents(T, spec.tree_caps)
    model = ev.Model(shape, max_batch=B, max_tree_nodes=64, max_ctx=max(ctx) + 72, page_size=spec.page_size,
                     act_scale_mode=spec.act_scale_mode)
    om = vo.OracleModel(shape, act_scale_mode=spec.act_scale_mode)
    t0 = time.time()
    for kind, layer in [("embed", 0)] + [(k, l) for l in range(shape.n_layers) for k in LAYER_KINDS] + [("lm_head", 0)]:
        w = wl.weight_matrix_bf16(shape, spec.seed, kind, layer, device="cuda")
        model.ev_model_set_weight(kind, layer, w)
        om.set_weight(kind, layer, bf16_cuda_to_bits(w))
        del w
    log(f"weights: GPU + oracle quantized in {time.time() - t0:.0f}s")
    if spec.act_scale_mode == 1:
        # the oracle calibrates (DESIGN.md R-static); the GPU model is given the oracle's constants, so both
        # sides are ONE model (the GPU's own calibration is checked against the oracle's in tests/test_gpu_8b.py)
        t0 = time.time()
        vo.calibrate(om, wl.calibration_hidden(spec))
        sc = [om.static[(s, l)] for l in range(shape.n_layers) for s in vo.SITES] + [om.static[("lm_in", 0)]]
        model.ev_model_set_static_scales(np.asarray(sc, dtype=np.float32))
        log(f"oracle calibration: {time.time() - t0:.0f}s")
    cache = ev.Cache(model, sum((L + 64) // spec.page_size + 2 for L in ctx), B)
    slots = [cache.ev_cache_add_seq(L + 64) for L in ctx]
    cache.ev_cache_prefill(slots, [wl.context_ids(spec, b, L) for b, L in zip(seqs, ctx)])
    tokens = np.stack([wl.draft_tokens_uniform(spec, parents, b) for b in seqs])
    buf = run_verify(model, cache, slots, tokens, np.tile(parents, (B, 1)), commit=False, want_logits=True, want_hidden=True)
    assert (buf.status.cpu().numpy() == 0).all()
    hid = buf.hidden.cpu().numpy().reshape(shape.n_layers + 1, B, T, shape.hidden)
    logits = buf.logits.cpu().numpy().reshape(B, T, shape.vocab)
    acc = buf.accept_len.cpu().numpy()
    nodes, outs = buf.accept_nodes.cpu().numpy(), buf.out_tokens.cpu().numpy()
    res = {"config": args.config, "workload": spec.name, "sequences": seqs, "context": ctx, "per_sequence": []}
    for i, (b, L) in enumerate(zip(seqs, ctx)):
        log(f"sequence {b} (context {L})")
        oc = vo.OracleKV(om, (L + T) // spec.page_size + 2, spec.page_size)
        oc.add_seq(0, L + T)
        for l in range(shape.n_layers):
            oc.import_dense(l, 0, export_kv_bits(cache, slots[i], l, l + 1, L)[0])
        oc.ctx_len[0] = L
        ref = oracle_run(om, oc, tokens[i], parents)
        entry = {"seq": b, "noise_floor": {}}
        for mode in ("f32", "f32perm"):
            entry["noise_floor"][mode] = compare(ref, oracle_run(om, oc, tokens[i], parents, accum=mode))
        gpu = dict(hidden=list(hid[:, i]), logits=logits[i])
        c = compare(ref, gpu)
        a = int(acc[i])
        ok, why = walk_ok(ref["logits"], nodes[i, :a + 1], outs[i, :a + 1], tokens[i], parents)
        c["accept_ok"], c["accept_note"] = bool(ok), why
        entry["gpu"] = c
        res["per_sequence"].append(entry)
        del oc
    return res


def verdicts(c, floor=None):
    v = {"hidden_le_1e-2": bool(max(c["hidden"][1:]) <= TOL_HIDDEN), "logits_le_2e-2_sigma": bool(c["logits_maxabs_over_sigma"] <= TOL_LOGIT_SIGMA),
         "argmax_outside_gaps": bool(c["argmax_agree_outside_gaps"] == c["n_outside_gaps"])}
    if "accept_ok" in c:
        v["accepted_tokens_and_indices"] = c["accept_ok"]
    if floor is not None:
        fl = [max(a, b) for a, b in zip(floor["f32"]["hidden"], floor["f32perm"]["hidden"])]
        v["le_2x_noise_floor_per_layer"] = bool(all(g <= 2 * max(f, 1e-7) for g, f in zip(c["hidden"][1:], fl[1:])))
        v["argmax_within_noise_floor"] = bool(c["argmax_agree"] >= min(floor["f32"]["argmax_agree"], floor["f32perm"]["argmax_agree"]))
    return v


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=0)
    ap.add_argument("--seqs", default="")
    ap.add_argument("--out", default="")
    args = ap.parse_args()
    res = run_tiny(args) if args.config == 0 else run_8b(args)
    if args.config == 0:
        for form, c in res["gpu"].items():
            c["verdict"] = verdicts(c, res["noise_floor"])
    else:
        for e in res["per_sequence"]:
            e["gpu"]["verdict"] = verdicts(e["gpu"], e["noise_floor"])
            for m in e["noise_floor"].values():
                m["verdict"] = verdicts(m)
    out = args.out or f"gpurun_out/parity_cfg{args.config}.json"
    os.makedirs(os.path.dirname(out) or ".", exist_ok=True)
    json.dump(res, open(out, "w"), indent=1)
    print(json.dumps(res)[:2000])


if __name__ == "__main__":
    main()
