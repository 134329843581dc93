#!/usr/bin/env python
"""Turns the JSON files tests/parity_protocol.py writes into the markdown report profiles/r2_parity_protocol.md:

    python tests/parity_report.py gpurun_out/parity_cfg{0,1,2,3,4}.json > profiles/r2_parity_protocol.md
"""
import json
import sys


def f(x):
    return f"{x:.1e}"


def curve(h, idx):
    return " / ".join(f(h[i]) for i in idx if i < len(h))


def main():
    print("# Round 2: parity protocol of SURVEY.md section 8(c)-6 (items 1, 4 and the 2x-noise-floor criterion)\n")
    print("Commands (B200 box; host side = the box's 16 cores):\n\n```")
    print("python tests/parity_protocol.py --config 0")
    print("python tests/parity_protocol.py --config 1\npython tests/parity_protocol.py --config 2 --seqs 0,31")
    print("python tests/parity_protocol.py --config 3 --seqs 0,63\npython tests/parity_protocol.py --config 4 --seqs 7")
    print("python tests/parity_report.py gpurun_out/parity_cfg{0,1,2,3,4}.json > profiles/r2_parity_protocol.md\n```\n")
    print("Noise floor = the ORACLE against itself: exact accumulation (default) vs a library fp32 GEMM (`f32`) vs the same GEMM over a")
    print("permuted K axis (`f32perm`) - two honest fp32 summation orders; nothing else changes.  GPU = the CUDA path, free-running,")
    print("same inputs.  rel-L2 = ||x - ref|| / ||ref|| of the residual stream after layer l over all tree nodes of the sequence;")
    print("logits: max|d| / sigma(oracle logits); argmax: nodes whose argmax equals the exact oracle's.  Literal north_star tolerances:")
    print("hidden <= 1e-2 every layer, logits <= 2e-2 sigma, accepted tokens / compaction indices equal outside sub-1e-3 top-2 gaps.")
    print("8B configs run the listed sequences (the GPU path is batch-invariant: a sequence's rows do not depend on the batch, tests/test_gpu_8b.py);")
    print("their context KV is the GPU's prefill, exported (DESIGN.md R-kv-input); config[4]: the oracle calibrates, the GPU model is given its scales.\n")
    for path in sys.argv[1:]:
        d = json.load(open(path))
        print(f"## config[{d['config']}] `{d['workload']}`\n")
        if d["config"] == 0:
            idx = [1, 2]
            print("| run | hidden rel-L2, layers 1 / 2 | logits max\\|d\\|/sigma | argmax agree |")
            print("|---|---|---|---|")
            for k, v in d["noise_floor"].items():
                print(f"| oracle {k} vs exact | {curve(v['hidden'], idx)} | {f(v['logits_maxabs_over_sigma'])} | {v['argmax_agree']}/{v['n_nodes']} |")
            for k, v in d["injection"].items():
                print(f"| oracle round={k} | {curve(v['hidden'], idx)} | {f(v['logits_maxabs_over_sigma'])} | {v['argmax_agree']}/{v['n_nodes']} |")
            for k, v in d["gpu"].items():
                print(f"| **GPU** ({k}) vs exact | {curve(v['hidden'], idx)} | {f(v['logits_maxabs_over_sigma'])} | {v['argmax_agree']}/{v['n_nodes']} |")
            print()
            for k, v in d["gpu"].items():
                vd = v["verdict"]
                print(f"* GPU, {k}: " + ", ".join(f"{n} **{'pass' if ok else 'FAIL'}**" for n, ok in vd.items()) + f" ({v['accept_note']})")
            print()
            continue
        idx = [1, 2, 4, 8, 16, 24, 32]
        print(f"sequences {d['sequences']}, contexts {d['context']}\n")
        print("| seq | run | hidden rel-L2, layers 1 / 2 / 4 / 8 / 16 / 24 / 32 | logits max\\|d\\|/sigma | argmax agree |")
        print("|---|---|---|---|---|")
        for e in d["per_sequence"]:
            for k, v in e["noise_floor"].items():
                print(f"| {e['seq']} | oracle {k} vs exact | {curve(v['hidden'], idx)} | {f(v['logits_maxabs_over_sigma'])} | {v['argmax_agree']}/{v['n_nodes']} |")
            v = e["gpu"]
            print(f"| {e['seq']} | **GPU** vs exact | {curve(v['hidden'], idx)} | {f(v['logits_maxabs_over_sigma'])} | {v['argmax_agree']}/{v['n_nodes']} |")
        print()
        for e in d["per_sequence"]:
            vd = e["gpu"]["verdict"]
            print(f"* GPU, sequence {e['seq']}: " + ", ".join(f"{n} **{'pass' if ok else 'FAIL'}**" for n, ok in vd.items()) + f" ({e['gpu']['accept_note']})")
            nf = e["noise_floor"]
            print(f"  * the oracle's own fp32 variants at the literal tolerances: " + "; ".join(
                f"{k}: hidden {'pass' if m['verdict']['hidden_le_1e-2'] else 'FAIL'}, logits {'pass' if m['verdict']['logits_le_2e-2_sigma'] else 'FAIL'}" for k, m in nf.items()))
        print()


if __name__ == "__main__":
    main()
