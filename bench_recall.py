#!/usr/bin/env python
"""Does the walk find what one-hop selection misses?  (the paper's central claim,
PAPER.md:17,154, measured on the synthetic planted structure because LongBench / RULER and the model
weights are not available here.)

The generator (synth/gen.py) plants, per layer l, pairs "query block i attends key block j" (cosine 0.6
between the block centroids) and chains: half of layer l's planted query blocks are layer l-1's targets,
so i -> j at layer l-1 and j -> k at layer l exist and only the walk state R^l = R^{l-1} W^l links i to k.
For the cfg-2 shape (32 layers x 32768 tokens, b = 512) this script runs the GPU selection path (sketch,
block scores, walk, top-tau) and reports, over layers 1..31:

  direct recall    share of planted pairs (i, j) of layer l with j in S_i^l
  two-hop recall   share of chains (i -> j at l-1, j -> k at l) with k in S_i^l
  for the walk carried across layers (the method) and for one-hop selection (R_prev = None at every layer),
  next to the share a random selection of the same size would reach.

  python bench_recall.py [--out gpurun_out/recall.json]
"""
from __future__ import annotations

import argparse
import json
import os
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

from synth import gen


def run(pkg, Qs, Ks, plan, *, n, B, r, s, density, flags, carry):
    cfg = gen.CONFIGS[1]
    signs, cols = gen.srht_params(2, cfg.d, r)
    from bench_parts import tau_budget
    pipe = pkg.PrefillPipeline([n], cfg.h_q, cfg.h_kv, cfg.d, B, r, s, [tau_budget(density, (n + B - 1) // B)], signs, cols,
                               flags=flags)
    direct = [0, 0]; hop2 = [0, 0]; rnd = []
    for l in range(len(Qs)):
        if not carry:
            pipe.reset()
        pipe.select(Qs[l], Ks[l])
        idx = pipe.idx.cpu().numpy(); cnt = pipe.count.cpu().numpy()
        sel = [set(idx[i, :cnt[i]].tolist()) for i in range(idx.shape[0])]
        if l == 0:
            continue
        for i, j in zip(plan.queries[l], plan.targets[l]):
            direct[0] += int(j in sel[i]); direct[1] += 1
        nxt = {int(q): int(t) for q, t in zip(plan.queries[l], plan.targets[l])}
        for i, j in zip(plan.queries[l - 1], plan.targets[l - 1]):
            k = nxt.get(int(j))
            if k is None or k == 0:              # block 0 is forced anyway
                continue
            hop2[0] += int(k in sel[i]); hop2[1] += 1
            rnd.append(max(0, cnt[i] - 2) / max(1, i - 1))
    del pipe
    return {"direct_recall": direct[0] / max(1, direct[1]), "pairs": direct[1],
            "two_hop_recall": hop2[0] / max(1, hop2[1]), "chains": hop2[1], "random": float(np.mean(rnd)) if rnd else None}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "recall.json"))
    ap.add_argument("--layers", type=int, default=None)
    args = ap.parse_args()
    import paper_2602_07397_b200 as pkg
    assert torch.cuda.is_available(), "needs a CUDA device; there is no CPU fallback"
    cfg = gen.CONFIGS[1]
    n, B, layers = cfg.seqlens[0], cfg.B, args.layers or cfg.layers
    plan = gen.make_plans(1, (n,))[0]
    Qs, Ks = [], []
    for l in range(layers):
        q, k, _ = gen.planted_qkv(2000 + l, n, cfg.h_q, cfg.h_kv, cfg.d, B, torch.bfloat16, plan.queries[l], plan.targets[l],
                                  device="cuda")
        Qs.append(q); Ks.append(k)
    D = pkg.SW_DEFAULT_FLAGS
    cases = [("element-wise s=1", dict(r=64, s=1, density=0.2, flags=D)),
             ("element-wise s=2 (cfg 2)", dict(r=64, s=2, density=0.2, flags=D)),
             ("element-wise s=2, 10 %", dict(r=64, s=2, density=0.1, flags=D)),
             ("element-wise s=8 (paper default)", dict(r=64, s=8, density=0.2, flags=D)),
             ("matrix power s=2", dict(r=64, s=2, density=0.2, flags=D | pkg.SW_POW_MATRIX)),
             ("raw scores s=1 (no softmax)", dict(r=64, s=1, density=0.2, flags=D & ~pkg.SW_SCORE_SOFTMAX)),
             ("element-wise s=2, r=32", dict(r=32, s=2, density=0.2, flags=D)),
             ("element-wise s=2, r=16", dict(r=16, s=2, density=0.2, flags=D))]
    rows, results = [], []
    for name, kw in cases:
        walk = run(pkg, Qs, Ks, plan, n=n, B=B, carry=True, **kw)
        one = run(pkg, Qs, Ks, plan, n=n, B=B, carry=False, **kw)
        results.append({"case": name, **{k: v for k, v in kw.items() if k != "flags"}, "flags": kw["flags"],
                        "walk": walk, "one_hop": one})
        rows.append(f"| {name} | {kw['r']} | {100 * kw['density']:.0f} % | {100 * walk['direct_recall']:.1f} % | "
                    f"{100 * one['direct_recall']:.1f} % | {100 * walk['two_hop_recall']:.1f} % | "
                    f"{100 * one['two_hop_recall']:.1f} % | {100 * walk['random']:.1f} % | {walk['pairs']} / {walk['chains']} |")
    hdr = ("| reading | r | density | direct recall, walk | direct recall, one-hop | two-hop recall, walk | "
           "two-hop recall, one-hop | random selection | pairs / chains |\n|---|---|---|---|---|---|---|---|---|")
    os.makedirs(os.path.dirname(args.out), exist_ok=True)
    meta = {"workload": f"cfg 2 shape: {layers} layers x {n} tokens, B = {B}", "gpu": torch.cuda.get_device_name(0),
            "generator": {"coherence_a": gen.COHERENCE_A, "plant_cos": gen.PLANT_COS, "plant_frac": gen.PLANT_FRAC,
                          "chain_frac": gen.CHAIN_FRAC, "sink_a": gen.SINK_A}}
    json.dump({"meta": meta, "results": results}, open(args.out, "w"), indent=1)
    with open(args.out[:-5] + ".md", "w") as f:
        f.write("# Planted-structure recall of the selection (bench_recall.py)\n\nCommand: `python bench_recall.py`\n\n"
                f"{meta['workload']}; {meta['gpu']}; generator {json.dumps(meta['generator'])}\n\n"
                "direct = planted pair (i, j) of layer l found in S_i^l; two-hop = chain i -> j (layer l-1), j -> k (layer l) "
                "with k in S_i^l; walk = R carried across layers (the method), one-hop = R_prev = None at every layer.\n\n")
        f.write(hdr + "\n" + "\n".join(rows) + "\n")
    print(hdr + "\n" + "\n".join(rows))


if __name__ == "__main__":
    main()
