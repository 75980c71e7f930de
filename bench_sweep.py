#!/usr/bin/env python
"""Secondary measurements of the Sketch&Walk hot path on one B200 (bench.py is the contract line; this
script fills the tables of BASELINE.md section 5 / DESIGN.md "Results"):

  cfg4   BASELINE.json configs[3]: 131072-token prefill (b = 2048), per-kernel times, roofline fraction
  cfg5   BASELINE.json configs[4]: packed 16K/32K/48K/64K batch, density x block size x s sweep;
         100 % density is the dense-attention reference built the same way (speedup column)
  paper  the paper's default operating point (s = 8, r = 64, 90 % sparsity) on cfg 2 / cfg 4 shapes

  python bench_sweep.py [--what cfg4,cfg5,paper] [--out gpurun_out/sweep.json]

Writes a JSON file and a markdown table beside it.  Inputs are the seeded planted-structure generator of
synth/gen.py; several distinct layer buffers (each >> L2) are cycled so every timed launch reads cold HBM.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch

from synth import gen
from bench import load_peaks

KERNELS = ["sketch_qk", "prefill_select", "attn"]


def tile_pairs(blocks, taus):
    return sum(sum(min(t, i + 1) for i in range(b)) for b, t in zip(blocks, taus))


def make_inputs(seed0, seqlens, h_q, h_kv, d, B, n_bufs, model_layers=32):
    plans = [gen.plant_plan(seed0 + 7919 * si, model_layers, (n + B - 1) // B) for si, n in enumerate(seqlens)]
    bufs = []
    for l in range(n_bufs):
        Qs, Ks, Vs = [], [], []
        for si, n in enumerate(seqlens):
            q, k, v = gen.planted_qkv(seed0 + l + 7919 * si, n, h_q, h_kv, d, B, torch.bfloat16,
                                      plans[si].queries[l], plans[si].targets[l], device="cuda")
            Qs.append(q); Ks.append(k); Vs.append(v)
        bufs.append(tuple(torch.cat(x) if len(x) > 1 else x[0] for x in (Qs, Ks, Vs)))
    return bufs


def time_stack(pkg, pipe, bufs, out, layers_run, passes, warm=1):
    """Per-kernel CUDA-event times (ms, mean over timed launches) of ``layers_run`` layers with the walk carried."""
    stream = torch.cuda.current_stream()

    def one_pass(events=None):
        pipe.reset()
        L = pipe.L
        for layer in range(layers_run):
            Q, K, V = bufs[layer % len(bufs)]
            ev = events[layer] if events is not None else None
            if ev is not None: ev[0].record(stream)
            pkg.sw_sketch_qk(L, Q, K, pipe.signs, pipe.cols, pipe.r, pipe.sketch_scale, pipe.qs, pipe.ks, pipe.qbar,
                             pipe.kbar)
            if ev is not None: ev[1].record(stream)
            nxt = 0 if pipe.cur < 0 else 1 - pipe.cur
            pkg.sw_prefill_select(L, pipe.qs, pipe.ks, pipe.r, pipe.s, pipe.flags, pipe.R_cur, pipe.R[nxt], pipe.W, None,
                                  pipe.tau, pipe.tau_max, pipe.idx, pipe.count, pipe.walk_ws)
            pipe.cur = nxt
            if ev is not None: ev[2].record(stream)
            pkg.sw_sparse_attn_prefill(L, Q, K, V, pipe.idx, pipe.count, pipe.tau_max, pipe.softmax_scale,
                                       pipe.flags, out, None, pipe.attn_ws)
            if ev is not None: ev[3].record(stream)

    for _ in range(warm):
        one_pass()
    torch.cuda.synchronize()
    evs = [[[torch.cuda.Event(enable_timing=True) for _ in range(len(KERNELS) + 1)] for _ in range(layers_run)]
           for _ in range(passes)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for p in range(passes):
        one_pass(evs[p])
    e1.record(stream)
    torch.cuda.synchronize()
    per = {k: [] for k in KERNELS}
    for st in evs:
        for li, ev in enumerate(st):
            if li == 0:
                continue                                    # layer 0 has no walk GEMM (R^0 = W^0): not typical
            for i, k in enumerate(KERNELS):
                per[k].append(ev[i].elapsed_time(ev[i + 1]))
    kern = {k: statistics.mean(v) for k, v in per.items()}
    layer_ms = e0.elapsed_time(e1) / (passes * layers_run)
    return kern, layer_ms


def measure(pkg, peaks, name, seqlens, bufs, *, h_q, h_kv, d, B, r, s, density, flags=None, layers_run=8, passes=2):
    signs, cols = gen.srht_params(11, d, r)
    kw = {} if flags is None else {"flags": flags}
    from bench_parts import tau_budget
    taus = [tau_budget(density, (n + B - 1) // B) for n in seqlens]
    pipe = pkg.PrefillPipeline(list(seqlens), h_q, h_kv, d, B, r, s, taus, signs, cols, **kw)
    pairs = tile_pairs(pipe.L.blocks, taus)
    pairs_dense = tile_pairs(pipe.L.blocks, pipe.L.blocks)
    out = torch.empty(sum(seqlens), h_q, d, dtype=torch.bfloat16, device="cuda")
    kern, layer_ms = time_stack(pkg, pipe, bufs, out, layers_run, passes)
    n = sum(seqlens)
    flops = 4.0 * B * B * d * h_q * pairs
    peak = peaks.get("bf16_tflops_sustained", peaks.get("bf16_tflops"))
    sel_ms = sum(kern[k] for k in KERNELS[:-1])
    sk_bytes = n * (h_q + h_kv) * d * 2
    res = {"name": name, "seqlens": list(seqlens), "block": B, "s": s, "r": r, "density": density,
           "pow_matrix": bool(flags is not None and (flags & pkg.SW_POW_MATRIX)),
           "blocks": list(pipe.L.blocks), "tau": taus, "tile_pairs": pairs, "work_fraction_of_causal_dense": pairs / pairs_dense,
           "kernel_ms": kern, "layer_ms": layer_ms, "tokens_per_s_per_layer": n / (layer_ms * 1e-3),
           "selection_ms": sel_ms, "selection_overhead_share": sel_ms / (sel_ms + kern["attn"]),
           "attn_tflops": flops / (kern["attn"] * 1e-3) / 1e12, "attn_roofline_frac": flops / (kern["attn"] * 1e-3) / 1e12 / peak,
           "attn_kernel": pkg.sw_get_prefill_kernel_used() if hasattr(pkg, "sw_get_prefill_kernel_used") else None,
           "attn_roofline_frac_of_burst": flops / (kern["attn"] * 1e-3) / 1e12 / peaks.get("bf16_tflops", peak),
           "sketch_gbs": sk_bytes / (kern["sketch_qk"] * 1e-3) / 1e9,
           "sketch_hbm_frac": sk_bytes / (kern["sketch_qk"] * 1e-3) / 1e9 / peaks.get("hbm_gbs")}
    del pipe, out
    return res


def fmt_row(r, dense=None):
    k = r["kernel_ms"]
    sp = "" if dense is None else f"{dense['kernel_ms']['attn'] / k['attn']:.2f}x / {dense['layer_ms'] / r['layer_ms']:.2f}x"
    return (f"| {r['name']} | {r['block']} | {r['s']}{'m' if r['pow_matrix'] else ''} | {100 * r['density']:.0f} % | "
            f"{100 * r['work_fraction_of_causal_dense']:.0f} % | "
            f"{k['sketch_qk']:.3f} | {k['prefill_select']:.3f} | "
            f"{k['attn']:.3f} | {r['layer_ms']:.3f} | {r['tokens_per_s_per_layer'] / 1e6:.2f} | "
            f"{r['attn_tflops']:.0f} ({100 * r['attn_roofline_frac']:.0f} %) | "
            f"{100 * r['selection_overhead_share']:.1f} % | {sp} |")


HEADER = ("| workload | B | s | density | work vs causal-dense | sketch ms | scores+walk+select ms | attn ms | "
          "layer ms | Mtok/s per layer | attn TFLOP/s (of sustained bf16) | selection share | speedup vs 100 % (attn / layer) |\n"
          "|---|---|---|---|---|---|---|---|---|---|---|---|---|")


def _brief(r, dense=None):
    out = {"workload": r["name"], "seqlens": r["seqlens"], "block": r["block"], "s": r["s"], "density": r["density"],
           "tau": r["tau"], "tile_pairs": r["tile_pairs"], "layer_ms": r["layer_ms"], "kernel_ms": r["kernel_ms"],
           "tokens_per_s_per_layer": r["tokens_per_s_per_layer"], "attn_tflops": r["attn_tflops"],
           "attn_roofline_frac": r["attn_roofline_frac"], "attn_roofline_frac_of_burst": r["attn_roofline_frac_of_burst"],
           "selection_overhead_share": r["selection_overhead_share"]}
    if dense is not None:
        out["speedup_vs_100pct_attn"] = dense["kernel_ms"]["attn"] / r["kernel_ms"]["attn"]
        out["speedup_vs_100pct_layer"] = dense["layer_ms"] / r["layer_ms"]
    return out


def driver_points(pkg, peaks):
    """The cfg 4 / cfg 5 / paper-default points bench.py carries in its JSON line (same code as the sweep, fewer
    points): one layer stack each, 3 layers with the walk carried, 2 distinct layer buffers (each >> L2)."""
    shape = dict(h_q=32, h_kv=8, d=128)
    res = {}
    c4 = gen.CONFIGS[3]
    bufs4 = make_inputs(4000, c4.seqlens, c4.h_q, c4.h_kv, c4.d, 64, n_bufs=2)
    kw = dict(B=64, r=64, layers_run=3, passes=1, **shape)
    d100 = measure(pkg, peaks, "cfg4 128K @100% (dense reference, same kernel)", c4.seqlens, bufs4, s=2, density=1.0, **kw)
    d20 = measure(pkg, peaks, "cfg4 128K @20%", c4.seqlens, bufs4, s=2, density=0.2, **kw)
    pdef = measure(pkg, peaks, "paper default: cfg4 shape, s=8, r=64, 10% density (PAPER.md:218,266)", c4.seqlens, bufs4,
                   s=8, density=0.10, **kw)
    res["cfg4_20pct"] = _brief(d20, d100)
    res["cfg4_100pct"] = _brief(d100)
    res["paper_default"] = _brief(pdef, d100)
    del bufs4
    torch.cuda.empty_cache()
    c5 = gen.CONFIGS[4]
    bufs5 = make_inputs(5000, c5.seqlens, c5.h_q, c5.h_kv, c5.d, 64, n_bufs=2)
    e100 = measure(pkg, peaks, "cfg5 varlen 16K+32K+48K+64K @100%", c5.seqlens, bufs5, s=2, density=1.0, **kw)
    e20 = measure(pkg, peaks, "cfg5 varlen 16K+32K+48K+64K @20%", c5.seqlens, bufs5, s=2, density=0.2, **kw)
    e5 = measure(pkg, peaks, "cfg5 varlen 16K+32K+48K+64K @5%", c5.seqlens, bufs5, s=2, density=0.05, **kw)
    res["cfg5_20pct"] = _brief(e20, e100)
    res["cfg5_5pct"] = _brief(e5, e100)
    del bufs5
    torch.cuda.empty_cache()
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--what", default="cfg4,cfg5,paper")
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "sweep.json"))
    ap.add_argument("--quick", action="store_true", help="fewer sweep points (debug)")
    args = ap.parse_args()
    what = set(args.what.split(","))
    import paper_2602_07397_b200 as pkg
    assert torch.cuda.is_available(), "needs a CUDA device; there is no CPU fallback"
    peaks = load_peaks()
    results, lines = [], [HEADER]
    shape = dict(h_q=32, h_kv=8, d=128)

    if "cfg4" in what or "paper" in what:
        c4 = gen.CONFIGS[3]
        bufs4 = make_inputs(4000, c4.seqlens, c4.h_q, c4.h_kv, c4.d, 64, n_bufs=4)
        if "cfg4" in what:
            for dens in ([0.2] if args.quick else [0.2, 1.0]):
                r = measure(pkg, peaks, "cfg4 128K", c4.seqlens, bufs4, B=64, r=64, s=2, density=dens, **shape)
                results.append(r)
            dense = results[-1] if not args.quick else None
            for r in results[-2:] if not args.quick else results[-1:]:
                lines.append(fmt_row(r, dense))
        if "paper" in what:
            base = len(results)
            for (s_, dens, fl) in [(8, 0.10, None), (8, 0.20, None), (2, 0.10, pkg.SW_DEFAULT_FLAGS | pkg.SW_POW_MATRIX)]:
                results.append(measure(pkg, peaks, "paper-default 128K", c4.seqlens, bufs4, B=64, r=64, s=s_,
                                       density=dens, flags=fl, **shape))
            for r in results[base:]:
                lines.append(fmt_row(r))
        del bufs4
        torch.cuda.empty_cache()

    if "cfg5" in what:
        c5 = gen.CONFIGS[4]
        dens_list = [0.05, 0.10, 0.20, 0.35, 0.50, 1.00]
        for B in (64, 128):
            bufs5 = make_inputs(5000, c5.seqlens, c5.h_q, c5.h_kv, c5.d, B, n_bufs=4)
            for s_ in ((2,) if args.quick else (1, 2, 3)):
                rows = []
                for dens in dens_list:
                    rows.append(measure(pkg, peaks, "cfg5 varlen 16K+32K+48K+64K", c5.seqlens, bufs5, B=B, r=64, s=s_,
                                        density=dens, layers_run=6, **shape))
                for r in rows:
                    lines.append(fmt_row(r, rows[-1]))
                results.extend(rows)
            del bufs5
            torch.cuda.empty_cache()

    os.makedirs(os.path.dirname(args.out), exist_ok=True)
    meta = {"peaks": {k: v for k, v in peaks.items() if not isinstance(v, dict)}, "gpu": torch.cuda.get_device_name(0),
            "generator": {"coherence_a": gen.COHERENCE_A, "plant_cos": gen.PLANT_COS, "plant_frac": gen.PLANT_FRAC,
                          "chain_frac": gen.CHAIN_FRAC, "sink_a": gen.SINK_A},
            "timing": "CUDA events per call on the launching stream, mean over layers 1.. of 2 passes after 1 warm-up pass; "
                      "4 distinct layer buffers cycled (each >> 126 MB L2)"}
    json.dump({"meta": meta, "results": results}, open(args.out, "w"), indent=1)
    md = args.out[:-5] + ".md"
    with open(md, "w") as f:
        f.write("# Sweep results (bench_sweep.py)\n\nCommand: `python bench_sweep.py --what " + args.what + "`\n\n")
        f.write(f"GPU: {meta['gpu']}; peaks: {json.dumps(meta['peaks'])}\n\n{meta['timing']}\n\n")
        f.write("`s` with suffix `m` = matrix-power reading (SW_POW_MATRIX, P4).\n\n")
        f.write("\n".join(lines) + "\n")
    print("\n".join(lines))


if __name__ == "__main__":
    main()
