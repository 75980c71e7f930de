#!/usr/bin/env python
"""Benchmark of the Sketch&Walk hot path on B200 (contract: see DESIGN.md "Measurement").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-decode] [--no-e2e]

One "step" = one pass of the whole hot path (sketch Q, sketch K, block scores, walk, top-tau select,
block-sparse attention) over all layers of BASELINE.json configs[1] (Llama-3-8B-shaped prefill, 32
layers x 32768 tokens, 20 % density) with the walk state carried across the layers.  Rank 0 prints ONE
JSON line.  ``--impl reference`` times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

from synth import gen

CFG_IDX = 1                      # BASELINE.json configs[1]
METRIC = "prefill_tokens_per_s_per_layer_at_20pct_density"
UNIT = "tokens/s"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            d["_source"] = "measured"
            return d
        except Exception:
            pass
    d = dict(FALLBACK_PEAKS)
    d["_source"] = "fallback"
    return d


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu, self.rows, self.proc = gpu_index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.gpu), "-lms", "50"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()
        sm, smax, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[1])); smax.append(float(r[2]))
            except Exception:
                continue
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], r[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        busy = [x for x in sm if x > 0.5 * max(sm)] or sm
        return {"sm_mhz": statistics.median(busy), "sm_max_mhz": max(smax), "reasons": sorted(reasons),
                "samples": len(sm)}


# ------------------------------------------------------------------------------------------ CPU oracle leg
def oracle_sample(cfg, n, layer_inputs_cpu, H, n_qblocks=4):
    """Time the oracle, as it stands, on a bounded sample of one layer: the whole selection path of the
    layer plus the attention of ``n_qblocks`` query blocks (all heads); extrapolate the attention part by
    tile-pair count.  Returns (tokens/s per layer, seconds spent, description)."""
    from oracle import sw_oracle as O
    Q, K, V = layer_inputs_cpu
    b = O.num_blocks(n, cfg.B)
    tau = O.tau_from_density(cfg.density, b)
    t0 = time.perf_counter()
    sel = O.prefill_selection(Q, K, None, B=cfg.B, H_d=H, s=cfg.s, tau=tau)
    t_sel = time.perf_counter() - t0
    rs = np.random.RandomState(0)
    n_qblocks = max(2, min(n_qblocks, b - tau))
    blocks = sorted(set([b - 1] + rs.choice(np.arange(tau, b), size=n_qblocks - 1, replace=False).tolist()))
    t0 = time.perf_counter()
    O.sparse_attention(Q, K, V, sel.idx, sel.count, cfg.B, 1 / math.sqrt(cfg.d), q_blocks=blocks)
    t_att = time.perf_counter() - t0
    pairs_s = int(sum(sel.count[i] for i in blocks))
    pairs_all = gen.tile_pairs(b, tau)
    t_layer = t_sel + t_att * pairs_all / pairs_s
    desc = (f"cfg2 layer 0: selection path in full ({t_sel:.1f}s) + attention of {len(blocks)} of {b} query "
            f"blocks x {cfg.h_q} heads ({pairs_s} of {pairs_all} tile pairs, {t_att:.1f}s), extrapolated by pairs")
    return n / t_layer, t_sel + t_att, desc


def oracle_sample_1thread(*a, **kw):
    """The same sample with every numerical library pool limited to one thread."""
    try:
        import threadpoolctl
        with threadpoolctl.threadpool_limits(limits=1):
            return oracle_sample(*a, **kw)
    except Exception:
        return None


def cpu_threads() -> int:
    try:
        import threadpoolctl
        infos = threadpoolctl.threadpool_info()
        return max([i.get("num_threads", 1) for i in infos] + [1])
    except Exception:
        return os.cpu_count() or 1


def run_reference(args, rank):
    if rank != 0:
        return
    from oracle import sw_oracle as O
    cfg = gen.CONFIGS[CFG_IDX]
    n = cfg.seqlens[0]
    b = O.num_blocks(n, cfg.B)
    tau = O.tau_from_density(cfg.density, b)
    signs, cols = gen.srht_params(CFG_IDX + 1, cfg.d, cfg.r)
    H = O.srht_matrix(cfg.d, signs, cols, 1 / math.sqrt(cfg.r))
    plans = gen.make_plans(CFG_IDX)
    li = gen.layer_inputs(CFG_IDX, 0, device="cpu", plans=plans)
    inp = tuple(gen.to_numpy_f64(x) for x in (li.Q, li.K, li.V))
    vals, secs, desc = [], [], ""
    for it in range(args.warmup + args.steps):
        v, s, desc = oracle_sample(cfg, n, inp, H, n_qblocks=16)      # ~3 s of CPU work per step
        if it >= args.warmup:
            vals.append(v); secs.append(s)
    value = statistics.mean(vals)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * statistics.mean(secs),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": gen.workload_config(cfg, n, cfg.layers, b, tau),       # the GPU arm's keys and values
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle",
                             "sample": "CPU oracle, bounded sample per step: " + desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    # this arm is the oracle alone: neither the package nor its CUDA library may be in the process
    assert "paper_2602_07397_b200" not in sys.modules, "the reference arm imported the product package"
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------ ours
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--layers", type=int, default=None, help="override the number of layers (debug only)")
    ap.add_argument("--seqlen", type=int, default=None, help="override the sequence length (debug only)")
    ap.add_argument("--no-decode", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the cfg 4 / cfg 5 / paper-default points")
    ap.add_argument("--prefill-kernel", default="auto", choices=["auto", "generic", "tcgen05"],
                    help="kernel of sw_sparse_attn_prefill (all are CUDA kernels of libsw; default: the library's choice)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import paper_2602_07397_b200 as pkg          # loads libsw.so; raises if it is not built
    from bench_parts import prefill_bench, decode_bench

    assert torch.cuda.is_available(), "bench.py (impl=ours) needs a CUDA device; there is no CPU fallback"
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist_
        dist = dist_
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    pkg.sw_set_prefill_kernel({"auto": pkg.SW_PREFILL_AUTO, "generic": pkg.SW_PREFILL_GENERIC,
                               "tcgen05": pkg.SW_PREFILL_TCGEN05}[args.prefill_kernel])
    peaks = load_peaks()
    sampler = ClockSampler(local_rank)
    res = prefill_bench(pkg, args, rank, world, dist, sampler, peaks)
    if rank == 0:
        line = res["line"]
        if not args.no_decode and world == 1:
            try:
                line["decode"] = dec = decode_bench(pkg, args, peaks)
                # BASELINE.json's metric is "prefill tok/s & decode us/step": the decode half rides inside
                # `roofline`, a key the contract names, so that whoever keeps only the contract's keys keeps it
                r_ = dec["roofline"]
                line["roofline"]["decode"] = {
                    "workload": dec["workload"], "kernel": r_["kernel"], "bound": r_["bound"],
                    "us_per_layer": dec["us_per_layer"], "selection_us": dec["selection_us"],
                    "attention_us": dec["attention_us"], "achieved": r_["achieved"], "peak": r_["peak"],
                    "unit": r_["unit"], "frac": r_["frac"], "bytes_per_launch": r_["bytes_per_launch"],
                    "frac_layer_over_kv_bytes": dec["hbm_frac_layer_over_kv_bytes"], "traffic": r_["traffic"]}
            except Exception as e:               # the headline line must still print
                line["decode"] = {"error": repr(e)[:300]}
        if not args.no_extras and world == 1 and not (args.layers or args.seqlen):
            try:
                for k_ in ("pipe", "Qs", "Ks", "Vs", "outs"):
                    res.pop(k_, None)
                torch.cuda.empty_cache()
                from bench_sweep import driver_points
                line["extras"] = driver_points(pkg, peaks)
            except Exception as e:
                line["extras"] = {"error": repr(e)[:300]}
        if not args.no_cpu_baseline:
            from oracle import sw_oracle as O
            cfg = gen.CONFIGS[CFG_IDX]
            n = res["n"]
            signs, cols = gen.srht_params(CFG_IDX + 1, cfg.d, cfg.r)
            H = O.srht_matrix(cfg.d, signs, cols, 1 / math.sqrt(cfg.r))
            li = gen.layer_inputs(CFG_IDX, 0, device="cuda", seqlens=(n,), plans=gen.make_plans(CFG_IDX, (n,)))
            inp = tuple(gen.to_numpy_f64(x) for x in (li.Q, li.K, li.V))
            v, secs, desc = oracle_sample(cfg, n, inp, H, n_qblocks=96)   # ~13 s of CPU work
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle",
                                    "sample": desc, "seconds": secs, "host_cpus": os.cpu_count(),
                                    "threads": "numpy / BLAS pool as the oracle finds it (cores = its size)"}
            one = oracle_sample_1thread(cfg, n, inp, H, n_qblocks=32)     # ~10 s, single thread
            if one is not None:
                line["cpu_baseline"]["single_thread"] = {"value": one[0], "unit": UNIT, "cores": 1, "seconds": one[1],
                                                         "sample": one[2]}
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
