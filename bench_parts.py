"""Timed regions of bench.py (prefill stack = the headline; decode step = extra keys)."""
from __future__ import annotations

import math
import os
import statistics
import time

import numpy as np
import torch

from paper_2602_07397_b200.replicas import max_over_ranks, rank_seed, whole_job_throughput
from synth import gen

CFG_IDX = 1
METRIC = "prefill_tokens_per_s_per_layer_at_20pct_density"
UNIT = "tokens/s"
KERNELS = ["sketch_qk", "prefill_select", "attn"]
ROOT = os.path.dirname(os.path.abspath(__file__))


tile_pairs = gen.tile_pairs


def tau_budget(density: float, b: int) -> int:
    """The benchmark's block budget for a nominal density: the smallest whole number of blocks >= density * b, at
    least one (exact rational arithmetic on the decimal the config states).  The library takes tau as given."""
    from fractions import Fraction
    return max(1, math.ceil(Fraction(str(density)) * b))


def _ncu_traffic(kernel: str):
    """dram bytes per launch of the dominant kernel from the committed ncu summary, or None."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        import json
        return json.load(open(p)).get(kernel)
    except Exception:
        return None


def prefill_bench(pkg, args, rank, world, dist, sampler, peaks):
    cfg = gen.CONFIGS[CFG_IDX]
    n = args.seqlen or cfg.seqlens[0]
    layers = args.layers or cfg.layers
    dev = torch.device("cuda", torch.cuda.current_device())
    signs, cols = gen.srht_params(CFG_IDX + 1, cfg.d, cfg.r)
    pipe = pkg.PrefillPipeline([n], cfg.h_q, cfg.h_kv, cfg.d, cfg.B, cfg.r, cfg.s,
                               [tau_budget(cfg.density, (n + cfg.B - 1) // cfg.B)], signs, cols)
    b = pipe.L.blocks[0]
    tau = pipe.tau_max
    pairs = tile_pairs(b, tau)

    # inputs: all layers resident in HBM (32 x 403 MB), each rank its own seeds (weak scaling)
    plans = gen.make_plans(CFG_IDX, (n,))
    Qs, Ks, Vs = [], [], []
    for layer in range(layers):
        g = torch.Generator(device=dev)  # noqa: F841  (generator lives inside gen.planted_qkv)
        q, k, v = gen.planted_qkv(rank_seed(1000 * (CFG_IDX + 1) + layer, rank), n, cfg.h_q, cfg.h_kv, cfg.d, cfg.B,
                                  torch.bfloat16, plans[0].queries[layer], plans[0].targets[layer], device=str(dev))
        Qs.append(q); Ks.append(k); Vs.append(v)
    outs = [torch.empty(n, cfg.h_q, cfg.d, dtype=torch.bfloat16, device=dev) for _ in range(2)]
    torch.cuda.synchronize()
    stream = torch.cuda.current_stream()

    def step(events=None):
        pipe.reset()
        L = pipe.L
        for layer in range(layers):
            Q, K, V = Qs[layer], Ks[layer], Vs[layer]
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
                                       pipe.flags, outs[layer & 1], None, pipe.attn_ws)
            if ev is not None: ev[3].record(stream)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    if rank == 0:
        sampler.start()          # before the warm-up steps (same load): nvidia-smi needs ~0.3 s to deliver its first sample
    for _ in range(args.warmup):
        step()
    barrier()
    events = [[[torch.cuda.Event(enable_timing=True) for _ in range(len(KERNELS) + 1)] for _ in range(layers)]
              for _ in range(args.steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    launches0 = pkg.sw_launch_count()
    e0.record(stream)
    for k in range(args.steps):
        step(events[k])
    e1.record(stream)
    barrier()
    launches = pkg.sw_launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None
    ms_total = max_over_ranks(e0.elapsed_time(e1), dist, dev)
    ms_step = ms_total / args.steps
    value = whole_job_throughput(n * layers, world, ms_step * 1e-3)

    # per-kernel device times (CUDA events on the launching stream, inside the timed region)
    per = {k: [] for k in KERNELS}
    for st in events:
        for ev in st:
            for i, k in enumerate(KERNELS):
                per[k].append(ev[i].elapsed_time(ev[i + 1]))
    kern_ms = {k: statistics.mean(v) for k, v in per.items()}
    attn_ms = kern_ms["attn"]
    attn_flops = 4.0 * cfg.B * cfg.B * cfg.d * cfg.h_q * pairs          # full tile counted for the diagonal
    achieved = attn_flops / (attn_ms * 1e-3) / 1e12
    peak = peaks.get("bf16_tflops_sustained", peaks.get("bf16_tflops"))
    sel_ms = sum(kern_ms[k] for k in KERNELS[:-1])
    layer_ms = ms_step / layers
    sketch_bytes = n * (cfg.h_q + cfg.h_kv) * cfg.d * 2
    sketch_gbs = sketch_bytes / (kern_ms["sketch_qk"] * 1e-3) / 1e9

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic",
        "config": gen.workload_config(cfg, n, layers, b, tau),
        "ms_per_layer": layer_ms,
        "kernel_ms_per_layer": kern_ms,
        "kernel_ms_per_layer_median": {k: statistics.median(v) for k, v in per.items()},
        "kernel_ms_per_layer_min": {k: min(v) for k, v in per.items()},
        "selection_overhead_share": sel_ms / (sel_ms + attn_ms),
        "sketch_hbm": {"achieved_gbs": sketch_gbs, "peak_gbs": peaks.get("hbm_gbs"),
                       "frac": sketch_gbs / peaks.get("hbm_gbs")},
        "roofline": {"kernel": "sw_sparse_attn_prefill", "bound": "tensor", "achieved": achieved, "peak": peak,
                     "unit": "TFLOP/s", "frac": achieved / peak, "traffic": _ncu_traffic("sw_sparse_attn_prefill"),
                     "traffic_source": _ncu_traffic("_source"), "traffic_commit": _ncu_traffic("_commit"),
                     "peak_source": f"{peaks['_source']} bf16 sustained (kernel timed inside a long step)",
                     "frac_of_sustained": achieved / peak,
                     "frac_of_burst": achieved / peaks.get("bf16_tflops", peak), "peak_burst": peaks.get("bf16_tflops"),
                     "flops_per_launch": attn_flops, "ms_per_launch": attn_ms,
                     "whole_layer_frac": (attn_flops / peak / 1e12) / (layer_ms * 1e-3)},
        "clocks": clocks,
        "gpu_launches": launches,                  # counted by libsw (sw_launch_count) over the timed region
    }
    # with the per-block sums left behind by whatever produces Q / K (here: sw_copy_pool, untimed),
    # the sketch step is two sw_sketch_from_pooled launches and the 336 MB re-read of Q and K is gone
    qsum = torch.empty(pipe.L.total_blocks, cfg.d, device=dev); ksum = torch.empty_like(qsum)
    scratch_q = torch.empty_like(Qs[0]); scratch_k = torch.empty_like(Ks[0])
    pkg.sw_copy_pool(pipe.L, Qs[0], scratch_q, qsum); pkg.sw_copy_pool(pipe.L, Ks[0], scratch_k, ksum)
    del scratch_q, scratch_k
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    p0.record(stream)
    for _ in range(layers):
        pkg.sw_sketch_from_pooled(pipe.L, qsum, cfg.h_q, pipe.signs, pipe.cols, pipe.r, pipe.sketch_scale, pipe.qs, pipe.qbar)
        pkg.sw_sketch_from_pooled(pipe.L, ksum, cfg.h_kv, pipe.signs, pipe.cols, pipe.r, pipe.sketch_scale, pipe.ks, pipe.kbar)
    p1.record(stream)
    torch.cuda.synchronize()
    pooled_ms = p0.elapsed_time(p1) / layers
    layer_pooled = layer_ms - kern_ms["sketch_qk"] + pooled_ms
    line["sketch_from_pooled"] = {"ms_per_layer_both_tensors": pooled_ms, "ms_per_layer_whole_path": layer_pooled,
                                  "tokens_per_s_per_layer": n / (layer_pooled * 1e-3),
                                  "selection_overhead_share": (sel_ms - kern_ms["sketch_qk"] + pooled_ms) /
                                                              (sel_ms - kern_ms["sketch_qk"] + pooled_ms + attn_ms),
                                  "note": "per-block sums supplied by the producer of Q / K (sw_copy_pool, outside the timed "
                                          "region): sw_sketch_qk's re-read of Q and K is replaced by 2 x sw_sketch_from_pooled"}
    res = {"line": line, "n": n, "pipe": pipe, "Qs": Qs, "Ks": Ks, "Vs": Vs, "outs": outs}

    # ---- e2e: the same stack through the public API with HOST buffers (pinned), H2D of every layer's
    # Q/K/V and D2H of every layer's output inside the timed region, copies overlapped on a second stream
    if not args.no_e2e:
        nh = min(2, layers)
        hQ = [torch.empty(Qs[0].shape, dtype=torch.bfloat16).pin_memory() for _ in range(nh)]
        hK = [torch.empty(Ks[0].shape, dtype=torch.bfloat16).pin_memory() for _ in range(nh)]
        hV = [torch.empty(Vs[0].shape, dtype=torch.bfloat16).pin_memory() for _ in range(nh)]
        for i in range(nh):
            hQ[i].copy_(Qs[i]); hK[i].copy_(Ks[i]); hV[i].copy_(Vs[i])
        hO = torch.empty(outs[0].shape, dtype=torch.bfloat16).pin_memory()
        dQ = [torch.empty_like(Qs[0]) for _ in range(2)]
        dK = [torch.empty_like(Ks[0]) for _ in range(2)]
        dV = [torch.empty_like(Vs[0]) for _ in range(2)]
        h2d_s, d2h_s = torch.cuda.Stream(), torch.cuda.Stream()      # one stream per PCIe direction
        ready = [torch.cuda.Event() for _ in range(2)]
        freed = [torch.cuda.Event() for _ in range(2)]
        odone = [torch.cuda.Event() for _ in range(2)]

        def e2e_step():
            pipe.reset()
            for layer in range(layers):
                sl = layer & 1
                with torch.cuda.stream(h2d_s):
                    if layer >= 2:
                        h2d_s.wait_event(freed[sl])
                    dQ[sl].copy_(hQ[layer % nh], non_blocking=True)
                    dK[sl].copy_(hK[layer % nh], non_blocking=True)
                    dV[sl].copy_(hV[layer % nh], non_blocking=True)
                    ready[sl].record(h2d_s)
                stream.wait_event(ready[sl])
                if layer >= 2:
                    stream.wait_event(odone[sl])
                pipe.layer(dQ[sl], dK[sl], dV[sl], out=outs[sl])
                freed[sl].record(stream)
                with torch.cuda.stream(d2h_s):
                    d2h_s.wait_event(freed[sl])
                    hO.copy_(outs[sl], non_blocking=True)
                    odone[sl].record(d2h_s)
            h2d_s.synchronize(); d2h_s.synchronize()

        e2e_steps = max(1, min(args.steps, 2))
        e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            e2e_step()
        barrier()
        dt = (time.perf_counter() - t0) / e2e_steps
        dt = max_over_ranks(dt, dist, dev)
        h2d = layers * (Qs[0].numel() + Ks[0].numel() + Vs[0].numel()) * 2
        d2h = layers * outs[0].numel() * 2
        line["e2e"] = {"value": whole_job_throughput(n * layers, world, dt), "unit": UNIT, "h2d_bytes_per_step": h2d,
                       "d2h_bytes_per_step": d2h, "ms_per_step": dt * 1e3, "steps": e2e_steps,
                       "note": "pinned host Q/K/V -> device, every layer's output -> host; H2D and D2H on their own streams, overlapping compute"}
    return res


def decode_bench(pkg, args, peaks, n_layer_bufs: int = 4, steps: int = 20):
    """cfg 3: batch 8 x 131072-token KV cache, one new token per sequence, 20 % density.  Reports the
    per-layer decode time (selection + attention) and the attention kernel's HBM fraction over the
    selected K/V bytes.  ``n_layer_bufs`` distinct layer caches (4.3 GB each >> L2) are cycled."""
    cfg = gen.CONFIGS[2]
    dev = torch.device("cuda", torch.cuda.current_device())
    batch, t = len(cfg.seqlens), cfg.seqlens[0]
    B, d, r = cfg.B, cfg.d, cfg.r
    mb = (t + B - 1) // B
    tau = tau_budget(cfg.density, mb)
    signs, cols = gen.srht_params(3, d, r)
    free, _ = torch.cuda.mem_get_info()
    per_layer = batch * t * cfg.h_kv * d * 2 * 2 + batch * mb * mb * 4
    n_layer_bufs = max(1, min(n_layer_bufs, int(free * 0.6 // per_layer)))
    dp = pkg.DecodePipeline(batch, mb, cfg.h_q, cfg.h_kv, d, B, r, cfg.s, [tau] * batch, signs, cols)
    seqlens = torch.full((batch,), t, dtype=torch.int32, device=dev)
    layers = []
    for l in range(n_layer_bufs):
        kc = torch.empty(batch, t, cfg.h_kv, d, dtype=torch.bfloat16, device=dev)
        vc = torch.empty_like(kc)
        Wc = torch.empty(batch, mb, mb, dtype=torch.float32, device=dev)
        kbar = torch.empty(batch, mb, d, dtype=torch.float32, device=dev)
        ks = torch.empty(batch, mb, r, dtype=torch.float32, device=dev)
        q_new = torch.empty(batch, cfg.h_q, d, dtype=torch.bfloat16, device=dev)
        k_new = torch.empty(batch, cfg.h_kv, d, dtype=torch.bfloat16, device=dev)
        for s_ in range(batch):
            plan = gen.plant_plan(3000 + 7919 * s_, cfg.layers, mb)
            q, k, v = gen.planted_qkv(3000 + l + 7919 * s_, t, cfg.h_q, cfg.h_kv, d, B, torch.bfloat16,
                                      plan.queries[l], plan.targets[l], device=str(dev))
            kc[s_].copy_(k); vc[s_].copy_(v)
            q_new[s_].copy_(q[t - 1]); k_new[s_].copy_(k[t - 1])
            # caches from the prefill selection path over the first t-1 tokens (untimed set-up)
            pp = pkg.PrefillPipeline([t - 1], cfg.h_q, cfg.h_kv, d, B, r, cfg.s, [tau_budget(cfg.density, (t + B - 2) // B)],
                                     signs, cols)
            pp.select(q[:t - 1], k[:t - 1])
            Wc[s_].copy_(pp.W.view(mb, mb)); kbar[s_].copy_(pp.kbar); ks[s_].copy_(pp.ks)
            del q, k, v, pp
        layers.append((kc, vc, Wc, kbar, ks, q_new, k_new))
    torch.cuda.synchronize()
    stream = torch.cuda.current_stream()
    out = torch.empty(batch, cfg.h_q, d, dtype=torch.bfloat16, device=dev)
    n_model_layers = cfg.layers

    def one_layer(l, ev=None):
        kc, vc, Wc, kbar, ks, q_new, k_new = layers[l % n_layer_bufs]
        if ev is not None: ev[0].record(stream)
        dp.select(q_new, k_new, seqlens, kbar, ks, Wc)
        if ev is not None: ev[1].record(stream)
        dp.attend(q_new, kc, vc, seqlens, out)
        if ev is not None: ev[2].record(stream)

    def decode_step(evs=None):
        dp.reset()
        for l in range(n_model_layers):
            one_layer(l, None if evs is None else evs[l])

    for _ in range(3):
        decode_step()
    torch.cuda.synchronize()
    evs = [[[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(n_model_layers)]
           for _ in range(steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = pkg.sw_launch_count()
    e0.record(stream)
    for k in range(steps):
        decode_step(evs[k])
    e1.record(stream)
    torch.cuda.synchronize()
    launches = pkg.sw_launch_count() - launches0
    us_layer_eager = e0.elapsed_time(e1) * 1e3 / (steps * n_model_layers)
    # the decode step is launch-bound at these kernel sizes (5 launches per layer, 24 + 135 us, through
    # ctypes): capture the 32-layer step once in a CUDA graph and replay it -- the library only launches
    # on the stream it is given, never synchronises or allocates, so its calls capture as they are
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        decode_step()
    for _ in range(3):
        graph.replay()
    torch.cuda.synchronize()
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g0.record(stream)
    for k in range(steps):
        graph.replay()
    g1.record(stream)
    torch.cuda.synchronize()
    us_layer = g0.elapsed_time(g1) * 1e3 / (steps * n_model_layers)
    sel_us = statistics.mean(e[0].elapsed_time(e[1]) * 1e3 for st in evs for e in st)
    att_us = statistics.mean(e[1].elapsed_time(e[2]) * 1e3 for st in evs for e in st)
    kv_bytes = batch * tau * B * cfg.h_kv * d * 2 * 2
    gbs = kv_bytes / (att_us * 1e-6) / 1e9

    def time_graph(fn, reps):
        g_ = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g_):
            fn()
        g_.replay()
        torch.cuda.synchronize()
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record(stream)
        for _ in range(reps):
            g_.replay()
        a1.record(stream)
        torch.cuda.synchronize()
        return a0.elapsed_time(a1) * 1e3 / reps

    # ---- paged KV cache: layer 0's cache scattered into a pool of B-token pages by a random permutation ----------
    extra = {}
    try:
        kc0, vc0 = layers[0][0], layers[0][1]
        n_pages = batch * mb
        gperm = torch.Generator(device=dev); gperm.manual_seed(77)
        perm = torch.randperm(n_pages, device=dev, generator=gperm)
        kpool = torch.empty(n_pages, B, cfg.h_kv, d, dtype=torch.bfloat16, device=dev); vpool = torch.empty_like(kpool)
        kpool[perm] = kc0.view(n_pages, B, cfg.h_kv, d); vpool[perm] = vc0.view(n_pages, B, cfg.h_kv, d)
        table = perm.view(batch, mb).to(torch.int32).contiguous()
        out_p = torch.empty_like(out)
        dp.attend_paged(layers[0][5], kpool, vpool, table, seqlens, out_p)
        dp.attend(layers[0][5], kc0, vc0, seqlens, out)
        torch.cuda.synchronize()
        same = bool(torch.equal(out_p, out))
        reps = 32
        us_paged = time_graph(lambda: [dp.attend_paged(layers[0][5], kpool, vpool, table, seqlens, out_p) for _ in range(reps)], 5) / reps
        us_contig = time_graph(lambda: [dp.attend(layers[0][5], kc0, vc0, seqlens, out) for _ in range(reps)], 5) / reps
        extra["paged"] = {"attention_us_paged": us_paged, "attention_us_contiguous": us_contig,
                          "paged_over_contiguous": us_paged / us_contig, "bit_equal_to_contiguous": same,
                          "hbm_frac_paged": kv_bytes / (us_paged * 1e-6) / 1e9 / peaks.get("hbm_gbs"),
                          "pages": n_pages, "page_tokens": B,
                          "note": "same data, pages scattered by a seeded random permutation; 32 launches per graph, "
                                  "860 MB read per launch >> L2"}
        del kpool, vpool
    except Exception as e:
        extra["paged"] = {"error": repr(e)[:200]}
    # ---- 64 consecutive decode steps with growing t, across a block boundary, one CUDA graph -----------------------
    try:
        n_steps = 64
        t0s = (mb - 1) * B - 20                              # block b_q completes at step 21, a new one starts at 22
        seq_g = torch.full((batch,), t0s, dtype=torch.int32, device=dev)

        def many_steps():
            seq_g.fill_(t0s)                                  # (captured: every replay starts from the same length)
            for _ in range(n_steps):
                dp.reset()
                for l in range(n_model_layers):
                    kc, vc, Wc, kbar, ks, q_new, k_new = layers[l % n_layer_bufs]
                    dp.select(q_new, k_new, seq_g, kbar, ks, Wc)
                    dp.attend(q_new, kc, vc, seq_g, out)
                seq_g.add_(1)

        us_total = time_graph(many_steps, 1)
        seq_g.fill_(t0s)
        extra["multi_step"] = {"steps": n_steps, "t_first": t0s, "t_last": t0s + n_steps - 1,
                               "us_per_layer": us_total / (n_steps * n_model_layers),
                               "us_per_step": us_total / n_steps,
                               "hbm_frac_layer_over_kv_bytes": kv_bytes / (us_total / (n_steps * n_model_layers) * 1e-6) / 1e9 / peaks.get("hbm_gbs"),
                               "note": "64 steps x 32 layers captured once (the sequence lengths advance on the device); the "
                                       "cached W rows, key-block means and sketches are updated in place by sw_decode_select"}
    except Exception as e:
        extra["multi_step"] = {"error": repr(e)[:200]}
    return {"workload": cfg.name, **extra, "metric": "decode_us_per_step_per_layer_at_20pct_density",
            "us_per_layer": us_layer, "us_per_layer_eager": us_layer_eager,
            "launch": "one CUDA graph per 32-layer decode step (us_per_layer); eager ctypes launches (us_per_layer_eager, selection_us, attention_us)",
            "selection_us": sel_us, "attention_us": att_us,
            "hbm_frac_layer_over_kv_bytes": kv_bytes / (us_layer * 1e-6) / 1e9 / peaks.get("hbm_gbs"),
            "hbm_frac_layer_over_kv_and_w_bytes": (kv_bytes + batch * mb * mb * 2) / (us_layer * 1e-6) / 1e9 / peaks.get("hbm_gbs"),
            "selection_overhead_share": sel_us / (sel_us + att_us), "batch": batch, "kv_len": t, "tau": tau,
            "splits": pkg.sw_decode_num_splits(batch, cfg.h_kv, d, tau), "layer_buffers_cycled": n_layer_bufs,
            "steps": steps, "gpu_launches": launches,
            "roofline": {"kernel": "sw_sparse_attn_decode", "bound": "hbm", "achieved": gbs,
                         "peak": peaks.get("hbm_gbs"), "unit": "GB/s", "frac": gbs / peaks.get("hbm_gbs"),
                         "bytes_per_launch": kv_bytes, "traffic": _ncu_traffic("sw_sparse_attn_decode")}}
