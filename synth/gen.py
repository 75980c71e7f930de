"""Seeded synthetic inputs shaped like the paper's workloads.

This module serves BOTH the CPU oracle (via tests / bench cpu_baseline) and the CUDA
path.  It holds none of the method's arithmetic: only random draws, the planted
block structure and the configuration table of BASELINE.json.  Random numbers the
method itself draws (the SRHT signs and sampled columns) are drawn
here and passed to both sides as inputs.

The paper evaluates on LongBench / RULER prompts through Llama / Qwen models
(PAPER.md:196-200); neither datasets nor weights exist here, so these inputs stand in
for them: Llama-3-8B attention shapes, block-coherent tokens (Assumption 2.2,
PAPER.md:111-115), heavy-tailed block attention through planted (query block -> key
block) pairs that form multi-hop chains across layers, an attention
sink in block 0 and a dominant diagonal block.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np
import torch

# ---------------------------------------------------------------------------
# BASELINE.json configs (index = position in BASELINE.json "configs")
# ---------------------------------------------------------------------------
@dataclass(frozen=True)
class Config:
    name: str
    layers: int
    h_q: int
    h_kv: int
    d: int
    B: int
    r: int
    s: int
    density: float
    seqlens: Tuple[int, ...]          # prefill: tokens per sequence; decode: cache length incl. new token
    dtype: str                        # "f32" | "bf16"
    planted: bool
    decode: bool = False


CONFIGS: Dict[int, Config] = {
    0: Config("cfg1_tiny_prefill", 2, 1, 1, 64, 64, 16, 2, 0.25, (1024,), "f32", False),
    1: Config("cfg2_llama8b_prefill_32k", 32, 32, 8, 128, 64, 64, 2, 0.20, (32768,), "bf16", True),
    2: Config("cfg3_decode_b8_128k", 32, 32, 8, 128, 64, 64, 2, 0.20, (131072,) * 8, "bf16", True, True),
    3: Config("cfg4_long_prefill_128k", 32, 32, 8, 128, 64, 64, 2, 0.20, (131072,), "bf16", True),
    4: Config("cfg5_varlen_sweep_64k", 32, 32, 8, 128, 64, 64, 2, 0.20,
              (16384, 32768, 49152, 65536), "bf16", True),
}

# generator parameters (recorded in bench output)
COHERENCE_A = 0.5        # token = a*sqrt(d)*centroid + N(0, I)
PLANT_COS = 0.6          # cosine between a planted query centroid and its target key centroid
PLANT_FRAC = 0.25        # share of query blocks (i >= 1) that get a planted target
CHAIN_FRAC = 0.5         # share of layer l+1's planted blocks drawn from layer l's targets
SINK_A = 0.5             # +a*sqrt(d)*g on all Q tokens and on block 0's K tokens


def srht_params(seed: int, d: int, r: int) -> Tuple[np.ndarray, np.ndarray]:
    """Rademacher signs[d] (int8, +-1) and r distinct column indices (int32, ascending)
    sampled uniformly without replacement -- the D and S of PAPER.md:434-436."""
    rng = np.random.RandomState(seed)
    signs = (rng.randint(0, 2, size=d).astype(np.int8) * 2 - 1).astype(np.int8)
    cols = np.sort(rng.choice(d, size=r, replace=False)).astype(np.int32)
    return signs, cols


def cu_seqlens_of(seqlens: Sequence[int]) -> np.ndarray:
    return np.concatenate([[0], np.cumsum(np.asarray(seqlens, dtype=np.int64))]).astype(np.int32)


def blocks_of(seqlens: Sequence[int], B: int) -> np.ndarray:
    return np.asarray([(n + B - 1) // B for n in seqlens], dtype=np.int32)


# ---------------------------------------------------------------------------
# planted structure (small, numpy, deterministic)
# ---------------------------------------------------------------------------
@dataclass
class PlantPlan:
    """Per layer: planted query blocks and their target key blocks (target < query)."""
    queries: List[np.ndarray] = field(default_factory=list)
    targets: List[np.ndarray] = field(default_factory=list)


def plant_plan(seed: int, layers: int, b: int) -> PlantPlan:
    rng = np.random.RandomState(seed ^ 0x5EED)
    plan = PlantPlan()
    prev_targets = np.zeros((0,), dtype=np.int64)
    n_plant = int(PLANT_FRAC * max(b - 1, 0))
    for _ in range(layers):
        chosen: List[int] = []
        if n_plant > 0:
            cand_chain = np.unique(prev_targets[prev_targets >= 1])
            n_chain = min(int(CHAIN_FRAC * n_plant), cand_chain.shape[0])
            if n_chain > 0:
                chosen.extend(rng.choice(cand_chain, size=n_chain, replace=False).tolist())
            pool = np.setdiff1d(np.arange(1, b), np.asarray(chosen, dtype=np.int64))
            rest = n_plant - len(chosen)
            if rest > 0 and pool.shape[0] > 0:
                chosen.extend(rng.choice(pool, size=min(rest, pool.shape[0]), replace=False).tolist())
        q = np.sort(np.asarray(chosen, dtype=np.int64))
        t = np.asarray([rng.randint(0, qi) for qi in q], dtype=np.int64)
        plan.queries.append(q)
        plan.targets.append(t)
        prev_targets = t
    return plan


# ---------------------------------------------------------------------------
# tensors
# ---------------------------------------------------------------------------
def _torch_dtype(name: str) -> torch.dtype:
    return {"f32": torch.float32, "bf16": torch.bfloat16}[name]


def _unit(x: torch.Tensor) -> torch.Tensor:
    return x / x.norm(dim=-1, keepdim=True).clamp_min(1e-20)


def iid_qkv(seed: int, n: int, h_q: int, h_kv: int, d: int, dtype: torch.dtype,
            device: str = "cpu") -> Tuple[torch.Tensor, torch.Tensor, torch.Tensor]:
    """cfg 1: Q, K, V ~ N(0, 1) iid, layout [n, heads, d]."""
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    Q = torch.randn(n, h_q, d, generator=g, device=device, dtype=torch.float32).to(dtype)
    K = torch.randn(n, h_kv, d, generator=g, device=device, dtype=torch.float32).to(dtype)
    V = torch.randn(n, h_kv, d, generator=g, device=device, dtype=torch.float32).to(dtype)
    return Q, K, V


def planted_qkv(seed: int, n: int, h_q: int, h_kv: int, d: int, B: int, dtype: torch.dtype,
                queries: np.ndarray, targets: np.ndarray, device: str = "cpu",
                chunk_tokens: int = 16384) -> Tuple[torch.Tensor, torch.Tensor, torch.Tensor]:
    """cfg 2-5, one layer of one sequence: block-coherent tokens with planted pairs and
    a sink.  Layout [n, heads, d].  Generated chunk-wise to bound fp32 temporaries."""
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    b = (n + B - 1) // B
    cQ = _unit(torch.randn(b, d, generator=g, device=device))
    cK = _unit(torch.randn(b, d, generator=g, device=device))
    sink = _unit(torch.randn(d, generator=g, device=device))
    if len(queries) > 0:
        qi = torch.as_tensor(queries, device=device, dtype=torch.long)
        ti = torch.as_tensor(targets, device=device, dtype=torch.long)
        tgt = cK[ti]
        perp = torch.randn(len(queries), d, generator=g, device=device)
        perp = _unit(perp - (perp * tgt).sum(-1, keepdim=True) * tgt)
        cQ[qi] = PLANT_COS * tgt + math.sqrt(1.0 - PLANT_COS ** 2) * perp
    amp = COHERENCE_A * math.sqrt(d)
    muQ = amp * cQ + SINK_A * math.sqrt(d) * sink[None, :]
    muK = amp * cK
    muK[0] = muK[0] + SINK_A * math.sqrt(d) * sink
    Q = torch.empty(n, h_q, d, device=device, dtype=dtype)
    K = torch.empty(n, h_kv, d, device=device, dtype=dtype)
    V = torch.empty(n, h_kv, d, device=device, dtype=dtype)
    blk = torch.arange(n, device=device) // B
    for lo in range(0, n, chunk_tokens):
        hi = min(lo + chunk_tokens, n)
        m = hi - lo
        Q[lo:hi] = (muQ[blk[lo:hi]][:, None, :]
                    + torch.randn(m, h_q, d, generator=g, device=device)).to(dtype)
        K[lo:hi] = (muK[blk[lo:hi]][:, None, :]
                    + torch.randn(m, h_kv, d, generator=g, device=device)).to(dtype)
        V[lo:hi] = torch.randn(m, h_kv, d, generator=g, device=device).to(dtype)
    return Q, K, V


@dataclass
class LayerInputs:
    Q: torch.Tensor            # [T, h_q, d]   packed over sequences
    K: torch.Tensor            # [T, h_kv, d]
    V: torch.Tensor            # [T, h_kv, d]
    cu_seqlens: np.ndarray     # [batch + 1]


def layer_inputs(cfg_idx: int, layer: int, device: str = "cpu",
                 seqlens: Optional[Sequence[int]] = None,
                 plans: Optional[List[PlantPlan]] = None) -> LayerInputs:
    """Inputs of one layer of config ``cfg_idx`` (seed = 1000*(cfg_idx+1) + layer, plus
    7919*sequence for batches).  ``seqlens`` overrides the config's lengths (tests use
    shortened sequences with the same recipe)."""
    cfg = CONFIGS[cfg_idx]
    seqlens = tuple(cfg.seqlens if seqlens is None else seqlens)
    dt = _torch_dtype(cfg.dtype)
    Qs, Ks, Vs = [], [], []
    for si, n in enumerate(seqlens):
        seed = 1000 * (cfg_idx + 1) + layer + 7919 * si
        if cfg.planted:
            b = (n + cfg.B - 1) // cfg.B
            plan = plans[si] if plans is not None else plant_plan(1000 * (cfg_idx + 1) + 7919 * si,
                                                                   cfg.layers, b)
            q, k, v = planted_qkv(seed, n, cfg.h_q, cfg.h_kv, cfg.d, cfg.B, dt,
                                  plan.queries[layer], plan.targets[layer], device)
        else:
            q, k, v = iid_qkv(seed, n, cfg.h_q, cfg.h_kv, cfg.d, dt, device)
        Qs.append(q); Ks.append(k); Vs.append(v)
    if len(seqlens) == 1:
        Q, K, V = Qs[0], Ks[0], Vs[0]
    else:
        Q, K, V = torch.cat(Qs), torch.cat(Ks), torch.cat(Vs)
    return LayerInputs(Q, K, V, cu_seqlens_of(seqlens))


def make_plans(cfg_idx: int, seqlens: Optional[Sequence[int]] = None) -> List[PlantPlan]:
    cfg = CONFIGS[cfg_idx]
    seqlens = tuple(cfg.seqlens if seqlens is None else seqlens)
    return [plant_plan(1000 * (cfg_idx + 1) + 7919 * si, cfg.layers, (n + cfg.B - 1) // cfg.B)
            for si, n in enumerate(seqlens)]


def tile_pairs(b: int, tau: int) -> int:
    """Size of a block-causal workload: (query block, selected key block) pairs of one sequence of ``b`` blocks at
    budget ``tau`` (row i selects min(tau, i + 1) blocks).  Both bench arms scale their work by this count."""
    return sum(min(tau, i + 1) for i in range(b))


def workload_config(cfg, n: int, layers: int, b: int, tau: int) -> dict:
    """``config`` of the JSON line: what is computed, identical for the GPU arm and the reference (oracle) arm."""
    return {"workload": cfg.name if (n, layers) == (cfg.seqlens[0], cfg.layers) else f"DEBUG n={n} L={layers}",
            "layers": layers, "seq_len": n, "h_q": cfg.h_q, "h_kv": cfg.h_kv, "head_dim": cfg.d,
            "block": cfg.B, "blocks": b, "tau": tau, "sketch_dim": cfg.r, "walk_power_s": cfg.s,
            "density": cfg.density, "tile_pairs_per_layer": tile_pairs(b, tau),
            "l2": "inputs larger than L2: 32 distinct layers x 403 MB cycle through the 126 MB L2",
            "generator": {"coherence_a": COHERENCE_A, "plant_cos": PLANT_COS,
                          "plant_frac": PLANT_FRAC, "chain_frac": CHAIN_FRAC, "sink_a": SINK_A}}


def to_numpy_f64(x: torch.Tensor) -> np.ndarray:
    """Exact widening of the values handed to the GPU (bf16/fp32 -> fp64)."""
    return x.detach().to("cpu").to(torch.float64).numpy()
