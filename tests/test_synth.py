"""Seeded generators: determinism, shapes, planted structure; oracle on cfg 1 runs in seconds."""
import math
import time

import numpy as np
import torch

from oracle import sw_oracle as O
from synth import gen


def test_srht_params_deterministic():
    s1, c1 = gen.srht_params(7, 128, 64)
    s2, c2 = gen.srht_params(7, 128, 64)
    assert np.array_equal(s1, s2) and np.array_equal(c1, c2)
    assert set(np.unique(s1)) <= {-1, 1} and len(set(c1.tolist())) == 64 and (np.diff(c1) > 0).all()


def test_plant_plan_chains():
    plan = gen.plant_plan(3, 6, 64)
    for l in range(6):
        assert (plan.targets[l] < plan.queries[l]).all() and (plan.queries[l] >= 1).all()
        assert len(plan.queries[l]) == int(gen.PLANT_FRAC * 63)
    for l in range(1, 6):
        chained = np.intersect1d(plan.queries[l], plan.targets[l - 1])
        assert len(chained) >= 1


def test_planted_layer_shapes_and_structure():
    cfg = gen.CONFIGS[1]
    li = gen.layer_inputs(1, 0, seqlens=(1024,))
    assert li.Q.shape == (1024, cfg.h_q, cfg.d) and li.K.shape == (1024, cfg.h_kv, cfg.d)
    assert li.Q.dtype == torch.bfloat16
    li2 = gen.layer_inputs(1, 0, seqlens=(1024,))
    assert torch.equal(li.Q, li2.Q) and torch.equal(li.V, li2.V)
    # planted pairs show up as large block scores qbar_i . kbar_target
    plan = gen.make_plans(1, (1024,))[0]
    qb = O.block_mean(O.head_mean(gen.to_numpy_f64(li.Q)), cfg.B)
    kb = O.block_mean(O.head_mean(gen.to_numpy_f64(li.K)), cfg.B)
    S = qb @ kb.T
    for qi, ti in zip(plan.queries[0], plan.targets[0]):
        if ti == 0:
            continue
        others = np.delete(S[qi, 1:qi], ti - 1) if qi > 2 else np.zeros(1)
        assert S[qi, ti] > others.max()


def test_varlen_packing():
    li = gen.layer_inputs(4, 1, seqlens=(128, 200, 64))
    assert li.cu_seqlens.tolist() == [0, 128, 328, 392]
    assert li.Q.shape[0] == 392


def test_oracle_cfg1_full_layer_in_seconds():
    cfg = gen.CONFIGS[0]
    li = gen.layer_inputs(0, 0)
    signs, cols = gen.srht_params(1, cfg.d, cfg.r)
    H = O.srht_matrix(cfg.d, signs, cols, 1 / math.sqrt(cfg.r))
    b = O.num_blocks(cfg.seqlens[0], cfg.B)
    tau = O.tau_from_density(cfg.density, b)
    assert (b, tau) == (16, 4)
    t0 = time.time()
    out, sel = O.prefill_layer(gen.to_numpy_f64(li.Q), gen.to_numpy_f64(li.K), gen.to_numpy_f64(li.V),
                               None, B=cfg.B, H_d=H, s=cfg.s, tau=tau)
    assert time.time() - t0 < 20
    assert out.shape == (1024, 1, 64) and np.isfinite(out).all()
    assert (sel.count == np.minimum(tau, np.arange(1, b + 1))).all()
