"""Full-size parity: the CUDA path at BASELINE.json's sizes, in the launch configuration bench.py times
(PrefillPipeline / DecodePipeline with the config's own shapes), against the fp64 CPU oracle.

The selection path (sketch -> block scores -> walk -> top-tau) is checked IN FULL for every layer run
(cheap for the oracle: O(n h d + b^3)); attention outputs are checked on a seeded SAMPLE of
(query block, head) pairs the oracle computes one by one -- always including blocks 0, 1, tau-1, tau,
b-1 and each sequence's last block.
"""
import math

import numpy as np
import pytest
import torch

from oracle import sw_oracle as O
from synth import gen

pytestmark = pytest.mark.gpu

REL = 1e-3
ATT_MAX, ATT_MEAN = 2e-2, 2e-3


@pytest.fixture(scope="module")
def sw():
    import paper_2602_07397_b200 as pkg
    return pkg


def rowwise_close(got, ref, rel=REL):
    scale = np.abs(ref).max(axis=-1, keepdims=True)
    return bool(np.all(np.abs(got - ref) <= rel * scale + 1e-30))


def check_sets(idx_gpu, cnt_gpu, sel, R_ref, flags=O.DEFAULT_FLAGS):
    """Overlap of the selected sets; differences are only allowed at near-ties (<= 1e-3 of the row max)."""
    b = R_ref.shape[0]
    inter = tot = 0
    for i in range(b):
        g_ = set(idx_gpu[i, :cnt_gpu[i]].tolist()); o_ = set(sel.idx[i, :sel.count[i]].tolist())
        assert cnt_gpu[i] == sel.count[i]
        inter += len(g_ & o_); tot += len(o_)
        if g_ != o_:
            row = R_ref[i]; scale = np.abs(row).max()
            free = [j for j in o_ if j not in (0, i)]
            kth = min(row[free]) if free else 0.0
            for j in g_ ^ o_:
                assert abs(row[j] - kth) <= 1e-3 * scale, (i, j, row[j], kth)
    return inter / tot


def sample_blocks(b, tau, rng, extra=4):
    must = {0, min(1, b - 1), max(0, min(tau - 1, b - 1)), min(tau, b - 1), b - 1}
    pool = np.setdiff1d(np.arange(b), np.asarray(sorted(must)))
    if pool.size:
        must |= set(rng.choice(pool, size=min(extra, pool.size), replace=False).tolist())
    return sorted(must)


def run_prefill_fullsize(sw, cfg_idx, layers, *, B=None, s=None, density=None, heads=(0, 13, 31), extra_blocks=3):
    cfg = gen.CONFIGS[cfg_idx]
    B = cfg.B if B is None else B
    s = cfg.s if s is None else s
    density = cfg.density if density is None else density
    seqlens = tuple(cfg.seqlens)
    signs, cols = gen.srht_params(cfg_idx + 1, cfg.d, cfg.r)
    H = O.srht_matrix(cfg.d, signs, cols, 1 / math.sqrt(cfg.r))
    pipe = sw.PrefillPipeline(seqlens, cfg.h_q, cfg.h_kv, cfg.d, B, cfg.r, s,
                              [O.tau_from_density(density, O.num_blocks(n, B)) for n in seqlens], signs, cols)
    plans = [gen.plant_plan(1000 * (cfg_idx + 1) + 7919 * si, cfg.layers, (n + B - 1) // B)
             for si, n in enumerate(seqlens)]
    rng = np.random.RandomState(cfg_idx)
    R_ref = [None] * len(seqlens)
    overlaps = []
    for layer in range(layers):
        Qs, Ks, Vs = [], [], []
        for si, n in enumerate(seqlens):
            q, k, v = gen.planted_qkv(1000 * (cfg_idx + 1) + layer + 7919 * si, n, cfg.h_q, cfg.h_kv, cfg.d, B,
                                      torch.bfloat16, plans[si].queries[layer], plans[si].targets[layer], "cuda")
            Qs.append(q); Ks.append(k); Vs.append(v)
        Q, K, V = (torch.cat(x) if len(x) > 1 else x[0] for x in (Qs, Ks, Vs))
        del Qs, Ks, Vs
        out = pipe.layer(Q, K, V)
        torch.cuda.synchronize()
        idx_gpu, cnt_gpu = pipe.idx.cpu().numpy(), pipe.count.cpu().numpy()
        R_gpu = pipe.R_cur.cpu().numpy()
        W_gpu = pipe.W.cpu().numpy()
        qs_gpu, ks_gpu = pipe.qs.cpu().numpy(), pipe.ks.cpu().numpy()
        tlo = blo = qlo = 0
        for si, n in enumerate(seqlens):
            b = O.num_blocks(n, B)
            tau = O.tau_from_density(density, b)
            Qn = gen.to_numpy_f64(Q[tlo:tlo + n]); Kn = gen.to_numpy_f64(K[tlo:tlo + n])
            sel = O.prefill_selection(Qn, Kn, R_ref[si], B=B, H_d=H, s=s, tau=tau)
            R_ref[si] = sel.R
            assert rowwise_close(qs_gpu[blo:blo + b], sel.qs)
            assert rowwise_close(ks_gpu[blo:blo + b], sel.ks)
            assert rowwise_close(W_gpu[qlo:qlo + b * b].reshape(b, b), sel.W)
            assert rowwise_close(R_gpu[qlo:qlo + b * b].reshape(b, b), sel.R)
            ov = check_sets(idx_gpu[blo:blo + b], cnt_gpu[blo:blo + b], sel, sel.R)
            assert ov >= 0.99, ov
            overlaps.append(ov)
            # attention on sampled (query block, head) pairs, given the GPU's own lists
            Vn = gen.to_numpy_f64(V[tlo:tlo + n])
            blocks = sample_blocks(b, tau, rng, extra_blocks)
            hs = sorted(set(min(h, cfg.h_q - 1) for h in heads))
            ref = O.sparse_attention(Qn, Kn, Vn, idx_gpu[blo:blo + b], cnt_gpu[blo:blo + b], B,
                                     1 / math.sqrt(cfg.d), q_blocks=blocks, q_heads=hs)
            for i in blocks:
                lo, hi = i * B, min((i + 1) * B, n)
                got = out[tlo + lo:tlo + hi][:, hs].float().cpu().numpy()
                err = np.abs(got - ref[lo:hi][:, hs])
                assert err.max() <= ATT_MAX and err.mean() <= ATT_MEAN, (layer, si, i, err.max(), err.mean())
            del Qn, Kn, Vn, ref
            tlo += n; blo += b; qlo += b * b
        del Q, K, V, out
    return overlaps


def test_cfg2_fullsize_prefill(sw):
    """BASELINE.json configs[1]: n = 32768, b = 512, tau = 103, 3 layers with the walk carried."""
    run_prefill_fullsize(sw, 1, layers=3)


def test_cfg4_fullsize_long_prefill(sw):
    """BASELINE.json configs[3]: n = 131072, b = 2048, tau = 410, 2 layers with the walk carried."""
    run_prefill_fullsize(sw, 3, layers=2, heads=(5, 30), extra_blocks=2)


@pytest.mark.parametrize("B,s,density", [(64, 2, 0.20), (128, 3, 0.05), (64, 1, 1.0), (128, 2, 0.5)])
def test_cfg5_fullsize_varlen_sweep_points(sw, B, s, density):
    """BASELINE.json configs[4]: packed 16K/32K/48K/64K batch; four corners of the density x block x s sweep
    (100 % density doubles as the dense-attention reference)."""
    run_prefill_fullsize(sw, 4, layers=2, B=B, s=s, density=density, heads=(2, 29), extra_blocks=1)


def test_cfg3_fullsize_decode(sw):
    """BASELINE.json configs[2]: batch 8 x 131072-token KV cache, one new token, tau = 410, 2 layers with the
    walk row carried.  All 8 sequences run on the GPU exactly as bench.py's decode leg does; sequences 0 and 7
    are followed by the oracle's literal full-matrix Alg. 2 (selection) and its decode attention."""
    cfg = gen.CONFIGS[2]
    batch, t = len(cfg.seqlens), cfg.seqlens[0]
    B, d, r, s = cfg.B, cfg.d, cfg.r, cfg.s
    mb = (t + B - 1) // B
    tau = O.tau_from_density(cfg.density, mb)
    signs, cols = gen.srht_params(3, d, r)
    H = O.srht_matrix(d, signs, cols, 1 / math.sqrt(r))
    dp = sw.DecodePipeline(batch, mb, cfg.h_q, cfg.h_kv, d, B, r, s, [tau] * batch, signs, cols)
    seqlens = torch.full((batch,), t, dtype=torch.int32, device="cuda")
    checked = (0, batch - 1)
    R_full = {c: None for c in checked}
    bq = (t - 1) // B
    for layer in range(2):
        kc = torch.empty(batch, t, cfg.h_kv, d, dtype=torch.bfloat16, device="cuda")
        vc = torch.empty_like(kc)
        Wc = torch.empty(batch, mb, mb, dtype=torch.float32, device="cuda")
        kbar = torch.empty(batch, mb, d, dtype=torch.float32, device="cuda")
        ks = torch.empty(batch, mb, r, dtype=torch.float32, device="cuda")
        q_new = torch.empty(batch, cfg.h_q, d, dtype=torch.bfloat16, device="cuda")
        k_new = torch.empty(batch, cfg.h_kv, d, dtype=torch.bfloat16, device="cuda")
        pre = {}
        for s_ in range(batch):
            plan = gen.plant_plan(3000 + 7919 * s_, cfg.layers, mb)
            q, k, v = gen.planted_qkv(3000 + layer + 7919 * s_, t, cfg.h_q, cfg.h_kv, d, B, torch.bfloat16,
                                      plan.queries[layer], plan.targets[layer], device="cuda")
            kc[s_].copy_(k); vc[s_].copy_(v); q_new[s_].copy_(q[t - 1]); k_new[s_].copy_(k[t - 1])
            pp = sw.PrefillPipeline([t - 1], cfg.h_q, cfg.h_kv, d, B, r, s,
                                    [O.tau_from_density(cfg.density, O.num_blocks(t - 1, B))], signs, cols)
            pp.select(q[:t - 1], k[:t - 1])
            Wc[s_].copy_(pp.W.view(mb, mb)); kbar[s_].copy_(pp.kbar); ks[s_].copy_(pp.ks)
            if s_ in checked:                                   # oracle caches over the first t-1 tokens
                sel = O.prefill_selection(gen.to_numpy_f64(q[:t - 1]), gen.to_numpy_f64(k[:t - 1]), None, B=B, H_d=H,
                                          s=s, tau=tau)
                pre[s_] = O.DecodeCache(sel.qbar, sel.kbar, sel.S)
            del q, k, v, pp
        dp.select(q_new, k_new, seqlens, kbar, ks, Wc)
        out = dp.attend(q_new, kc, vc, seqlens)
        torch.cuda.synchronize()
        idx_gpu, cnt_gpu = dp.idx.cpu().numpy(), dp.count.cpu().numpy()
        for s_ in checked:
            sel, R_full[s_], cache2 = O.decode_layer_literal(gen.to_numpy_f64(q_new[s_]), gen.to_numpy_f64(k_new[s_]),
                                                             pre[s_], t, R_full[s_], B=B, H_d=H, s=s, tau=tau)
            ref_r = R_full[s_][bq]
            assert rowwise_close(kbar[s_].cpu().numpy(), cache2.kbar)
            assert rowwise_close(dp.rvec[dp.cur][s_, :bq + 1].cpu().numpy()[None], ref_r[None, :bq + 1])
            got = idx_gpu[s_, :cnt_gpu[s_]]
            assert cnt_gpu[s_] == len(sel) == tau and bq in got and 0 in got
            assert np.all(np.diff(got) > 0)
            diff = set(got.tolist()) ^ set(sel.tolist())
            assert len(set(got.tolist()) & set(sel.tolist())) >= 0.99 * tau
            if diff:                                             # only near-ties may differ
                thr = np.sort(ref_r[1:bq])[::-1][tau - 3]
                assert all(abs(ref_r[j] - thr) <= 1e-3 * np.abs(ref_r).max() for j in diff)
            ref = O.decode_attention(gen.to_numpy_f64(q_new[s_]), gen.to_numpy_f64(kc[s_]), gen.to_numpy_f64(vc[s_]),
                                     got, B, 1 / math.sqrt(d))
            err = np.abs(out[s_].float().cpu().numpy() - ref)
            assert err.max() <= ATT_MAX and err.mean() <= ATT_MEAN, (layer, s_, err.max(), err.mean())
        del kc, vc, Wc, kbar, ks
