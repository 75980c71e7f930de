"""GPU edge cases of the C ABI: empty inputs, the launch counter, and CUDA-graph capture of the decode
step (the library launches only on the caller's stream and never synchronises or allocates)."""
import math

import numpy as np
import pytest
import torch

from oracle import sw_oracle as O
from synth import gen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sw():
    import paper_2602_07397_b200 as pkg
    return pkg


def test_empty_batch_launches_nothing_and_touches_nothing(sw):
    L = sw.make_layout([], 64)
    assert (L.batch, L.total_tokens, L.total_blocks) == (0, 0, 0)
    d, r, h_q, h_kv = 128, 64, 8, 2
    signs, cols = gen.srht_params(1, d, r)
    sg = torch.as_tensor(signs.astype(np.int8)).cuda(); cl = torch.as_tensor(cols.astype(np.int32)).cuda()
    # (NULL pointers stay an error even for an empty layout, so the dummies own one token of storage)
    x = torch.zeros(1, h_q, d, dtype=torch.bfloat16, device="cuda")
    k = torch.zeros(1, h_kv, d, dtype=torch.bfloat16, device="cuda")
    sentinel = torch.full((4, r), 7.0, device="cuda")
    idx = torch.full((4, 3), 9, dtype=torch.int32, device="cuda"); cnt = torch.full((4,), 9, dtype=torch.int32, device="cuda")
    tau = torch.zeros(1, dtype=torch.int32, device="cuda")
    n0 = sw.sw_launch_count()
    sw.sw_sketch(L, x, sg, cl, r, 1 / math.sqrt(r), sentinel, None)
    sw.sw_block_scores(L, sentinel, sentinel, r, 2, sw.SW_DEFAULT_FLAGS, sentinel, None)
    other = torch.full((4, r), 7.0, device="cuda")
    sw.sw_walk_update(L, None, sentinel, 2, sw.SW_DEFAULT_FLAGS, other, None)
    sw.sw_select_topk(L, sentinel, tau, 3, sw.SW_DEFAULT_FLAGS, idx, cnt)
    sw.sw_sparse_attn_prefill(L, x, k, k, idx, cnt, 3, 0.1, sw.SW_DEFAULT_FLAGS, x, None, None)
    torch.cuda.synchronize()
    assert sw.sw_launch_count() == n0
    assert (sentinel == 7.0).all() and (idx == 9).all() and (cnt == 9).all() and (x == 0).all() and (other == 7.0).all()


def test_launch_counter_counts_kernels(sw):
    L = sw.make_layout([640], 64)
    r = 16
    qs = torch.randn(L.total_blocks, r, device="cuda"); ks = torch.randn(L.total_blocks, r, device="cuda")
    W = torch.empty(L.total_sq, device="cuda"); R = torch.empty(L.total_sq, device="cuda")
    n0 = sw.sw_launch_count()
    sw.sw_block_scores(L, qs, ks, r, 2, sw.SW_DEFAULT_FLAGS, W, None)          # one fused launch
    assert sw.sw_launch_count() - n0 == 1
    sw.sw_walk_update(L, None, W, 2, sw.SW_DEFAULT_FLAGS, R, None)             # R^0 = W^0 copy + rescale
    assert sw.sw_launch_count() - n0 == 3
    sw.sw_block_scores(L, qs[:, :2].contiguous(), ks[:, :2].contiguous(), 2, 2, sw.SW_DEFAULT_FLAGS, W, None)
    assert sw.sw_launch_count() - n0 == 5                                      # r = 2: tile kernel + row kernel
    torch.cuda.synchronize()


def test_decode_step_captures_into_a_cuda_graph(sw):
    """Three layers of (fused selection -> split-KV attention) captured once and replayed: same block lists
    and outputs as the eager launches."""
    cfg = gen.CONFIGS[2]
    B, r, s, d, h_q, h_kv = cfg.B, cfg.r, cfg.s, cfg.d, 8, 2
    batch, t, tau, layers = 2, 64 * 40 + 17, 9, 3
    mb = O.num_blocks(t, B)
    signs, cols = gen.srht_params(3, d, r)
    dp = sw.DecodePipeline(batch, mb, h_q, h_kv, d, B, r, s, [tau] * batch, signs, cols)
    torch.manual_seed(7)
    seqlens = torch.full((batch,), t, dtype=torch.int32, device="cuda")
    bufs = []
    for _ in range(layers):
        W = torch.rand(batch, mb, mb, device="cuda").tril_()
        W /= W.sum(-1, keepdim=True)
        bufs.append(dict(W=W, kbar=torch.randn(batch, mb, d, device="cuda"), ks=torch.randn(batch, mb, r, device="cuda"),
                         q=torch.randn(batch, h_q, d, device="cuda").bfloat16(),
                         k=torch.randn(batch, h_kv, d, device="cuda").bfloat16(),
                         kc=torch.randn(batch, t, h_kv, d, device="cuda").bfloat16(),
                         vc=torch.randn(batch, t, h_kv, d, device="cuda").bfloat16()))
    kbar0 = [b_["kbar"].clone() for b_ in bufs]; ks0 = [b_["ks"].clone() for b_ in bufs]
    outs = [torch.empty(batch, h_q, d, dtype=torch.bfloat16, device="cuda") for _ in range(layers)]
    idxs = [torch.empty(batch, tau, dtype=torch.int32, device="cuda") for _ in range(layers)]

    def restore():                                   # the selection updates the key-block caches in place
        for b_, kb, ks_ in zip(bufs, kbar0, ks0):
            b_["kbar"].copy_(kb); b_["ks"].copy_(ks_)

    def step():
        dp.reset()
        for l, b_ in enumerate(bufs):
            dp.select(b_["q"], b_["k"], seqlens, b_["kbar"], b_["ks"], b_["W"])
            idxs[l].copy_(dp.idx)
            dp.attend(b_["q"], b_["kc"], b_["vc"], seqlens, outs[l])

    restore(); step(); torch.cuda.synchronize()
    ref_idx = [i.clone() for i in idxs]; ref_out = [o.clone() for o in outs]
    restore(); torch.cuda.synchronize()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        step()
    for o in outs:
        o.zero_()
    for i in idxs:
        i.zero_()
    restore(); torch.cuda.synchronize()
    graph.replay()
    torch.cuda.synchronize()
    for l in range(layers):
        assert torch.equal(idxs[l], ref_idx[l])
        assert torch.equal(outs[l], ref_out[l])
        assert (idxs[l][:, -1] == (t - 1) // B).all()          # the current block is always selected
