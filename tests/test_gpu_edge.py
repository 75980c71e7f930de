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


def _random_decode_caches(batch, mb, d, r, seed):
    g = torch.Generator(device="cuda"); g.manual_seed(seed)
    Wc = torch.rand(batch, mb, mb, device="cuda", generator=g).tril_()
    Wc /= Wc.sum(-1, keepdim=True)
    kbar = torch.randn(batch, mb, d, device="cuda", generator=g)
    ks = torch.randn(batch, mb, r, device="cuda", generator=g) * 0.3
    return Wc, kbar, ks


@pytest.mark.parametrize("mb", [304, 301])      # max_blocks % 4 == 0: cp.async stream of the cached W; else plain loads
def test_decode_selection_ragged_batch_fused_equals_row_mode(sw, mb):
    """A batch of sequences of very different lengths through sw_decode_select (three kernels: the W stream dealt over
    the whole grid in chunks numbered across sequences, the score kernel beside it, the per-sequence tail) against the
    five row-mode calls, which tests/test_gpu_parity.py checks against the oracle one sequence at a time.  Lengths: a
    first block (b_q = 0: nothing to stream), b_q a multiple of the 256-column stream tile, the longest the cache
    holds, short ones between -- the partial slots of a tile then come from CTAs shared with other sequences."""
    B, d, r, h_q, h_kv, s = 64, 128, 64, 8, 2, 2
    ts = [5, 64 * 3 + 5, 64 * 256 + 1, 64 * (mb - 1) + 7, 64 * 17, 64 * 257]
    batch = len(ts)
    taus = [max(1, min(40, (t + B - 1) // B // 3 + 1)) for t in ts]
    signs, cols = gen.srht_params(3, d, r)
    seqlens = torch.tensor(ts, dtype=torch.int32, device="cuda")
    pipes = [sw.DecodePipeline(batch, mb, h_q, h_kv, d, B, r, s, taus, signs, cols) for _ in range(2)]
    caches = [_random_decode_caches(batch, mb, d, r, 11) for _ in range(2)]
    for layer in range(3):
        torch.manual_seed(40 + layer)
        q = torch.randn(batch, h_q, d).bfloat16().cuda(); k = torch.randn(batch, h_kv, d).bfloat16().cuda()
        for dp, (Wc, kbar, ks), fused in zip(pipes, caches, (True, False)):
            dp.idx.fill_(-7); dp.count.fill_(-7)
            dp.select(q, k, seqlens, kbar, ks, Wc, fused=fused)
        torch.cuda.synchronize()
        (Wf, kbf, ksf), (Wu, kbu, ksu) = caches
        assert torch.allclose(kbf, kbu, rtol=0, atol=1e-6) and torch.allclose(ksf, ksu, rtol=0, atol=1e-5)
        rf = pipes[0].rvec[pipes[0].cur].cpu().numpy(); ru = pipes[1].rvec[pipes[1].cur].cpu().numpy()
        for s_, t in enumerate(ts):
            bq = (t - 1) // B
            scale = np.abs(ru[s_]).max()
            assert np.abs(rf[s_] - ru[s_]).max() <= 1e-5 * scale, (layer, s_)
            assert (rf[s_, bq + 1:] == 0).all()
            wf = Wf[s_, bq].cpu().numpy(); wu = Wu[s_, bq].cpu().numpy()
            assert np.abs(wf - wu).max() <= 1e-6 * max(np.abs(wu).max(), 1e-30)
            cf, cu = pipes[0].count[s_].item(), pipes[1].count[s_].item()
            assert cf == cu == min(taus[s_], bq + 1)
            got = pipes[0].idx[s_, :cf].cpu().numpy(); ref = pipes[1].idx[s_, :cu].cpu().numpy()
            assert np.all(np.diff(got) > 0) and bq in got
            diff = set(got.tolist()) ^ set(ref.tolist())
            free = [j for j in ref.tolist() if j not in (0, bq)]
            kth = min(ru[s_][free]) if free else 0.0
            assert all(abs(ru[s_][j] - kth) <= 1e-5 * scale for j in diff), (layer, s_, diff)


def test_decode_chain_reads_nothing_before_its_producers_finish(sw):
    """sw_decode_select + sw_sparse_attn_decode are five kernels chained as programmatic dependents: each may become
    resident while its predecessor runs and must read nothing an earlier kernel writes before griddepcontrol.wait.
    (Loads the compiler treats as invariant -- __ldg, const __restrict__ -- were once scheduled above the wait: the
    attention kernel read count[] / idx[] the selection had not written yet.)  The block lists are poisoned before
    every step; the output of the chained step must equal that of the attention call alone on the finished lists."""
    batch, t, h_q, h_kv, d, B, r, s = 4, 64 * 512, 8, 2, 128, 64, 64, 2
    mb = t // B
    tau = mb // 5
    signs, cols = gen.srht_params(3, d, r)
    dp = sw.DecodePipeline(batch, mb, h_q, h_kv, d, B, r, s, [tau] * batch, signs, cols)
    seqlens = torch.full((batch,), t, dtype=torch.int32, device="cuda")
    g = torch.Generator(device="cuda"); g.manual_seed(5)
    kc = torch.randn(batch, t, h_kv, d, device="cuda", generator=g).bfloat16()
    vc = torch.randn(batch, t, h_kv, d, device="cuda", generator=g).bfloat16()
    Wc, kbar, ks = _random_decode_caches(batch, mb, d, r, 6)
    out = torch.empty(batch, h_q, d, dtype=torch.bfloat16, device="cuda")
    for it in range(60):
        q = torch.randn(batch, h_q, d, device="cuda", generator=g).bfloat16()
        k = torch.randn(batch, h_kv, d, device="cuda", generator=g).bfloat16()
        dp.idx.fill_(it % 7); dp.count.fill_(1 + it % 5); out.zero_()
        if it % 3 == 0:
            torch.cuda.synchronize()
        dp.reset()
        for _ in range(1 + it % 3):
            dp.select(q, k, seqlens, kbar, ks, Wc)
            dp.attend(q, kc, vc, seqlens, out)
        torch.cuda.synchronize()
        chained = out.clone()
        assert (dp.count == tau).all()
        dp.attend(q, kc, vc, seqlens, out)
        torch.cuda.synchronize()
        assert torch.equal(chained, out), it


@pytest.mark.parametrize("batch", [300, 512])       # 512 = the largest batch one call takes (kMaxBatch)
def test_decode_selection_many_short_sequences(sw, batch):
    """300 / 512 sequences of 1 .. 8 blocks in one sw_decode_select call (more sequences than threads of the
    streaming kernel's prefix pass, chunk ranges that span many sequences, CTAs without work; at 512 the total of the
    prefix pass sits in the last slot of its table) against the row-mode calls."""
    B, d, r, h_q, h_kv, s, mb = 64, 64, 16, 4, 2, 2, 8
    rng = np.random.default_rng(3)
    ts = rng.integers(1, mb * B + 1, size=batch).tolist()
    ts[0], ts[1], ts[2] = 1, mb * B, B + 1
    taus = [3] * batch
    signs, cols = gen.srht_params(3, d, r)
    seqlens = torch.tensor(ts, dtype=torch.int32, device="cuda")
    pipes = [sw.DecodePipeline(batch, mb, h_q, h_kv, d, B, r, s, taus, signs, cols) for _ in range(2)]
    caches = [_random_decode_caches(batch, mb, d, r, 21) for _ in range(2)]
    for layer in range(2):
        torch.manual_seed(60 + layer)
        q = torch.randn(batch, h_q, d).bfloat16().cuda(); k = torch.randn(batch, h_kv, d).bfloat16().cuda()
        for dp, (Wc, kbar, ks), fused in zip(pipes, caches, (True, False)):
            dp.select(q, k, seqlens, kbar, ks, Wc, fused=fused)
        torch.cuda.synchronize()
        rf = pipes[0].rvec[pipes[0].cur]; ru = pipes[1].rvec[pipes[1].cur]
        scale = ru.abs().amax(dim=1, keepdim=True).clamp_min(1e-30)
        assert ((rf - ru).abs() <= 1e-5 * scale).all()
        assert torch.allclose(caches[0][1], caches[1][1], rtol=0, atol=1e-6)
        assert torch.equal(pipes[0].count, pipes[1].count)
        # the rows are short and random: no near-ties at 1e-5, the lists must agree
        assert torch.equal(pipes[0].idx, pipes[1].idx)


def test_decode_selection_idle_slots(sw):
    """seqlens entries outside [1, max_blocks * B] mark idle slots of a decode batch (include/sw.h): the call leaves
    their caches alone and reports an empty selection, and the live sequences come out as they do when the idle
    slots hold ordinary sequences instead."""
    B, d, r, h_q, h_kv, s, mb = 64, 128, 64, 8, 2, 2, 300
    live = {1: 64 * 280 + 9, 3: 64 * 3, 4: 64 * 299 + 1}
    idle = {0: 0, 2: mb * B + 1, 5: -4}
    batch = 6
    taus = [7] * batch
    signs, cols = gen.srht_params(3, d, r)
    torch.manual_seed(70)
    q = torch.randn(batch, h_q, d).bfloat16().cuda(); k = torch.randn(batch, h_kv, d).bfloat16().cuda()
    res = []
    for fill in (None, 64 * 100 + 5):                     # idle slots as given / replaced by an ordinary sequence
        ts = [live.get(i, idle.get(i) if fill is None else fill) for i in range(batch)]
        seqlens = torch.tensor(ts, dtype=torch.int32, device="cuda")
        dp = sw.DecodePipeline(batch, mb, h_q, h_kv, d, B, r, s, taus, signs, cols)
        Wc, kbar, ks = _random_decode_caches(batch, mb, d, r, 31)
        W0, kbar0, ks0 = Wc.clone(), kbar.clone(), ks.clone()
        for layer in range(2):                            # the second step runs with a walk state (the W stream)
            dp.idx.fill_(-7); dp.count.fill_(-7)
            dp.select(q, k, seqlens, kbar, ks, Wc)
        torch.cuda.synchronize()
        res.append((dp.rvec[dp.cur].clone(), dp.idx.clone(), dp.count.clone(), Wc, kbar, ks))
        if fill is None:
            for i in idle:
                assert dp.count[i].item() == 0 and (dp.idx[i] == -1).all() and (dp.rvec[dp.cur][i] == 0).all()
                assert torch.equal(Wc[i], W0[i]) and torch.equal(kbar[i], kbar0[i]) and torch.equal(ks[i], ks0[i])
    (ra, ia, ca, Wa, kba, ksa), (rb, ib, cb, Wb, kbb, ksb) = res
    for i, t in live.items():
        scale = rb[i].abs().max()
        assert ((ra[i] - rb[i]).abs() <= 1e-5 * scale).all()
        assert ca[i].item() == cb[i].item() == min(taus[i], (t - 1) // B + 1)
        assert torch.equal(kba[i], kbb[i]) and torch.equal(ksa[i], ksb[i]) and torch.equal(Wa[i], Wb[i])
        diff = set(ia[i].tolist()) ^ set(ib[i].tolist())
        ref = [j for j in ib[i, :cb[i]].tolist() if j not in (0, (t - 1) // B)]
        kth = min(rb[i][ref]).item() if ref else 0.0
        assert all(abs(rb[i][j].item() - kth) <= 1e-5 * scale for j in diff)


class _Guarded:
    """Device tensors carved out of larger allocations with a band of canary values on both sides (bands of 256 bytes
    or more, so that the carved tensor keeps the alignment of a fresh allocation).  check() fails when a kernel wrote
    outside the tensor it was given.  Stands in for compute-sanitizer's memcheck, which this GPU pool does not allow
    (profiles/sanitizer_r3.md)."""
    BAND = 1024                                           # elements

    def __init__(self):
        self.items = []

    def new(self, shape, dtype, fill=None):
        n = int(np.prod(shape))
        canary = {torch.float32: 12345.0, torch.bfloat16: 12288.0, torch.int32: 0x5A5A5A5A, torch.uint8: 0xA5}[dtype]
        buf = torch.full((n + 2 * self.BAND,), canary, dtype=dtype, device="cuda")
        view = buf[self.BAND:self.BAND + n].view(*shape)
        if fill is not None:
            view.copy_(fill) if torch.is_tensor(fill) else view.fill_(fill)
        self.items.append((buf, n, canary))
        return view

    def check(self, what):
        torch.cuda.synchronize()
        for k, (buf, n, canary) in enumerate(self.items):
            lo, hi = buf[:self.BAND], buf[self.BAND + n:]
            assert bool((lo == canary).all()) and bool((hi == canary).all()), f"{what}: buffer {k} was overrun"


def test_outputs_and_workspaces_stay_inside_their_buffers(sw):
    """Every output and workspace of the four chains (fused prefill selection with the tensor-core walk, fused decode
    selection with a walk state, prefill attention, split-KV decode attention) sits between canary bands; the sizes
    are ragged (b = 513 + 130 blocks, max_blocks = 301, partial last blocks) so that any rounding up to a tile
    would land in a band."""
    g = _Guarded()
    B, d, r, h_q, h_kv, s = 64, 128, 64, 8, 2, 2
    flags = sw.SW_DEFAULT_FLAGS
    signs, cols = gen.srht_params(3, d, r)
    signs_d = torch.as_tensor(np.asarray(signs, np.int8)).cuda(); cols_d = torch.as_tensor(np.asarray(cols, np.int32)).cuda()
    torch.manual_seed(90)
    # ---- prefill: sketch -> fused selection (two layers: the second runs the walk GEMM) -> attention
    seqlens = (64 * 512 + 17, 64 * 129 + 63)
    L = sw.make_layout(seqlens, B)
    T = sum(seqlens)
    taus = [b // 5 for b in L.blocks]; tau_max = max(taus)
    tau_d = torch.tensor(taus, dtype=torch.int32, device="cuda")
    q = torch.randn(T, h_q, d, device="cuda").bfloat16(); k = torch.randn(T, h_kv, d, device="cuda").bfloat16()
    v = torch.randn(T, h_kv, d, device="cuda").bfloat16()
    qs = g.new((L.total_blocks, r), torch.float32); ks = g.new((L.total_blocks, r), torch.float32)
    qbar = g.new((L.total_blocks, d), torch.float32); kbar = g.new((L.total_blocks, d), torch.float32)
    W = g.new((L.total_sq,), torch.float32); R = [g.new((L.total_sq,), torch.float32) for _ in range(2)]
    idx = g.new((L.total_blocks, tau_max), torch.int32); cnt = g.new((L.total_blocks,), torch.int32)
    ws = g.new((sw.sw_workspace_bytes(sw.SW_OP_WALK_UPDATE, L),), torch.uint8)
    out = g.new((T, h_q, d), torch.bfloat16); lse = g.new((T, h_q), torch.float32)
    for layer in range(2):
        sw.sw_sketch_qk(L, q, k, signs_d, cols_d, r, 1 / math.sqrt(r), qs, ks, qbar, kbar)
        sw.sw_prefill_select(L, qs, ks, r, s, flags, R[0] if layer else None, R[layer], W, None, tau_d, tau_max, idx, cnt, ws)
        g.check(f"prefill selection, layer {layer}")
    assert sw.sw_get_walk_kernel_used() == sw.SW_WALK_TCGEN05
    sw.sw_sparse_attn_prefill(L, q, k, v, idx, cnt, tau_max, 1 / math.sqrt(d), flags, out, lse, None)
    g.check("prefill attention")
    assert torch.isfinite(out.float()).all()
    del q, k, v
    # ---- decode: fused selection (two steps: the second streams the cached W) -> split-KV attention
    g = _Guarded()
    mb, batch = 301, 3
    ts = [64 * 300 + 1, 64 * 257, 64 * 40 + 33]
    tau = 23
    seql = torch.tensor(ts, dtype=torch.int32, device="cuda"); tau_b = torch.full((batch,), tau, dtype=torch.int32, device="cuda")
    Wc0, kb0, ks0 = _random_decode_caches(batch, mb, d, r, 41)
    Wc = g.new((batch, mb, mb), torch.float32, Wc0); kbc = g.new((batch, mb, d), torch.float32, kb0)
    ksc = g.new((batch, mb, r), torch.float32, ks0)
    rv = [g.new((batch, mb), torch.float32) for _ in range(2)]
    idx = g.new((batch, tau), torch.int32); cnt = g.new((batch,), torch.int32)
    ws = g.new((sw.sw_decode_select_workspace_bytes(batch, mb),), torch.uint8)
    qn = torch.randn(batch, h_q, d, device="cuda").bfloat16(); kn = torch.randn(batch, h_kv, d, device="cuda").bfloat16()
    for step in range(2):
        sw.sw_decode_select(batch, B, mb, qn, kn, seql, signs_d, cols_d, r, 1 / math.sqrt(r), s, flags, kbc, ksc, Wc,
                            mb * mb, rv[0] if step else None, rv[step], tau_b, tau, idx, cnt, ws)
        g.check(f"decode selection, step {step}")
    assert (cnt == tau).all()
    tmax = max(ts)
    kc = torch.randn(batch, tmax, h_kv, d, device="cuda").bfloat16(); vc = torch.randn(batch, tmax, h_kv, d, device="cuda").bfloat16()
    out = g.new((batch, h_q, d), torch.bfloat16); lse = g.new((batch, h_q), torch.float32)
    aws = g.new((sw.sw_decode_workspace_bytes(batch, h_q, h_kv, d, tau),), torch.uint8)
    sw.sw_sparse_attn_decode(batch, B, qn, kc, vc, seql, idx, cnt, tau, 1 / math.sqrt(d), out, lse, aws)
    g.check("decode attention")
    assert torch.isfinite(out.float()).all()
