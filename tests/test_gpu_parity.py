"""GPU parity: every C-ABI call of libsw against the CPU oracle on the same seeded inputs.
Tolerances are the ones BASELINE.json's north_star states:
  * selected block indices bit-exact when the GPU selector is fed the oracle's scores;
  * sketch / score / walk values within 1e-3 relative (row-norm-wise: |d| <= 1e-3 max_j |ref[i,j]|);
  * end-to-end block sets overlap >= 99 %, differences only at near-ties (<= 1e-3 of the row max);
  * attention outputs within max-abs 2e-2 and mean-abs 2e-3 (bf16 I/O, fp32 accumulation).
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


def record_overlap(test, case, overlaps):
    """Append the measured selection overlap (GPU block lists vs the oracle's, per layer and sequence) of an
    end-to-end case to the markdown table named by $SW_OVERLAP_LOG (profiles/overlap_r3.md is such a file); no-op
    when the variable is unset.  The figures are recorded for every reading, also where no threshold is asserted."""
    import os
    path = os.environ.get("SW_OVERLAP_LOG")
    if not path:
        return
    new = not os.path.exists(path)
    with open(path, "a") as f:
        if new:
            f.write("| test | case | min overlap | mean overlap | per layer / sequence |\n|---|---|---|---|---|\n")
        f.write(f"| `{test}` | {case} | {min(overlaps):.5f} | {float(np.mean(overlaps)):.5f} | "
                f"{' '.join(f'{o:.4f}' for o in overlaps)} |\n")


def rowwise_close(got, ref, rel=REL):
    got = np.asarray(got, np.float64); ref = np.asarray(ref, np.float64)
    scale = np.abs(ref).max(axis=-1, keepdims=True)
    return bool((np.abs(got - ref) <= rel * scale + 1e-30).all())


def dev(x, dtype=None):
    t = torch.as_tensor(np.ascontiguousarray(x))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def H_of(d, r, seed=5):
    signs, cols = gen.srht_params(seed, d, r)
    return signs, cols, O.srht_matrix(d, signs, cols, 1 / math.sqrt(r))


# ------------------------------------------------------------------------------ sketch
@pytest.mark.parametrize("seqlens,heads,d,r,B,dtype", [
    ((1024,), 1, 64, 16, 64, torch.float32),          # cfg 1
    ((1000,), 32, 128, 64, 64, torch.bfloat16),       # ragged tail, Llama Q heads
    ((333,), 8, 128, 64, 64, torch.bfloat16),         # K heads
    ((130, 64, 257), 8, 128, 32, 128, torch.bfloat16),  # varlen, B = 128
    ((70,), 4, 64, 64, 64, torch.bfloat16),           # r = d
    ((5,), 2, 128, 1, 64, torch.float32),             # single partial block, r = 1
])
def test_sketch(sw, seqlens, heads, d, r, B, dtype):
    torch.manual_seed(0)
    T = sum(seqlens)
    x = (torch.randn(T, heads, d) * 2 + 0.3).to(dtype)
    signs, cols, H = H_of(d, r)
    L = sw.make_layout(seqlens, B)
    sk = torch.empty(L.total_blocks, r, device="cuda"); mean = torch.empty(L.total_blocks, d, device="cuda")
    sw.sw_sketch(L, x.cuda(), dev(signs), dev(cols), r, 1 / math.sqrt(r), sk, mean)
    xn = gen.to_numpy_f64(x)
    ref_mean, ref_sk, lo = [], [], 0
    for n in seqlens:
        m = O.block_mean(O.head_mean(xn[lo:lo + n]), B)
        ref_mean.append(m); ref_sk.append(O.sketch(m, H)); lo += n
    ref_mean, ref_sk = np.concatenate(ref_mean), np.concatenate(ref_sk)
    assert rowwise_close(mean.cpu().numpy(), ref_mean)
    assert rowwise_close(sk.cpu().numpy(), ref_sk)


def test_sketch_strided_and_nosigns(sw):
    torch.manual_seed(1)
    T, heads, d, r, B = 200, 4, 128, 64, 64
    big = torch.randn(T, heads + 2, d + 8, dtype=torch.float32).to(torch.bfloat16).cuda()
    x = big[:, 1:1 + heads, 8:]                          # non-compact strides, 16-byte aligned
    _, cols, _ = H_of(d, r)
    H = O.srht_matrix(d, np.ones(d), cols, 1 / math.sqrt(r))
    L = sw.make_layout((T,), B)
    sk = torch.empty(L.total_blocks, r, device="cuda")
    sw.sw_sketch(L, x, None, dev(cols), r, 1 / math.sqrt(r), sk, None)
    ref = O.sketch(O.block_mean(O.head_mean(gen.to_numpy_f64(x)), B), H)
    assert rowwise_close(sk.cpu().numpy(), ref)


def _ref_sketch(xn, seqlens, B, H):
    ref_mean, ref_sk, lo = [], [], 0
    for n in seqlens:
        m = O.block_mean(O.head_mean(xn[lo:lo + n]), B)
        ref_mean.append(m); ref_sk.append(O.sketch(m, H)); lo += n
    return np.concatenate(ref_mean), np.concatenate(ref_sk)


@pytest.mark.parametrize("seqlens,h_q,h_kv,d,r,B,dtype", [
    ((1024,), 1, 1, 64, 16, 64, torch.float32),                 # cfg 1
    ((2048 + 19,), 32, 8, 128, 64, 64, torch.bfloat16),         # cfg 2 recipe, ragged tail (a 19-token block)
    ((192, 700, 1024, 5), 32, 8, 128, 64, 64, torch.bfloat16),  # varlen; a 5-token sequence
    ((1000,), 12, 3, 128, 32, 128, torch.bfloat16),             # B = 128
    ((300,), 6, 6, 64, 64, 64, torch.bfloat16),                 # h_q = h_kv, d = 64
])
def test_sketch_qk_one_launch(sw, seqlens, h_q, h_kv, d, r, B, dtype):
    """sw_sketch_qk (Q and K in one launch) against the oracle's head mean -> block mean -> SRHT (Alg. 1 Steps
    1-4), and against two sw_sketch calls."""
    torch.manual_seed(2)
    T = sum(seqlens)
    q = (torch.randn(T, h_q, d) + 0.3).to(dtype); k = (torch.randn(T, h_kv, d) - 0.2).to(dtype)
    signs, cols, H = H_of(d, r)
    L = sw.make_layout(seqlens, B)
    nb = L.total_blocks
    out = {n: torch.full((nb, w), float("nan"), device="cuda") for n, w in [("qs", r), ("ks", r), ("qbar", d), ("kbar", d)]}
    launches0 = sw.sw_launch_count()
    sw.sw_sketch_qk(L, q.cuda(), k.cuda(), dev(signs), dev(cols), r, 1 / math.sqrt(r), out["qs"], out["ks"], out["qbar"],
                    out["kbar"])
    assert sw.sw_launch_count() - launches0 == 1
    for x, sk, mean, heads in [(q, "qs", "qbar", h_q), (k, "ks", "kbar", h_kv)]:
        ref_mean, ref_sk = _ref_sketch(gen.to_numpy_f64(x), seqlens, B, H)
        assert rowwise_close(out[mean].cpu().numpy(), ref_mean)
        assert rowwise_close(out[sk].cpu().numpy(), ref_sk)
        one = torch.empty(nb, r, device="cuda")
        sw.sw_sketch(L, x.cuda(), dev(signs), dev(cols), r, 1 / math.sqrt(r), one, None)
        assert rowwise_close(out[sk].cpu().numpy(), one.cpu().numpy().astype(np.float64), rel=1e-5)


@pytest.mark.parametrize("seqlens,heads,d,r,B,dtype", [
    ((2048 + 19,), 8, 128, 64, 64, torch.bfloat16),
    ((192, 700, 5), 32, 128, 64, 64, torch.bfloat16),
    ((1024,), 1, 64, 16, 64, torch.float32),                    # fp32 source: the bf16 cast pre-pass of P17
])
def test_sketch_from_pooled_sums_of_a_producer(sw, seqlens, heads, d, r, B, dtype):
    """Sketch fused upstream: sw_copy_pool copies x and leaves the per-block sums behind;
    sw_sketch_from_pooled turns them into the sketch sw_sketch computes by re-reading x.  Both against the oracle."""
    torch.manual_seed(3)
    T = sum(seqlens)
    big = (torch.randn(T, heads + 1, d) + 0.25).to(dtype).cuda()
    x = big[:, 1:]                                              # strided source
    signs, cols, H = H_of(d, r)
    L = sw.make_layout(seqlens, B)
    nb = L.total_blocks
    dst = torch.full((T, heads, d), float("nan"), dtype=torch.bfloat16, device="cuda")
    sums = torch.full((nb, d), float("nan"), device="cuda")
    sw.sw_copy_pool(L, x, dst, sums)
    assert torch.equal(dst, x.to(torch.bfloat16))               # the copy (round-to-nearest cast for fp32)
    xn = gen.to_numpy_f64(x)
    lo, blk = 0, 0
    for n in seqlens:                                           # sums = plain sums over heads and valid tokens
        for i in range(O.num_blocks(n, B)):
            ref = xn[lo + i * B: lo + min((i + 1) * B, n)].sum(axis=(0, 1))
            assert np.abs(sums[blk].cpu().numpy() - ref).max() <= 1e-3 * max(np.abs(ref).max(), 1.0)
            blk += 1
        lo += n
    sk = torch.full((nb, r), float("nan"), device="cuda"); mean = torch.full((nb, d), float("nan"), device="cuda")
    sw.sw_sketch_from_pooled(L, sums, heads, dev(signs), dev(cols), r, 1 / math.sqrt(r), sk, mean)
    ref_mean, ref_sk = _ref_sketch(xn, seqlens, B, H)
    assert rowwise_close(mean.cpu().numpy(), ref_mean)
    assert rowwise_close(sk.cpu().numpy(), ref_sk)
    direct = torch.empty(nb, r, device="cuda")
    sw.sw_sketch(L, x, dev(signs), dev(cols), r, 1 / math.sqrt(r), direct, None)
    assert rowwise_close(sk.cpu().numpy(), direct.cpu().numpy().astype(np.float64), rel=1e-5)


# ------------------------------------------------------------------------------ block scores
FLAG_SETS = [O.DEFAULT_FLAGS, O.DEFAULT_FLAGS & ~O.SCORE_SOFTMAX, O.DEFAULT_FLAGS & ~O.CAUSAL,
             O.DEFAULT_FLAGS | O.POW_MATRIX, 0]


@pytest.mark.parametrize("blocks", [(16,), (100,), (37, 130, 64)])
@pytest.mark.parametrize("flags", FLAG_SETS)
@pytest.mark.parametrize("s", [1, 2, 3])
def test_block_scores(sw, blocks, flags, s):
    rng = np.random.RandomState(3)
    r, B = 64, 64
    L = sw.make_layout([b * B for b in blocks], B)
    qs = rng.randn(L.total_blocks, r).astype(np.float32) * 1.5
    ks = rng.randn(L.total_blocks, r).astype(np.float32) * 1.5
    W = torch.full((L.total_sq,), float("nan"), device="cuda"); A = torch.full_like(W, float("nan"))
    sw.sw_block_scores(L, dev(qs), dev(ks), r, s, flags, W, A)
    Wn, An = W.cpu().numpy(), A.cpu().numpy()
    lo = off = 0
    for b in blocks:
        S = O.block_scores(qs[lo:lo + b].astype(np.float64), ks[lo:lo + b].astype(np.float64))
        A_ref = O.masked_softmax(S, flags)
        W_ref = A_ref if (flags & O.POW_MATRIX) else O.power(A_ref, s, flags)
        assert rowwise_close(An[off:off + b * b].reshape(b, b), A_ref)
        assert rowwise_close(Wn[off:off + b * b].reshape(b, b), W_ref)
        lo += b; off += b * b


# ------------------------------------------------------------------------------ walk
@pytest.mark.parametrize("blocks", [(16,), (100,), (300,), (37, 130, 64)])
@pytest.mark.parametrize("flags", [O.DEFAULT_FLAGS, O.DEFAULT_FLAGS & ~O.ROWNORM, O.DEFAULT_FLAGS & ~O.CAUSAL,
                                   O.DEFAULT_FLAGS | O.POW_MATRIX])
def test_walk_update(sw, blocks, flags):
    rng = np.random.RandomState(4)
    B, s = 64, 3
    L = sw.make_layout([b * B for b in blocks], B)
    As, Rs = [], []
    for b in blocks:
        As.append(O.masked_softmax(rng.randn(b, b) * 2, flags))
        Rs.append(O.masked_softmax(rng.randn(b, b) * 2, flags))
    mat = bool(flags & O.POW_MATRIX)
    Wsrc = [a if mat else O.power(a, s, flags) for a in As]
    Wd = dev(np.concatenate([w.ravel() for w in Wsrc]), torch.float32)
    Rp = dev(np.concatenate([r.ravel() for r in Rs]), torch.float32)
    ws = torch.empty(sw.sw_workspace_bytes(sw.SW_OP_WALK_UPDATE, L), dtype=torch.uint8, device="cuda")
    for prev in (None, Rp):
        out = torch.full((L.total_sq,), float("nan"), device="cuda")
        sw.sw_walk_update(L, prev, Wd, s, flags, out, ws)
        on = out.cpu().numpy(); off = 0
        for k, b in enumerate(blocks):
            # the oracle gets the fp32-rounded operands the GPU saw
            A32 = Wsrc[k].astype(np.float32).astype(np.float64) if mat else None
            if mat:
                ref = O.walk_update(None if prev is None else Rs[k].astype(np.float32).astype(np.float64),
                                    A32, s, flags)
            else:
                W32 = Wsrc[k].astype(np.float32).astype(np.float64)
                R0 = np.eye(b) if prev is None else Rs[k].astype(np.float32).astype(np.float64)
                ref = R0 @ W32
                if flags & O.ROWNORM:
                    ref = O.row_rescale(ref)
            assert rowwise_close(on[off:off + b * b].reshape(b, b), ref)
            off += b * b


# tcgen05 3xTF32 walk GEMM (walk_tc.cu): same product, both kernels, fp32-class accuracy.
@pytest.mark.parametrize("b", [256, 300, 512, 1000, 1156])
@pytest.mark.parametrize("flags", [O.DEFAULT_FLAGS, O.DEFAULT_FLAGS & ~O.ROWNORM, O.DEFAULT_FLAGS & ~O.CAUSAL,
                                   O.DEFAULT_FLAGS | O.POW_MATRIX, O.CAUSAL | O.ROWNORM])
def test_walk_update_tcgen05(sw, b, flags):
    rng = np.random.RandomState(40 + b)
    B, s = 64, 2
    L = sw.make_layout([b * B], B)
    if flags & O.SCORE_SOFTMAX:
        A = O.masked_softmax(rng.randn(b, b) * 2, flags)
        R = O.masked_softmax(rng.randn(b, b) * 2, flags)
    else:                                   # raw signed scores reading (P5)
        A = np.tril(rng.randn(b, b)); R = np.tril(rng.randn(b, b))
    mat = bool(flags & O.POW_MATRIX)
    Wsrc = (A if mat else O.power(A, s, flags)).astype(np.float32)
    R32 = R.astype(np.float32)
    Wd, Rp = dev(Wsrc.ravel()), dev(R32.ravel())
    ws = torch.empty(sw.sw_workspace_bytes(sw.SW_OP_WALK_UPDATE, L), dtype=torch.uint8, device="cuda")
    if mat:
        ref = O.walk_update(R32.astype(np.float64), Wsrc.astype(np.float64), s, flags)
    else:
        ref = R32.astype(np.float64) @ Wsrc.astype(np.float64)
        if flags & O.ROWNORM:
            ref = O.row_rescale(ref)
    outs = {}
    for kern in (sw.SW_WALK_SIMT, sw.SW_WALK_TCGEN05):
        prev = sw.sw_set_walk_kernel(kern)
        try:
            out = torch.full((b * b,), float("nan"), device="cuda")
            sw.sw_walk_update(L, Rp, Wd, s, flags, out, ws)
            torch.cuda.synchronize()
            assert sw.sw_get_walk_kernel_used() == kern
        finally:
            sw.sw_set_walk_kernel(prev)
        outs[kern] = out.cpu().numpy().reshape(b, b)
        assert rowwise_close(outs[kern], ref)
        if flags & O.CAUSAL:
            assert not np.triu(outs[kern], 1).any()
    # the split keeps fp32-class accuracy: a single TF32 product would be off by ~5e-4 of the row max
    scale = np.abs(ref).max(axis=-1, keepdims=True)
    err_tc = (np.abs(outs[sw.SW_WALK_TCGEN05] - ref) / scale).max()
    assert err_tc <= 1e-5, err_tc


def test_walk_tcgen05_needs_workspace_and_shape(sw):
    B = 64
    prev = sw.sw_set_walk_kernel(sw.SW_WALK_TCGEN05)
    try:
        for blocks, ws_ok in (((512,), False), ((100,), True), ((100, 255), True)):
            L = sw.make_layout([b * B for b in blocks], B)
            x = torch.zeros(L.total_sq, device="cuda")
            out = torch.zeros(L.total_sq, device="cuda")
            ws = torch.empty(sw.sw_workspace_bytes(sw.SW_OP_WALK_UPDATE, L) if ws_ok else 16, dtype=torch.uint8,
                             device="cuda")
            with pytest.raises(sw.SwError) as e:
                sw.sw_walk_update(L, x, x, 1, O.DEFAULT_FLAGS, out, ws)
            assert e.value.code == (sw.SW_ERR_UNSUPPORTED if ws_ok else sw.SW_ERR_WORKSPACE)
    finally:
        sw.sw_set_walk_kernel(prev)


@pytest.mark.parametrize("blocks", [(256, 301, 512), (130, 600), (257,)])
@pytest.mark.parametrize("flags", [O.DEFAULT_FLAGS, O.DEFAULT_FLAGS & ~O.CAUSAL])
def test_walk_update_tcgen05_varlen_batch(sw, blocks, flags):
    """The tensor-core walk on a packed varlen batch (one stacked operand image per operand), sizes that are no
    multiple of the 128-row tiles or of 4, against the oracle's fp64 product of the fp32 operands."""
    rng = np.random.RandomState(sum(blocks))
    B, s = 64, 2
    L = sw.make_layout([b * B for b in blocks], B)
    As = [O.power(O.masked_softmax(rng.randn(b, b) * 2, flags), s, flags).astype(np.float32) for b in blocks]
    Rs = [O.masked_softmax(rng.randn(b, b) * 2, flags).astype(np.float32) for b in blocks]
    Wd = dev(np.concatenate([a.ravel() for a in As])); Rp = dev(np.concatenate([r.ravel() for r in Rs]))
    ws = torch.full((sw.sw_workspace_bytes(sw.SW_OP_WALK_UPDATE, L),), 0xFF, dtype=torch.uint8, device="cuda")   # NaN bits
    prev = sw.sw_set_walk_kernel(sw.SW_WALK_TCGEN05)
    try:
        out = torch.full((L.total_sq,), float("nan"), device="cuda")
        sw.sw_walk_update(L, Rp, Wd, s, flags, out, ws)
        torch.cuda.synchronize()
        assert sw.sw_get_walk_kernel_used() == sw.SW_WALK_TCGEN05
    finally:
        sw.sw_set_walk_kernel(prev)
    on = out.cpu().numpy(); off = 0
    for k, b in enumerate(blocks):
        ref = Rs[k].astype(np.float64) @ As[k].astype(np.float64)
        if flags & O.ROWNORM:
            ref = O.row_rescale(ref)
        got = on[off:off + b * b].reshape(b, b)
        assert np.isfinite(got).all()
        scale = np.abs(ref).max(axis=-1, keepdims=True)
        assert (np.abs(got - ref) / scale).max() <= 1e-5
        off += b * b


@pytest.mark.parametrize("blocks,r", [((16,), 16), ((100,), 64), ((37, 130, 64), 64), ((512,), 64), ((300, 700), 32),
                                      ((1030,), 64), ((50,), 2),
                                      # long rows: the strip of score rows leaves the key ring of the fused score kernel two stages
                                      ((1500,), 64), ((2049, 700), 32)])
@pytest.mark.parametrize("flags,s", [(O.DEFAULT_FLAGS, 2), (O.DEFAULT_FLAGS & ~O.SCORE_SOFTMAX, 3),
                                     (O.DEFAULT_FLAGS | O.POW_MATRIX, 2), (O.DEFAULT_FLAGS & ~O.ROWNORM, 1),
                                     (O.DEFAULT_FLAGS & ~O.CAUSAL, 2), (O.DEFAULT_FLAGS, 8)])
def test_prefill_select_fused_chain(sw, blocks, r, flags, s):
    """sw_prefill_select (scores + softmax + power + operand images | walk GEMM | rescale + top-tau: at most three
    launches) against the oracle's Alg. 1 Steps 5-7, three layers with R carried, and against the three plain calls
    on the same inputs.  Sizes cover the SIMT and the tensor-core walk, varlen batches, b % 4 != 0 and r = 2 (which
    the fused score kernel does not take: the plain chain runs)."""
    B, layers = 64, 3
    L = sw.make_layout([b * B for b in blocks], B)
    taus = [O.tau_from_density(0.2, b) for b in blocks]
    tau_max = max(taus)
    tau_d = dev(np.asarray(taus, np.int32))
    ws = torch.full((max(sw.sw_workspace_bytes(sw.SW_OP_WALK_UPDATE, L), 16),), 0xFF, dtype=torch.uint8, device="cuda")
    nb = L.total_blocks
    R_gpu = [torch.full((L.total_sq,), float("nan"), device="cuda") for _ in range(2)]
    R_pl = [torch.full((L.total_sq,), float("nan"), device="cuda") for _ in range(2)]
    R_ref = [None] * len(blocks)
    cur = -1
    for layer in range(layers):
        rng = np.random.RandomState(1000 * layer + nb)
        qs = (rng.randn(nb, r) * 1.2).astype(np.float32); ks = (rng.randn(nb, r) * 1.2).astype(np.float32)
        W = torch.full((L.total_sq,), float("nan"), device="cuda"); A = torch.full_like(W, float("nan"))
        idx = torch.full((nb, tau_max), -7, dtype=torch.int32, device="cuda"); cnt = torch.full((nb,), -7, dtype=torch.int32, device="cuda")
        nxt = 0 if cur < 0 else 1 - cur
        n0 = sw.sw_launch_count()
        sw.sw_prefill_select(L, dev(qs), dev(ks), r, s, flags, None if cur < 0 else R_gpu[cur], R_gpu[nxt], W, A, tau_d,
                             tau_max, idx, cnt, ws)
        launches = sw.sw_launch_count() - n0
        if r >= 4 and not ((flags & O.POW_MATRIX) and s > 1):
            assert launches == (2 if cur < 0 else 3), launches
        # the three plain calls on the same inputs
        W2 = torch.empty_like(W); idx2 = torch.empty_like(idx); cnt2 = torch.empty_like(cnt)
        sw.sw_block_scores(L, dev(qs), dev(ks), r, s, flags, W2, None)
        sw.sw_walk_update(L, None if cur < 0 else R_pl[cur], W2, s, flags, R_pl[nxt], ws)
        sw.sw_select_topk(L, R_pl[nxt], tau_d, tau_max, flags, idx2, cnt2)
        torch.cuda.synchronize()
        cur = nxt
        Wn, An, Rn, Rp = W.cpu().numpy(), A.cpu().numpy(), R_gpu[cur].cpu().numpy(), R_pl[cur].cpu().numpy()
        idx_g, cnt_g = idx.cpu().numpy(), cnt.cpu().numpy()
        assert np.array_equal(cnt_g, cnt2.cpu().numpy())
        lo = off = 0
        for k, b in enumerate(blocks):
            S = O.block_scores(qs[lo:lo + b].astype(np.float64), ks[lo:lo + b].astype(np.float64))
            A_ref = O.masked_softmax(S, flags)
            W_ref = A_ref if (flags & O.POW_MATRIX) else O.power(A_ref, s, flags)
            R_ref[k] = O.walk_update(R_ref[k], A_ref, s, flags)
            sl = slice(off, off + b * b)
            assert rowwise_close(An[sl].reshape(b, b), A_ref)
            assert rowwise_close(Wn[sl].reshape(b, b), W_ref)
            assert rowwise_close(Rn[sl].reshape(b, b), R_ref[k])
            assert rowwise_close(Rn[sl].reshape(b, b), Rp[sl].reshape(b, b).astype(np.float64), rel=1e-4)
            if flags & O.CAUSAL:
                assert not np.triu(Rn[sl].reshape(b, b), 1).any()
            idx_ref, cnt_ref = O.select_topk(R_ref[k], taus[k], flags)
            assert np.array_equal(cnt_g[lo:lo + b], cnt_ref)
            for i in range(b):
                forced = ({i} if flags & O.FORCE_LAST else set()) | ({0} if flags & O.FORCE_FIRST else set())
                assert near_tie_only(idx_g[lo + i, :cnt_ref[i]], idx_ref[i, :cnt_ref[i]], R_ref[k][i], forced), (layer, k, i)
                assert (idx_g[lo + i, cnt_ref[i]:] == -1).all()
            lo += b; off += b * b


def test_walk_s1_identity_is_block_scores(sw):
    # north_star: s = 1, R^0 = I  =>  R == A (one-hop)
    rng = np.random.RandomState(8)
    b, B = 80, 64
    L = sw.make_layout([b * B], B)
    A = O.masked_softmax(rng.randn(b, b), O.DEFAULT_FLAGS).astype(np.float32)
    out = torch.empty(b * b, device="cuda")
    sw.sw_walk_update(L, None, dev(A.ravel()), 1, O.DEFAULT_FLAGS & ~O.ROWNORM, out, None)
    assert np.array_equal(out.cpu().numpy().reshape(b, b), A)


# ------------------------------------------------------------------------------ select
@pytest.mark.parametrize("blocks,taus", [((16,), (4,)), ((100,), (20,)), ((300,), (60,)), ((37, 130, 64), (8, 26, 13)),
                                         ((50,), (1,)), ((50,), (2,)), ((20,), (64,))])
@pytest.mark.parametrize("flags", [O.DEFAULT_FLAGS, O.DEFAULT_FLAGS & ~O.CAUSAL, O.CAUSAL, O.CAUSAL | O.FORCE_FIRST,
                                   O.CAUSAL | O.FORCE_LAST])
def test_select_topk_bit_exact_given_oracle_scores(sw, blocks, taus, flags):
    rng = np.random.RandomState(6)
    B = 64
    L = sw.make_layout([b * B for b in blocks], B)
    Rs = []
    for b in blocks:
        R = rng.rand(b, b).astype(np.float32)
        R[rng.rand(b, b) < 0.3] = 0.25                        # deliberate ties
        R[rng.rand(b, b) < 0.05] = 0.0
        if flags & O.CAUSAL:
            R = np.tril(R)
        Rs.append(R)
    tau_max = max(taus) + 3
    idx = torch.full((L.total_blocks, tau_max), -7, dtype=torch.int32, device="cuda")
    cnt = torch.full((L.total_blocks,), -7, dtype=torch.int32, device="cuda")
    sw.sw_select_topk(L, dev(np.concatenate([r.ravel() for r in Rs])), dev(np.asarray(taus, np.int32)), tau_max,
                      flags, idx, cnt)
    idx, cnt = idx.cpu().numpy(), cnt.cpu().numpy()
    lo = 0
    for b, tau, R in zip(blocks, taus, Rs):
        ref_idx, ref_cnt = O.select_topk(R.astype(np.float64), tau, flags)
        assert np.array_equal(cnt[lo:lo + b], ref_cnt)
        assert np.array_equal(idx[lo:lo + b, :tau], ref_idx)
        assert (idx[lo:lo + b, tau:] == -1).all()
        lo += b


def test_select_topk_negative_nan_inf(sw):
    rng = np.random.RandomState(9)
    b, B, tau = 70, 64, 9
    R = rng.randn(b, b).astype(np.float32)
    R[5, 2] = np.nan; R[9, 1] = -np.inf; R[11, 3] = np.inf; R[20, :8] = -0.0; R[20, 8:12] = 0.0
    flags = O.CAUSAL
    L = sw.make_layout([b * B], B)
    idx = torch.empty(b, tau, dtype=torch.int32, device="cuda"); cnt = torch.empty(b, dtype=torch.int32, device="cuda")
    sw.sw_select_topk(L, dev(R.ravel()), dev(np.asarray([tau], np.int32)), tau, flags, idx, cnt)
    ref_idx, ref_cnt = O.select_topk(R.astype(np.float64), tau, flags)
    assert np.array_equal(idx.cpu().numpy(), ref_idx) and np.array_equal(cnt.cpu().numpy(), ref_cnt)


@pytest.mark.parametrize("b", [300, 2048, 2500])
def test_select_topk_degenerate_and_clustered_rows(sw, b):
    """Rows whose scores are all equal (ties go to the lower index), two-valued, or packed into one binade
    (every radix pass sees heavy bin contention); b = 2500 takes the path that re-reads the row instead of
    keeping it in registers.  Bit-exact against the oracle."""
    rng = np.random.RandomState(b)
    B, tau = 64, max(3, b // 5)
    R = np.tril(rng.rand(b, b)).astype(np.float32)
    R[b - 1, :] = 0.25                                        # all equal
    R[b - 2, :] = np.where(rng.rand(b) < 0.5, 0.5, 0.25)      # two values
    R[b - 3, :] = (1.0 + rng.rand(b) * 2.0 ** -12).astype(np.float32)   # one binade, 11 significant bits
    R[b - 4, :] = 0.0
    R = np.tril(R)
    flags = O.DEFAULT_FLAGS
    L = sw.make_layout([b * B], B)
    idx = torch.empty(b, tau, dtype=torch.int32, device="cuda"); cnt = torch.empty(b, dtype=torch.int32, device="cuda")
    sw.sw_select_topk(L, dev(R.ravel()), dev(np.asarray([tau], np.int32)), tau, flags, idx, cnt)
    ref_idx, ref_cnt = O.select_topk(R.astype(np.float64), tau, flags)
    assert np.array_equal(cnt.cpu().numpy(), ref_cnt)
    assert np.array_equal(idx.cpu().numpy(), ref_idx)


# ------------------------------------------------------------------------------ prefill attention
def random_lists(rng, b, tau, causal=True):
    R = rng.rand(b, b)
    return O.select_topk(np.tril(R) if causal else R, tau, O.DEFAULT_FLAGS if causal else (O.DEFAULT_FLAGS & ~O.CAUSAL))


def attn_case(sw, seqlens, h_q, h_kv, d, B, tau_frac, dtype, causal=True, seed=0, heads_checked=None,
              kernel=None):
    kernel = sw.SW_PREFILL_AUTO if kernel is None else kernel
    prev = sw.sw_set_prefill_kernel(kernel)
    try:
        _attn_case(sw, seqlens, h_q, h_kv, d, B, tau_frac, dtype, causal, seed, heads_checked)
        if kernel != sw.SW_PREFILL_AUTO:
            assert sw.sw_get_prefill_kernel_used() == kernel
    finally:
        sw.sw_set_prefill_kernel(prev)


def _attn_case(sw, seqlens, h_q, h_kv, d, B, tau_frac, dtype, causal, seed, heads_checked):
    rng = np.random.RandomState(seed)
    torch.manual_seed(seed)
    T = sum(seqlens)
    q = torch.randn(T, h_q, d).to(dtype); k = torch.randn(T, h_kv, d).to(dtype); v = torch.randn(T, h_kv, d).to(dtype)
    L = sw.make_layout(seqlens, B)
    flags = O.DEFAULT_FLAGS if causal else (O.DEFAULT_FLAGS & ~O.CAUSAL)
    taus = [max(1, int(math.ceil(tau_frac * b))) for b in L.blocks]
    tau_max = max(taus)
    idx_all = np.full((L.total_blocks, tau_max), -1, np.int32); cnt_all = np.zeros(L.total_blocks, np.int32)
    lo = 0
    for b, tau in zip(L.blocks, taus):
        i, c = random_lists(rng, b, tau, causal)
        idx_all[lo:lo + b, :tau] = i; cnt_all[lo:lo + b] = c; lo += b
    out = torch.full((T, h_q, d), float("nan"), dtype=dtype, device="cuda")
    lse = torch.empty(T, h_q, device="cuda")
    ws = torch.empty(sw.sw_workspace_bytes(sw.SW_OP_ATTN_PREFILL, L, h_q, h_kv, d, tau_max,
                                           sw.SW_F32 if dtype == torch.float32 else sw.SW_BF16) + 16,
                     dtype=torch.uint8, device="cuda")
    scale = 1 / math.sqrt(d)
    sw.sw_sparse_attn_prefill(L, q.cuda(), k.cuda(), v.cuda(), dev(idx_all), dev(cnt_all), tau_max, scale, flags, out,
                              lse, ws)
    # the oracle sees what the tensor cores see: operands rounded to bf16 (P17)
    qn, kn, vn = (gen.to_numpy_f64(t.to(torch.bfloat16)) for t in (q, k, v))
    got, got_lse = out.float().cpu().numpy(), lse.cpu().numpy()
    assert np.isfinite(got).all()
    tlo = blo = 0
    for n, b in zip(seqlens, L.blocks):
        ref, ref_lse = O.sparse_attention(qn[tlo:tlo + n], kn[tlo:tlo + n], vn[tlo:tlo + n], idx_all[blo:blo + b],
                                          cnt_all[blo:blo + b], B, scale, flags, q_heads=heads_checked, return_lse=True)
        hs = list(range(h_q)) if heads_checked is None else heads_checked
        err = np.abs(got[tlo:tlo + n][:, hs] - ref[:, hs])
        assert err.max() <= ATT_MAX and err.mean() <= ATT_MEAN, (err.max(), err.mean())
        assert np.abs(got_lse[tlo:tlo + n][:, hs] - ref_lse[:, hs]).max() <= 2e-2
        tlo += n; blo += b


@pytest.mark.parametrize("case", [
    dict(seqlens=(1024,), h_q=1, h_kv=1, d=64, B=64, tau_frac=0.25, dtype=torch.float32),      # cfg 1 shape
    dict(seqlens=(1000,), h_q=8, h_kv=2, d=128, B=64, tau_frac=0.2, dtype=torch.bfloat16),     # GQA 4, ragged
    dict(seqlens=(700,), h_q=4, h_kv=4, d=128, B=128, tau_frac=0.5, dtype=torch.bfloat16),     # B = 128, MHA
    dict(seqlens=(130, 64, 257), h_q=4, h_kv=1, d=64, B=64, tau_frac=0.5, dtype=torch.bfloat16),  # varlen
    dict(seqlens=(515,), h_q=8, h_kv=2, d=128, B=64, tau_frac=1.0, dtype=torch.bfloat16),      # 100 % density
    dict(seqlens=(320,), h_q=2, h_kv=1, d=128, B=64, tau_frac=0.6, dtype=torch.bfloat16, causal=False),
    dict(seqlens=(40,), h_q=2, h_kv=2, d=64, B=64, tau_frac=1.0, dtype=torch.bfloat16),        # one partial block
])
def test_sparse_attn_prefill(sw, case):
    attn_case(sw, **case)


# the same problems through each kernel explicitly: shapes that fit the tcgen05 kernel (d = 128, GQA 4)
TC_CASES = [
    dict(seqlens=(1000,), h_q=8, h_kv=2, d=128, B=64, tau_frac=0.2, dtype=torch.bfloat16),     # ragged tail
    dict(seqlens=(1100,), h_q=4, h_kv=1, d=128, B=128, tau_frac=0.4, dtype=torch.bfloat16),    # B = 128
    dict(seqlens=(130, 64, 257, 1), h_q=8, h_kv=2, d=128, B=64, tau_frac=0.5, dtype=torch.bfloat16),  # varlen
    dict(seqlens=(515,), h_q=8, h_kv=2, d=128, B=64, tau_frac=1.0, dtype=torch.bfloat16),      # 100 % density
    dict(seqlens=(320,), h_q=4, h_kv=1, d=128, B=64, tau_frac=0.6, dtype=torch.bfloat16, causal=False),
    dict(seqlens=(40,), h_q=4, h_kv=1, d=128, B=64, tau_frac=1.0, dtype=torch.bfloat16),       # one partial block
    dict(seqlens=(700,), h_q=4, h_kv=1, d=128, B=64, tau_frac=0.1, dtype=torch.bfloat16),      # odd chunk counts
    dict(seqlens=(600,), h_q=8, h_kv=2, d=128, B=64, tau_frac=0.3, dtype=torch.float32),       # P17 cast pre-pass
    dict(seqlens=(4096 + 33,), h_q=8, h_kv=2, d=128, B=64, tau_frac=0.2, dtype=torch.bfloat16,
         heads_checked=[0, 3, 6]),                                                             # long rows
]


@pytest.mark.parametrize("kernel", ["generic", "tcgen05"])
@pytest.mark.parametrize("case", TC_CASES)
def test_sparse_attn_prefill_each_kernel(sw, case, kernel):
    attn_case(sw, kernel=sw.SW_PREFILL_TCGEN05 if kernel == "tcgen05" else sw.SW_PREFILL_GENERIC, **case)


@pytest.mark.parametrize("kernel", ["generic", "tcgen05"])
@pytest.mark.parametrize("B", [64, 128])
def test_sparse_attn_prefill_list_order_and_skipped_entries(sw, kernel, B):
    """include/sw.h: the block lists are order free, and entries that are -1, past the end of the sequence or hidden
    entirely by the causal mask are skipped wherever they stand (the tcgen05 kernel requests the K tiles of list
    positions 0 and 1 before it has built its chunk list).  Three calls on the same selection -- ascending lists,
    every row randomly permuted, every row permuted with such entries planted at random positions (position 0
    included) -- must agree with each other and with the oracle on the ascending lists."""
    rng = np.random.RandomState(17)
    torch.manual_seed(17)
    seqlens, h_q, h_kv, d = (900, 300), 8, 2, 128
    T = sum(seqlens)
    q = torch.randn(T, h_q, d).bfloat16(); k = torch.randn(T, h_kv, d).bfloat16(); v = torch.randn(T, h_kv, d).bfloat16()
    L = sw.make_layout(seqlens, B)
    taus = [max(1, int(math.ceil(0.4 * b))) for b in L.blocks]
    tau_max = max(taus) + 3                                        # room for the planted entries
    asc = np.full((L.total_blocks, tau_max), -1, np.int32); cnt = np.zeros(L.total_blocks, np.int32)
    lo = 0
    for b, tau in zip(L.blocks, taus):
        i, c = random_lists(rng, b, tau, True)
        asc[lo:lo + b, :tau] = i; cnt[lo:lo + b] = c; lo += b
    perm = asc.copy(); junk = asc.copy(); cnt_junk = cnt.copy()
    lo = 0
    for b in L.blocks:
        for i in range(b):
            row = asc[lo + i, :cnt[lo + i]]
            perm[lo + i, :len(row)] = rng.permutation(row)
            extra = [-1, b + 5, i + 1 + rng.randint(0, 3)]         # -1, past the end, hidden by the mask (j > i)
            mixed = list(rng.permutation(row))
            for e in extra:
                mixed.insert(rng.randint(0, len(mixed) + 1) if i % 2 else 0, e)
            junk[lo + i, :len(mixed)] = mixed; cnt_junk[lo + i] = len(mixed)
        lo += b
    scale = 1 / math.sqrt(d)
    prev = sw.sw_set_prefill_kernel(sw.SW_PREFILL_TCGEN05 if kernel == "tcgen05" else sw.SW_PREFILL_GENERIC)
    try:
        outs = []
        for lists, counts in ((asc, cnt), (perm, cnt), (junk, cnt_junk)):
            out = torch.full((T, h_q, d), float("nan"), dtype=torch.bfloat16, device="cuda")
            sw.sw_sparse_attn_prefill(L, q.cuda(), k.cuda(), v.cuda(), dev(lists), dev(counts), tau_max, scale,
                                      O.DEFAULT_FLAGS, out, None, None)
            outs.append(out.float().cpu().numpy())
    finally:
        sw.sw_set_prefill_kernel(prev)
    assert all(np.isfinite(o).all() for o in outs)
    # another key order = another summation order of the same softmax: bf16 output rounding is the difference
    for o in outs[1:]:
        err = np.abs(o - outs[0])
        assert err.max() <= ATT_MAX and err.mean() <= ATT_MEAN, (err.max(), err.mean())
    qn, kn, vn = (gen.to_numpy_f64(t) for t in (q, k, v))
    hs = [0, 5]
    tlo = blo = 0
    for n, b in zip(seqlens, L.blocks):
        ref = O.sparse_attention(qn[tlo:tlo + n], kn[tlo:tlo + n], vn[tlo:tlo + n], asc[blo:blo + b], cnt[blo:blo + b], B,
                                 scale, O.DEFAULT_FLAGS, q_heads=hs)
        for o in outs:
            err = np.abs(o[tlo:tlo + n][:, hs] - ref[:, hs])
            assert err.max() <= ATT_MAX and err.mean() <= ATT_MEAN, (err.max(), err.mean())
        tlo += n; blo += b


def test_prefill_tcgen05_rejects_unfit_shapes(sw):
    prev = sw.sw_set_prefill_kernel(sw.SW_PREFILL_TCGEN05)
    try:
        with pytest.raises(sw.SwError) as e:
            _attn_case(sw, (128,), 2, 2, 64, 64, 1.0, torch.bfloat16, True, 0, None)
        assert e.value.code == sw.SW_ERR_UNSUPPORTED
    finally:
        sw.sw_set_prefill_kernel(prev)


def test_sparse_attn_prefill_full_density_is_dense_causal(sw):
    # north_star pin, on the GPU path: 100 % density == dense causal softmax attention (torch SDPA fp64)
    torch.manual_seed(3)
    n, h_q, h_kv, d, B = 448, 8, 2, 128, 64
    q = torch.randn(n, h_q, d).bfloat16(); k = torch.randn(n, h_kv, d).bfloat16(); v = torch.randn(n, h_kv, d).bfloat16()
    b = n // B
    L = sw.make_layout((n,), B)
    idx = np.tile(np.arange(b, dtype=np.int32), (b, 1)); cnt = np.arange(1, b + 1, dtype=np.int32)
    idx = np.where(np.arange(b)[None, :] <= np.arange(b)[:, None], idx, -1).astype(np.int32)
    out = torch.empty(n, h_q, d, dtype=torch.bfloat16, device="cuda")
    sw.sw_sparse_attn_prefill(L, q.cuda(), k.cuda(), v.cuda(), dev(idx), dev(cnt), b, 1 / math.sqrt(d),
                              O.DEFAULT_FLAGS, out, None, None)
    qq = q.double().permute(1, 0, 2)[None]
    kk = k.double().permute(1, 0, 2).repeat_interleave(4, 0)[None]
    vv = v.double().permute(1, 0, 2).repeat_interleave(4, 0)[None]
    ref = torch.nn.functional.scaled_dot_product_attention(qq, kk, vv, is_causal=True)[0].permute(1, 0, 2).numpy()
    err = np.abs(out.float().cpu().numpy() - ref)
    assert err.max() <= ATT_MAX and err.mean() <= ATT_MEAN


# ------------------------------------------------------------------------------ decode attention
@pytest.mark.parametrize("ts,h_q,h_kv,d,B,tau", [
    ((64 * 9 + 1, 64 * 9 + 32, 64 * 10), 32, 8, 128, 64, 5),      # t mod B in {1, B/2, 0}
    ((700,), 8, 2, 128, 64, 11),                                     # all blocks selected
    ((300, 90), 4, 4, 64, 64, 3),
    ((1000, 513), 16, 2, 128, 128, 4),                               # B = 128, group 8
])
def test_sparse_attn_decode(sw, ts, h_q, h_kv, d, B, tau):
    rng = np.random.RandomState(2)
    torch.manual_seed(2)
    batch, tmax = len(ts), max(ts)
    q = torch.randn(batch, h_q, d).bfloat16()
    kc = torch.randn(batch, tmax, h_kv, d).bfloat16(); vc = torch.randn(batch, tmax, h_kv, d).bfloat16()
    idx = np.full((batch, tau), -1, np.int32); cnt = np.zeros(batch, np.int32)
    for s_, t in enumerate(ts):
        bq = (t - 1) // B
        sel = O.select_topk_row(rng.rand(bq + 1), bq, tau, O.DEFAULT_FLAGS)
        idx[s_, :len(sel)] = sel; cnt[s_] = len(sel)
    out = torch.full((batch, h_q, d), float("nan"), dtype=torch.bfloat16, device="cuda")
    lse = torch.empty(batch, h_q, device="cuda")
    ws = torch.empty(sw.sw_decode_workspace_bytes(batch, h_q, h_kv, d, tau), dtype=torch.uint8, device="cuda")
    scale = 1 / math.sqrt(d)
    sw.sw_sparse_attn_decode(batch, B, q.cuda(), kc.cuda(), vc.cuda(), dev(np.asarray(ts, np.int32)), dev(idx),
                             dev(cnt), tau, scale, out, lse, ws)
    got = out.float().cpu().numpy()
    for s_, t in enumerate(ts):
        ref = O.decode_attention(gen.to_numpy_f64(q[s_]), gen.to_numpy_f64(kc[s_, :t]), gen.to_numpy_f64(vc[s_, :t]),
                                 idx[s_, :cnt[s_]], B, scale)
        err = np.abs(got[s_] - ref)
        assert err.max() <= ATT_MAX and err.mean() <= ATT_MEAN, (err.max(), err.mean())


@pytest.mark.parametrize("ts,h_q,h_kv,d,B,tau", [
    ((64 * 9 + 1, 64 * 9 + 32, 64 * 10), 32, 8, 128, 64, 5),
    ((1000, 513), 16, 2, 128, 128, 4),
])
def test_sparse_attn_decode_paged(sw, ts, h_q, h_kv, d, B, tau):
    """Paged KV cache: the logical blocks of every sequence are scattered over one pool of pages in a random
    order (sequences interleaved, unused pages filled with NaN); the result must equal the oracle's on the
    logically contiguous cache, and the contiguous call's bit for bit."""
    rng = np.random.RandomState(4)
    torch.manual_seed(4)
    batch, tmax = len(ts), max(ts)
    mb = O.num_blocks(tmax, B)
    q = torch.randn(batch, h_q, d).bfloat16()
    kc = torch.randn(batch, tmax, h_kv, d).bfloat16(); vc = torch.randn(batch, tmax, h_kv, d).bfloat16()
    idx = np.full((batch, tau), -1, np.int32); cnt = np.zeros(batch, np.int32)
    for s_, t in enumerate(ts):
        bq = (t - 1) // B
        sel = O.select_topk_row(rng.rand(bq + 1), bq, tau, O.DEFAULT_FLAGS)
        idx[s_, :len(sel)] = sel; cnt[s_] = len(sel)
    n_pages = batch * mb + 7
    perm = rng.permutation(n_pages)
    table = np.full((batch, mb), -1, np.int32)
    kpool = torch.full((n_pages, B, h_kv, d), float("nan"), dtype=torch.bfloat16)
    vpool = torch.full((n_pages, B, h_kv, d), float("nan"), dtype=torch.bfloat16)
    nxt = 0
    for s_, t in enumerate(ts):
        for j in range(O.num_blocks(t, B)):
            pg = int(perm[nxt]); nxt += 1
            table[s_, j] = pg
            m = min(B, t - j * B)
            kpool[pg, :m] = kc[s_, j * B:j * B + m]; vpool[pg, :m] = vc[s_, j * B:j * B + m]
    scale = 1 / math.sqrt(d)
    ws = torch.empty(sw.sw_decode_workspace_bytes(batch, h_q, h_kv, d, tau), dtype=torch.uint8, device="cuda")
    seql = dev(np.asarray(ts, np.int32))
    out_p = torch.full((batch, h_q, d), float("nan"), dtype=torch.bfloat16, device="cuda")
    out_c = torch.full((batch, h_q, d), float("nan"), dtype=torch.bfloat16, device="cuda")
    sw.sw_sparse_attn_decode_paged(batch, B, q.cuda(), kpool.cuda(), vpool.cuda(), dev(table), seql, dev(idx), dev(cnt),
                                   tau, scale, out_p, None, ws)
    sw.sw_sparse_attn_decode(batch, B, q.cuda(), kc.cuda(), vc.cuda(), seql, dev(idx), dev(cnt), tau, scale, out_c,
                             None, ws)
    assert torch.equal(out_p, out_c)
    got = out_p.float().cpu().numpy()
    assert np.isfinite(got).all()
    for s_, t in enumerate(ts):
        ref = O.decode_attention(gen.to_numpy_f64(q[s_]), gen.to_numpy_f64(kc[s_, :t]), gen.to_numpy_f64(vc[s_, :t]),
                                 idx[s_, :cnt[s_]], B, scale)
        err = np.abs(got[s_] - ref)
        assert err.max() <= ATT_MAX and err.mean() <= ATT_MEAN, (err.max(), err.mean())


# ------------------------------------------------------------------------------ paper default s = 8, heavy tails
def heavy_tailed_sketches(seed, b, r, sigma=4.0, sink=6.0):
    """Sketch rows whose block-score rows are heavy-tailed: S ~ sigma N(0, 1) (spread of ~6 sigma >= 12 over a
    row, PAPER.md:117 Assumption 2.3) plus a sink column 0.  fp32."""
    rng = np.random.RandomState(seed)
    a = math.sqrt(sigma)
    qs = (rng.randn(b, r) * a).astype(np.float32)
    ks = (rng.randn(b, r) * a).astype(np.float32)
    qs[:, 0] = math.sqrt(sink) * r ** 0.25
    ks[:, 0] = 0.0
    ks[0, 0] = math.sqrt(sink) * r ** 0.25
    return qs, ks


@pytest.mark.parametrize("b", [128, 512, 1024])
@pytest.mark.parametrize("flags", [O.DEFAULT_FLAGS, O.DEFAULT_FLAGS | O.POW_MATRIX])
def test_selection_chain_paper_default_s8_heavy_tails(sw, b, flags):
    """Block scores -> walk -> top-tau at the paper's s = 8 on heavy-tailed score rows, three layers
    with R carried, against the fp64 oracle.  In fp32 W = A^8 leaves the normal range for A < ~2e-5 (reading
    P20 in DESIGN.md): such entries are <= 1e-37 of the row maximum, far inside the 1e-3 value tolerance, and
    the candidates they decide between are near-ties in north_star's sense (within 1e-3 of the row max of each
    other), which is what the set comparison allows.  The overlap with the oracle's lists stays >= 99 % all the same
    (measured 0.9916 .. 1.0000 per layer, profiles/overlap_r3.md) and is asserted."""
    r, B, s, layers = 64, 64, 8, 3
    if flags & O.POW_MATRIX:
        s = 3
    tau = O.tau_from_density(0.10, b)
    L = sw.make_layout([b * B], B)
    ws = torch.empty(sw.sw_workspace_bytes(sw.SW_OP_WALK_UPDATE, L), dtype=torch.uint8, device="cuda")
    R_prev_gpu, R_ref = None, None
    overlaps = []
    tau_d = dev(np.asarray([tau], np.int32))
    for layer in range(layers):
        qs, ks = heavy_tailed_sketches(50 + layer, b, r)
        S = O.block_scores(qs.astype(np.float64), ks.astype(np.float64))
        assert np.ptp(S[b - 1]) >= 12.0
        A_ref = O.masked_softmax(S, flags)
        W_ref = A_ref if (flags & O.POW_MATRIX) else O.power(A_ref, s, flags)
        R_ref = O.walk_update(R_ref, A_ref, s, flags)
        W = torch.empty(L.total_sq, device="cuda"); R = torch.empty(L.total_sq, device="cuda")
        sw.sw_block_scores(L, dev(qs), dev(ks), r, s, flags, W, None)
        sw.sw_walk_update(L, R_prev_gpu, W, s, flags, R, ws)
        idx = torch.empty(b, tau, dtype=torch.int32, device="cuda"); cnt = torch.empty(b, dtype=torch.int32, device="cuda")
        sw.sw_select_topk(L, R, tau_d, tau, flags, idx, cnt)
        torch.cuda.synchronize()
        assert rowwise_close(W.cpu().numpy().reshape(b, b), W_ref)
        assert rowwise_close(R.cpu().numpy().reshape(b, b), R_ref)
        idx_ref, cnt_ref = O.select_topk(R_ref, tau, flags)
        idx_g, cnt_g = idx.cpu().numpy(), cnt.cpu().numpy()
        assert np.array_equal(cnt_g, cnt_ref)
        overlaps.append(sum(len(set(idx_g[i, :cnt_g[i]].tolist()) & set(idx_ref[i, :cnt_ref[i]].tolist()))
                            for i in range(b)) / int(cnt_ref.sum()))
        for i in range(b):
            assert near_tie_only(idx_g[i, :cnt_g[i]], idx_ref[i, :cnt_ref[i]], R_ref[i], {0, i}), (layer, i)
            # everything the oracle ranks clearly above the cut is selected by the GPU too
            clear = [j for j in idx_ref[i, :cnt_ref[i]] if R_ref[i, j] > 2 * REL * np.abs(R_ref[i]).max()]
            assert set(clear) <= set(idx_g[i, :cnt_g[i]].tolist())
        R_prev_gpu = R
    record_overlap("test_selection_chain_paper_default_s8_heavy_tails",
                   f"b={b} s={s} {'matrix power' if flags & O.POW_MATRIX else 'element-wise power'}", overlaps)
    assert min(overlaps) >= 0.99, overlaps


# ------------------------------------------------------------------------------ decode selection path
def near_tie_only(got, sel, ref_r, forced):
    """Selected sets may differ only at near-ties: every index in the symmetric difference lies within
    1e-3 of the row max of the lowest selected free score (north_star)."""
    got = np.asarray(got); sel = np.asarray(sel)
    if np.array_equal(got, sel):
        return True
    free = [j for j in sel.tolist() if j not in forced]
    kth = min(ref_r[free]) if free else 0.0
    scale = np.abs(ref_r).max()
    return all(abs(ref_r[j] - kth) <= REL * scale for j in set(got.tolist()) ^ set(sel.tolist()))


def decode_case(sw, t, tau, fused, flags, B=64, s=None, layers=3, scale_q=1.0):
    """GPU decode selection against the oracle's literal full-matrix Alg. 2, ``layers`` layers with the walk row
    carried, caches built by the GPU prefill path."""
    cfg = gen.CONFIGS[2]
    r, d, h_q, h_kv = cfg.r, cfg.d, 8, 2
    s = cfg.s if s is None else s
    signs, cols, H = H_of(d, r, seed=3)
    n_pre = t - 1
    b_pre, mb = O.num_blocks(n_pre, B), O.num_blocks(t, B)
    dp = sw.DecodePipeline(1, mb, h_q, h_kv, d, B, r, s, [tau], signs, cols, flags)
    R_full = None
    bq = (t - 1) // B
    forced = {bq} | ({0} if flags & O.FORCE_FIRST else set())
    for layer in range(layers):
        torch.manual_seed(100 + layer)
        Q = ((torch.randn(t, h_q, d) + 0.5) * scale_q).bfloat16(); K = (torch.randn(t, h_kv, d) + 0.5).bfloat16()
        # caches from the GPU prefill selection path over the first t-1 tokens
        pp = sw.PrefillPipeline([n_pre], h_q, h_kv, d, B, r, s, [O.tau_from_density(0.5, O.num_blocks(n_pre, B))], signs,
                                cols, flags)
        pp.select(Q[:n_pre].cuda(), K[:n_pre].cuda())
        kbar = torch.zeros(1, mb, d, device="cuda"); ks = torch.zeros(1, mb, r, device="cuda")
        kbar[0, :b_pre] = pp.kbar; ks[0, :b_pre] = pp.ks
        Wc = torch.zeros(1, mb, mb, device="cuda")
        Wc[0, :b_pre, :b_pre] = pp.W.view(b_pre, b_pre)
        seqlens = dev(np.asarray([t], np.int32))
        dp.select(Q[t - 1:t].cuda(), K[t - 1:t].cuda(), seqlens, kbar, ks, Wc, fused=fused)
        torch.cuda.synchronize()
        # oracle, literal
        Qn, Kn = gen.to_numpy_f64(Q), gen.to_numpy_f64(K)
        pre = O.prefill_selection(Qn[:n_pre], Kn[:n_pre], None, B=B, H_d=H, s=s, tau=tau, flags=flags)
        sel, R_full, cache2 = O.decode_layer_literal(Qn[t - 1], Kn[t - 1], O.DecodeCache(pre.qbar, pre.kbar, pre.S), t,
                                                     R_full, B=B, H_d=H, s=s, tau=tau, flags=flags)
        assert rowwise_close(kbar[0].cpu().numpy(), cache2.kbar)
        r_gpu = dp.rvec[dp.cur][0].cpu().numpy()
        assert rowwise_close(r_gpu[None, :bq + 1], R_full[bq][None, :bq + 1]), \
            np.abs(r_gpu[:bq + 1] - R_full[bq][:bq + 1]).max() / np.abs(R_full[bq]).max()
        assert (r_gpu[bq + 1:] == 0).all()
        got = dp.idx[0, :dp.count[0].item()].cpu().numpy()
        assert dp.count[0].item() == len(sel) and (dp.idx[0, len(sel):] == -1).all()
        assert near_tie_only(got, sel, R_full[bq], forced), (got, sel)
        assert bq in got


@pytest.mark.parametrize("fused", [True, False])
@pytest.mark.parametrize("t,tau", [(64 * 5 + 1, 4), (64 * 5 + 32, 4), (64 * 6, 4), (64 * 70 + 9, 12),
                                   (64 * 300 + 1, 40), (64 * 301, 40),
                                   # max_blocks % 4 == 0: the cp.async ring of the fused kernel (else plain loads)
                                   (64 * 7 + 3, 4), (64 * 71 + 9, 12), (64 * 299 + 5, 40), (64 * 300, 40),
                                   # b_q a multiple of 64: the column tile of b_q has no row of the cached W
                                   (64 * 64 + 1, 12), (64 * 128 + 17, 30),
                                   # block size 128 (given as a negative t: |t| tokens)
                                   (-(128 * 9 + 77), 4), (-(128 * 40), 9)])
def test_decode_selection_matches_literal_alg2(sw, t, tau, fused):
    """GPU decode selection -- the fused sw_decode_select launch, or the five row-vector calls (sketch_append x2,
    block_scores_row, walk_update_row, select_topk_row) -- against the oracle's literal full-matrix Alg. 2,
    three layers, caches built by the GPU prefill path.  The larger t span several column tiles and CTAs."""
    B = 64
    if t < 0:
        t, B = -t, 128
    decode_case(sw, t, tau, fused, O.DEFAULT_FLAGS, B=B)


@pytest.mark.parametrize("fused", [True, False])
@pytest.mark.parametrize("flags", [O.DEFAULT_FLAGS & ~O.SCORE_SOFTMAX, O.DEFAULT_FLAGS & ~O.FORCE_FIRST,
                                   O.DEFAULT_FLAGS & ~O.ROWNORM, O.CAUSAL | O.SCORE_SOFTMAX])
@pytest.mark.parametrize("t,tau", [(64 * 5 + 32, 4), (64 * 71 + 9, 12), (64 * 300, 40)])
def test_decode_selection_flag_variants(sw, t, tau, fused, flags):
    """The readings other than the default on the decode path: raw signed scores (P5), no forced first block
    (P7), no row rescale (P9), nothing forced but the current block."""
    decode_case(sw, t, tau, fused, flags)


@pytest.mark.parametrize("fused", [True, False])
@pytest.mark.parametrize("t,tau", [(64 * 71 + 9, 12), (64 * 300, 40)])
def test_decode_selection_paper_default_s8(sw, t, tau, fused):
    """The paper's walk exponent s = 8, element-wise, on the decode path."""
    decode_case(sw, t, tau, fused, O.DEFAULT_FLAGS, s=8)


def test_decode_select_non_causal_is_rejected(sw):
    """Alg. 2 Step 4(ii) is not carried by the row-vector form (P11): SW_ERR_UNSUPPORTED."""
    cfg = gen.CONFIGS[2]
    signs, cols, _ = H_of(cfg.d, cfg.r, seed=3)
    flags = O.DEFAULT_FLAGS & ~O.CAUSAL
    mb, t = 6, 64 * 5 + 7
    for fused in (True, False):
        dp = sw.DecodePipeline(1, mb, 8, 2, cfg.d, 64, cfg.r, 2, [3], signs, cols, flags)
        q = torch.randn(1, 8, cfg.d).bfloat16().cuda(); k = torch.randn(1, 2, cfg.d).bfloat16().cuda()
        kbar = torch.zeros(1, mb, cfg.d, device="cuda"); ks = torch.zeros(1, mb, cfg.r, device="cuda")
        Wc = torch.zeros(1, mb, mb, device="cuda")
        with pytest.raises(sw.SwError) as e:
            dp.select(q, k, dev(np.asarray([t], np.int32)), kbar, ks, Wc, fused=fused)
        assert e.value.code == sw.SW_ERR_UNSUPPORTED
        assert (Wc == 0).all()                               # the walk never ran
        if fused:
            assert (kbar == 0).all() and (ks == 0).all()     # nothing was launched


@pytest.mark.parametrize("nblk", [3, 299])
@pytest.mark.parametrize("fused", [True, False])
def test_decode_many_steps_across_a_block_boundary(sw, fused, nblk):
    """Twelve consecutive decode steps, two layers, caches carried on the GPU with no maintenance other
    than the calls themselves: the running key-block mean / sketch and the cached-W row of the current
    block (Alg. 2 Step 4) are updated in place, a block completes at step 7 and a new one starts at step 8.
    Every step is compared with the oracle's literal Alg. 2 carrying its own caches."""
    cfg = gen.CONFIGS[2]
    B, r, s, d, h_q, h_kv, tau, layers = cfg.B, cfg.r, cfg.s, cfg.d, 8, 2, 3, 2
    signs, cols, H = H_of(d, r, seed=3)
    flags = O.DEFAULT_FLAGS
    t0, steps = 64 * nblk + 58, 12                           # nblk = 299: 300 blocks, the cp.async W stream
    n_pre, t_end = t0 - 1, t0 + steps - 1
    b_pre, mb = O.num_blocks(n_pre, B), O.num_blocks(t_end, B)
    assert mb == b_pre + 1
    dp = sw.DecodePipeline(1, mb, h_q, h_kv, d, B, r, s, [tau], signs, cols, flags)
    torch.manual_seed(11)
    Q = [(torch.randn(t_end, h_q, d) + 0.5).bfloat16() for _ in range(layers)]
    K = [(torch.randn(t_end, h_kv, d) + 0.5).bfloat16() for _ in range(layers)]
    gpu, ora = [], []
    for l in range(layers):
        pp = sw.PrefillPipeline([n_pre], h_q, h_kv, d, B, r, s, [O.tau_from_density(0.5, O.num_blocks(n_pre, B))], signs,
                                cols, flags)
        pp.select(Q[l][:n_pre].cuda(), K[l][:n_pre].cuda())
        kbar = torch.zeros(1, mb, d, device="cuda"); ks = torch.zeros(1, mb, r, device="cuda")
        kbar[0, :b_pre] = pp.kbar; ks[0, :b_pre] = pp.ks
        Wc = torch.full((1, mb, mb), float("nan"), device="cuda")      # rows the calls must fill themselves
        Wc[0, :b_pre, :b_pre] = pp.W.view(b_pre, b_pre)
        Wc[0, :b_pre, b_pre:] = 0.0
        gpu.append((kbar, ks, Wc))
        pre = O.prefill_selection(gen.to_numpy_f64(Q[l][:n_pre]), gen.to_numpy_f64(K[l][:n_pre]), None, B=B, H_d=H,
                                  s=s, tau=tau, flags=flags)
        ora.append(O.DecodeCache(pre.qbar, pre.kbar, pre.S))
    for t in range(t0, t_end + 1):
        dp.reset()
        R_full = None
        seqlens = dev(np.asarray([t], np.int32))
        bq = (t - 1) // B
        for l in range(layers):
            kbar, ks, Wc = gpu[l]
            dp.select(Q[l][t - 1:t].cuda(), K[l][t - 1:t].cuda(), seqlens, kbar, ks, Wc, fused=fused)
            torch.cuda.synchronize()
            sel, R_full, ora[l] = O.decode_layer_literal(gen.to_numpy_f64(Q[l][t - 1]), gen.to_numpy_f64(K[l][t - 1]),
                                                         ora[l], t, R_full, B=B, H_d=H, s=s, tau=tau, flags=flags)
            assert rowwise_close(kbar[0, :bq + 1].cpu().numpy(), ora[l].kbar[:bq + 1])
            assert rowwise_close(dp.rvec[dp.cur][0, :bq + 1].cpu().numpy()[None], R_full[bq][None, :bq + 1])
            # the cached row of the current block is the new row of W (what a later step will read)
            W_ref = O.power(O.masked_softmax(ora[l].S, flags), s, flags)
            assert rowwise_close(Wc[0, bq, :bq + 1].cpu().numpy()[None], W_ref[bq][None, :bq + 1])
            assert (Wc[0, bq, bq + 1:] == 0).all()
            got = dp.idx[0, :dp.count[0].item()].cpu().numpy()
            if not np.array_equal(got, sel):                 # only near-ties may differ
                diff = set(got.tolist()) ^ set(sel.tolist())
                ref_r = R_full[bq]
                assert all(np.abs(ref_r[j] - np.sort(ref_r[1:bq])[::-1][tau - 3]) <= 1e-3 * np.abs(ref_r).max()
                           for j in diff)
            assert bq in got and len(got) == min(tau, bq + 1)


# ------------------------------------------------------------------------------ end to end
def check_overlap(idx_gpu, cnt_gpu, sel, R_ref):
    b = R_ref.shape[0]
    inter = tot = 0
    for i in range(b):
        g_ = set(idx_gpu[i, :cnt_gpu[i]].tolist()); o_ = set(sel.idx[i, :sel.count[i]].tolist())
        assert cnt_gpu[i] == sel.count[i]
        inter += len(g_ & o_); tot += len(o_)
        if g_ != o_:                                           # differences only at near-ties
            row = R_ref[i]; scale = np.abs(row).max()
            free = [j for j in o_ if j not in (0, i)]
            kth = min(row[free]) if free else 0.0
            for j in g_ ^ o_:
                assert abs(row[j] - kth) <= 1e-3 * scale, (i, j, row[j], kth)
    return inter / tot


def run_prefill_stack(sw, cfg_idx, seqlens, layers, *, flags=O.DEFAULT_FLAGS, s=None, density=None, fused=True):
    cfg = gen.CONFIGS[cfg_idx]
    s = cfg.s if s is None else s
    density = cfg.density if density is None else density
    seqlens = tuple(cfg.seqlens if seqlens is None else seqlens)
    signs, cols, H = H_of(cfg.d, cfg.r, seed=cfg_idx + 1)
    dtype = torch.float32 if cfg.dtype == "f32" else torch.bfloat16
    pipe = sw.PrefillPipeline(seqlens, cfg.h_q, cfg.h_kv, cfg.d, cfg.B, cfg.r, s,
                              [O.tau_from_density(density, O.num_blocks(n, cfg.B)) for n in seqlens], signs, cols,
                              flags=flags, dtype=dtype, keep_A=True)
    plans = gen.make_plans(cfg_idx, seqlens) if cfg.planted else None
    R_ref = [None] * len(seqlens)
    overlaps = []
    for layer in range(layers):
        li = gen.layer_inputs(cfg_idx, layer, device="cuda", seqlens=seqlens, plans=plans)
        out = pipe.layer(li.Q, li.K, li.V, fused=fused)
        torch.cuda.synchronize()
        Qn, Kn, Vn = (gen.to_numpy_f64(x) for x in (li.Q, li.K, li.V))
        idx_gpu, cnt_gpu = pipe.idx.cpu().numpy(), pipe.count.cpu().numpy()
        R_gpu = pipe.R_cur.cpu().numpy()
        got = out.float().cpu().numpy()
        tlo = blo = qlo = 0
        for si, n in enumerate(seqlens):
            b = O.num_blocks(n, cfg.B)
            tau = O.tau_from_density(density, b)
            sel = O.prefill_selection(Qn[tlo:tlo + n], Kn[tlo:tlo + n], R_ref[si], B=cfg.B, H_d=H, s=s, tau=tau, flags=flags)
            R_ref[si] = sel.R
            assert rowwise_close(pipe.qs[blo:blo + b].cpu().numpy(), sel.qs)
            assert rowwise_close(pipe.W[qlo:qlo + b * b].cpu().numpy().reshape(b, b), sel.A if flags & O.POW_MATRIX else sel.W)
            assert rowwise_close(R_gpu[qlo:qlo + b * b].reshape(b, b), sel.R)
            ov = check_overlap(idx_gpu[blo:blo + b], cnt_gpu[blo:blo + b], sel, sel.R)
            overlaps.append(ov)
            heads = sorted(set([0, cfg.h_q // 2, cfg.h_q - 1]))
            qb = torch.as_tensor(Qn[tlo:tlo + n]).bfloat16().double().numpy()
            kb = torch.as_tensor(Kn[tlo:tlo + n]).bfloat16().double().numpy()
            vb = torch.as_tensor(Vn[tlo:tlo + n]).bfloat16().double().numpy()
            ref = O.sparse_attention(qb, kb, vb, idx_gpu[blo:blo + b], cnt_gpu[blo:blo + b], cfg.B,
                                     1 / math.sqrt(cfg.d), flags=flags, q_heads=heads)
            err = np.abs(got[tlo:tlo + n][:, heads] - ref[:, heads])
            assert err.max() <= ATT_MAX and err.mean() <= ATT_MEAN, (err.max(), err.mean())
            tlo += n; blo += b; qlo += b * b
    return overlaps


@pytest.mark.parametrize("fused", [True, False])
@pytest.mark.parametrize("cfg_idx,seqlens,layers", [(0, None, 2), (1, (2048 + 19,), 4), (4, (192, 700, 1024), 3)])
def test_end_to_end_prefill_stack(sw, cfg_idx, seqlens, layers, fused):
    """Whole hot path, several layers with the walk carried across them; cfg 1 in full, cfg 2 / cfg 5 recipes
    at reduced length (full-size samples live in test_gpu_fullsize.py).  ``fused`` = sw_sketch_qk +
    sw_prefill_select, otherwise the plain calls."""
    ov = run_prefill_stack(sw, cfg_idx, seqlens, layers, fused=fused)
    record_overlap("test_end_to_end_prefill_stack", f"{gen.CONFIGS[cfg_idx].name} seqlens={seqlens} fused={fused}", ov)
    assert min(ov) >= 0.99, ov


@pytest.mark.parametrize("name,flags,s,density", [
    ("matrix power s=2 (P4, PAPER.md:25,31)", O.DEFAULT_FLAGS | O.POW_MATRIX, 2, 0.20),
    ("raw signed scores (P5, PAPER.md:782-784)", O.DEFAULT_FLAGS & ~O.SCORE_SOFTMAX, 2, 0.20),
    ("paper default s=8, r=64, 10% density (PAPER.md:218,266)", O.DEFAULT_FLAGS, 8, 0.10),
    ("no row rescale (P9 off)", O.DEFAULT_FLAGS & ~O.ROWNORM, 2, 0.20),
])
def test_end_to_end_prefill_stack_other_readings(sw, name, flags, s, density):
    """The readings other than the default, end to end (cfg-2 recipe, n ~ 4K, 3 layers with the walk carried):
    values within 1e-3 of the row max at every stage, selected sets equal to the oracle's up to near-ties
    (north_star), and north_star's >= 99 % overlap for every reading, the paper's default s = 8 and the raw-score
    reading included (measured 1.0000 on all four, profiles/overlap_r3.md)."""
    ov = run_prefill_stack(sw, 1, (4096 + 37,), 3, flags=flags, s=s, density=density)
    record_overlap("test_end_to_end_prefill_stack_other_readings", name, ov)
    assert min(ov) >= 0.99, (name, ov)
