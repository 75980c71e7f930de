"""Pins for the CPU oracle (oracle/sw_oracle.py) against what the paper and the
mathematics fix -- never against itself.  Each test names the passage it pins."""
import itertools
import math
import os

import numpy as np
import pytest
import scipy.linalg
import scipy.special
import torch

from oracle import sw_oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")
RNG = np.random.RandomState(1234)


def read_golden(name):
    out = {}
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            parts = line.split()
            out[parts[0]] = np.asarray([float(x) for x in parts[1:]])
    return out


# --------------------------------------------------------------------- Hadamard
@pytest.mark.parametrize("d", [1, 2, 4, 8, 16, 64, 128])
def test_hadamard_orthogonality(d):
    # PAPER.md:435  W^T W = d I
    W = O.hadamard(d)
    assert np.array_equal(W @ W.T, d * np.eye(d))
    assert np.array_equal(W, W.T)
    assert set(np.unique(W)) <= {-1.0, 1.0}


@pytest.mark.parametrize("d", [2, 8, 64, 128])
def test_hadamard_is_sylvester_library(d):
    # natural (Sylvester) order == scipy.linalg.hadamard  (reading P2)
    assert np.array_equal(O.hadamard(d), scipy.linalg.hadamard(d).astype(np.float64))


def _fwht_butterfly(x):
    x = np.array(x, dtype=np.float64, copy=True)
    h = 1
    n = x.shape[-1]
    while h < n:
        for i in range(0, n, 2 * h):
            a = x[..., i:i + h].copy()
            b = x[..., i + h:i + 2 * h].copy()
            x[..., i:i + h] = a + b
            x[..., i + h:i + 2 * h] = a - b
        h *= 2
    return x


@pytest.mark.parametrize("d", [2, 4, 16, 128])
def test_matrix_product_equals_textbook_fwht(d):
    x = RNG.randn(5, d)
    W = O.hadamard(d)
    assert np.allclose(x @ W, _fwht_butterfly(x), rtol=0, atol=1e-11)
    assert np.allclose((x @ W) @ W, d * x, rtol=0, atol=1e-10)   # FWHT(FWHT(x)) = d x


def test_srht_matrix_structure():
    d, r = 16, 4
    signs = np.array([1, -1] * 8)
    cols = np.array([0, 3, 7, 12])
    H = O.srht_matrix(d, signs, cols, 1.0 / math.sqrt(r))
    W = scipy.linalg.hadamard(d)
    for x in range(d):
        for c in range(r):
            assert H[x, c] == signs[x] * W[x, cols[c]] / math.sqrt(r)
    # dropping D or transposing S would break H^T H = (d/r) I_r  (columns of D W are orthogonal)
    assert np.allclose(H.T @ H, (d / r) * np.eye(r))


# --------------------------------------------------------------------- pooling
def test_block_mean_bilinearity_def_a1():
    # Def. A.1: A_true[i,j] = 1/B^2 sum_s sum_t q_s . k_t  == qbar_i . kbar_j
    n, B, d = 48, 16, 8
    Q = RNG.randn(n, d); K = RNG.randn(n, d)
    qb, kb = O.block_mean(Q, B), O.block_mean(K, B)
    for i in range(3):
        for j in range(3):
            brute = 0.0
            for s in range(B):
                for t in range(B):
                    brute += Q[i * B + s] @ K[j * B + t]
            assert abs(qb[i] @ kb[j] - brute / B ** 2) < 1e-12


def test_block_mean_partial_last_block():
    # P12: divide by the number of valid tokens
    X = np.arange(10, dtype=np.float64)[:, None] * np.ones((1, 3))
    m = O.block_mean(X, 4)
    assert m.shape == (3, 3)
    assert np.allclose(m[:, 0], [1.5, 5.5, 8.5])


def test_head_mean():
    X = RNG.randn(7, 4, 5)
    ref = sum(X[:, u, :] for u in range(4)) / 4.0
    assert np.allclose(O.head_mean(X), ref, atol=1e-15)


# --------------------------------------------------------------------- sketch + scores
@pytest.mark.parametrize("d", [2, 8, 64])
def test_full_sketch_is_exact(d):
    # r = d (all columns, any signs): sqrt(r) * S == qbar . kbar exactly (orthogonality)
    b = 6
    qb, kb = RNG.randn(b, d), RNG.randn(b, d)
    signs = RNG.randint(0, 2, d) * 2 - 1
    H = O.srht_matrix(d, signs, np.arange(d), 1.0 / math.sqrt(d))
    S = O.block_scores(O.sketch(qb, H), O.sketch(kb, H))
    assert np.allclose(math.sqrt(d) * S, qb @ kb.T, atol=1e-12)


def test_srht_unbiased_over_all_subsets():
    # Lemma A.6 Step 3: E_S[(u^T H)(H^T v)] = u^T v, exact mean over all C(8, r)
    d = 8
    u, v = RNG.randn(d), RNG.randn(d)
    signs = np.array([1, -1, -1, 1, 1, 1, -1, 1])
    for r in (1, 2, 4):
        acc, cnt = 0.0, 0
        for cols in itertools.combinations(range(d), r):
            H = O.srht_matrix(d, signs, np.array(cols), 1.0 / math.sqrt(r))
            acc += (u @ H) @ (H.T @ v)
            cnt += 1
        assert abs(acc / cnt - u @ v) < 1e-12


def test_srht_error_shrinks_with_r():
    # Thm 2.5: error ~ 1/sqrt(r); statistical sanity check only
    d = 128
    errs = {}
    for r in (8, 32, 128):
        e = []
        for trial in range(40):
            rs = np.random.RandomState(trial)
            u, v = rs.randn(d), rs.randn(d)
            signs = rs.randint(0, 2, d) * 2 - 1
            cols = rs.choice(d, r, replace=False)
            H = O.srht_matrix(d, signs, cols, 1.0 / math.sqrt(r))
            e.append(abs((u @ H) @ (H.T @ v) - u @ v) / (np.linalg.norm(u) * np.linalg.norm(v)))
        errs[r] = np.mean(e)
    assert errs[8] > errs[32] > errs[128]
    assert errs[128] < 1e-12


def test_remark_a9_printed_numbers():
    # PAPER.md:553-559, fixture tests/golden/remark_a9.txt; r = d = 2, no signs
    g = read_golden("remark_a9.txt")
    d = 2
    H = O.srht_matrix(d, np.ones(d), np.arange(d), 1.0 / math.sqrt(d))
    qs = O.sketch(g["qbar_i"][None, :], H)
    ks = O.sketch(np.stack([g["kbar_j"], g["kbar_k"]]), H)
    S = math.sqrt(d) * O.block_scores(qs, ks)
    assert abs(S[0, 0] - g["dot_qi_kj"][0]) < 1e-12
    assert abs(S[0, 1] - g["dot_qi_kk"][0]) < 1e-12
    kj = O.sketch(g["kbar_j"][None, :], H)
    kk = O.sketch(g["kbar_k"][None, :], H)
    assert abs(math.sqrt(d) * O.block_scores(kj, kk)[0, 0] - g["dot_kj_kk"][0]) < 1e-12


def test_remark_a9_two_hop_walk_finds_k():
    # Blocks (causal order): k = 0, j = 1, i = 2.  Layer 0: i -> j strong, i -> k zero.
    # Layer 1: j -> k strong ("q_j . k_k for the next layer").  Raw scores, s = 1.
    g = read_golden("remark_a9.txt")
    flags = O.CAUSAL                                     # literal Alg. 1: no softmax, no rescale
    d = 2
    H = O.srht_matrix(d, np.ones(d), np.arange(d), 1.0 / math.sqrt(d))
    z = np.zeros(2)
    q0 = np.stack([z, z, g["qbar_i"]]); k0 = np.stack([g["kbar_k"], g["kbar_j"], z])
    q1 = np.stack([z, g["kbar_j"], z]); k1 = np.stack([g["kbar_k"], z, z])
    A0 = O.masked_softmax(O.block_scores(O.sketch(q0, H), O.sketch(k0, H)), flags)
    A1 = O.masked_softmax(O.block_scores(O.sketch(q1, H), O.sketch(k1, H)), flags)
    assert abs(A0[2, 0]) < 1e-15 and A0[2, 1] > 0.5     # one-hop misses k (dot = 0)
    R0 = O.walk_update(None, A0, 1, flags)
    R1 = O.walk_update(R0, A1, 1, flags)
    assert R1[2, 0] > 0.25                               # the walk reaches k through j
    assert abs(R1[2, 0] - A0[2, 1] * A1[1, 0]) < 1e-15


def test_complexity_example_arithmetic():
    g = read_golden("complexity_example.txt")
    B, tau, r = g["B"][0], g["tau"][0], g["r"][0]
    n, d = 32768, 128
    b = n / B
    red = B / (tau + r / (b * d))
    assert abs(red - g["reduction"][0]) < 0.01


def test_masked_softmax_properties():
    b = 9
    S = RNG.randn(b, b) * 3
    A = O.masked_softmax(S, O.DEFAULT_FLAGS)
    assert np.allclose(A.sum(axis=1), 1.0, atol=1e-14)
    assert np.array_equal(A[0], np.eye(b)[0])
    assert np.array_equal(np.triu(A, 1), np.zeros((b, b)))
    for i in range(b):                                   # library softmax on the unmasked prefix
        assert np.allclose(A[i, :i + 1], scipy.special.softmax(S[i, :i + 1]), atol=1e-15)
    A_nc = O.masked_softmax(S, O.SCORE_SOFTMAX)
    assert np.allclose(A_nc, scipy.special.softmax(S, axis=1), atol=1e-15)
    A_raw = O.masked_softmax(S, O.CAUSAL)
    assert np.array_equal(A_raw, np.tril(S))


def test_softmax_and_raw_select_identically_one_hop():
    # P5: softmax is monotone per row => for s = 1, a single layer, same selection
    b, tau = 12, 4
    S = RNG.randn(b, b)
    f_soft = O.DEFAULT_FLAGS
    f_raw = O.DEFAULT_FLAGS & ~O.SCORE_SOFTMAX
    i1, c1 = O.select_topk(O.walk_update(None, O.masked_softmax(S, f_soft), 1, f_soft), tau, f_soft)
    # raw scores can be negative while masked entries are 0 -> compare on candidates only (j <= i)
    R_raw = O.walk_update(None, O.masked_softmax(S, f_raw), 1, f_raw & ~O.ROWNORM)
    i2, c2 = O.select_topk(R_raw, tau, f_raw)
    assert np.array_equal(i1, i2) and np.array_equal(c1, c2)


# --------------------------------------------------------------------- walk
def test_walk_s1_identity_is_one_hop():
    # north_star: s = 1 and R^0 = I => the walk reduces to one-hop block scores
    b = 7
    A = O.masked_softmax(RNG.randn(b, b), O.DEFAULT_FLAGS)
    R = O.walk_update(None, A, 1, O.DEFAULT_FLAGS & ~O.ROWNORM)
    assert np.array_equal(R, A)
    Rm = O.walk_update(None, A, 1, (O.DEFAULT_FLAGS | O.POW_MATRIX) & ~O.ROWNORM)
    assert np.allclose(Rm, A, atol=1e-16)


@pytest.mark.parametrize("s", [1, 2, 3])
def test_walk_path_sum_identity(s):
    # R^k[i,j] = sum over paths of prod_l (A^l[m_l, m_{l+1}])^s
    b, L = 5, 3
    flags = O.DEFAULT_FLAGS & ~O.ROWNORM
    As = [O.masked_softmax(RNG.randn(b, b), flags) for _ in range(L)]
    R = None
    for A in As:
        R = O.walk_update(R, A, s, flags)
    for i in range(b):
        for j in range(b):
            tot = 0.0
            for m1 in range(b):
                for m2 in range(b):
                    tot += (As[0][i, m1] ** s) * (As[1][m1, m2] ** s) * (As[2][m2, j] ** s)
            assert abs(R[i, j] - tot) < 1e-13


def test_walk_is_product_of_w():
    # R^k = W^0 W^1 ... W^k  (numpy.linalg.multi_dot as the library routine)
    b, L, s = 8, 4, 2
    flags = O.DEFAULT_FLAGS & ~O.ROWNORM
    As = [O.masked_softmax(RNG.randn(b, b), flags) for _ in range(L)]
    R = None
    for A in As:
        R = O.walk_update(R, A, s, flags)
    ref = np.linalg.multi_dot([A ** s for A in As])
    assert np.allclose(R, ref, atol=1e-14)
    assert np.array_equal(np.triu(R, 1), np.zeros((b, b)))   # lower-triangularity preserved (P6)


def test_walk_matrix_power_mode():
    b, s = 6, 3
    flags = (O.DEFAULT_FLAGS | O.POW_MATRIX) & ~O.ROWNORM
    A = O.masked_softmax(RNG.randn(b, b), flags)
    R0 = O.masked_softmax(RNG.randn(b, b), flags)
    R = O.walk_update(R0, A, s, flags)
    assert np.allclose(R, R0 @ np.linalg.matrix_power(A, s), atol=1e-14)
    assert np.allclose(O.power(A, s, flags), np.linalg.matrix_power(A, s), atol=1e-14)
    assert np.allclose(O.power(A, s, O.DEFAULT_FLAGS), A * A * A, atol=1e-16)


def test_row_rescale_never_changes_selection():
    # P9: positive per-row scaling commutes with the walk and with top-tau
    b, L, s, tau = 16, 5, 2, 5
    f_on, f_off = O.DEFAULT_FLAGS, O.DEFAULT_FLAGS & ~O.ROWNORM
    As = [O.masked_softmax(RNG.randn(b, b) * 2, f_on) for _ in range(L)]
    R_on = R_off = None
    for A in As:
        R_on = O.walk_update(R_on, A, s, f_on)
        R_off = O.walk_update(R_off, A, s, f_off)
        assert np.array_equal(O.select_topk(R_on, tau, f_on)[0], O.select_topk(R_off, tau, f_off)[0])
        assert np.allclose(np.abs(R_on).max(axis=1), 1.0)
        ratio = R_off / np.where(R_on == 0, 1, R_on)
        for i in range(b):                               # each row differs by one positive scalar
            nz = R_on[i] != 0
            assert np.allclose(ratio[i, nz], ratio[i, nz][0], rtol=1e-10)


# --------------------------------------------------------------------- selection
def _brute_topk(row, cand_hi, forced, tau):
    budget = min(tau, cand_hi)
    forced = forced[:budget]
    rest = np.asarray([j for j in range(cand_hi) if j not in forced], dtype=np.int64)
    order = np.lexsort((rest, -row[rest]))               # library sort: score desc, index asc
    pick = rest[order][:budget - len(forced)]
    return sorted(list(forced) + pick.tolist())


@pytest.mark.parametrize("tau", [1, 2, 3, 5, 20])
def test_select_topk_brute_force(tau):
    b = 14
    R = np.tril(RNG.rand(b, b))
    idx, cnt = O.select_topk(R, tau, O.DEFAULT_FLAGS)
    for i in range(b):
        forced = [i] if i == 0 else [i, 0]
        ref = _brute_topk(R[i], i + 1, forced, tau)
        assert cnt[i] == min(tau, i + 1) == len(ref)
        assert idx[i, :cnt[i]].tolist() == ref
        assert (idx[i, cnt[i]:] == -1).all()
        sel = idx[i, :cnt[i]]
        assert len(set(sel.tolist())) == len(sel) and (np.diff(sel) > 0).all()
        if tau >= 2 and i >= 1:
            assert 0 in sel and i in sel
        if tau == 1:
            assert sel.tolist() == [i]                   # the diagonal block has priority (P7)


def test_select_topk_ties_lowest_index_first():
    b, tau = 8, 4
    R = np.tril(np.ones((b, b)))
    idx, cnt = O.select_topk(R, tau, O.DEFAULT_FLAGS)
    assert idx[7, :4].tolist() == [0, 1, 2, 7]
    assert idx[2, :3].tolist() == [0, 1, 2]
    R[7, 5] = 2.0
    assert O.select_topk(R, tau, O.DEFAULT_FLAGS)[0][7, :4].tolist() == [0, 1, 5, 7]


def test_select_topk_noncausal_and_noforce():
    b, tau = 6, 2
    R = RNG.rand(b, b)
    idx, cnt = O.select_topk(R, tau, 0)
    for i in range(b):
        assert idx[i].tolist() == sorted(np.argsort(-R[i], kind="stable")[:tau].tolist())
    assert (cnt == tau).all()


def test_select_row_decode_contains_current_block():
    # TopK(R[b_q, 1:b_curr], tau-1) U {b_curr}
    b = 10
    r = RNG.rand(b)
    for b_q in (0, 1, 5, 9):
        for tau in (1, 3, 7):
            sel = O.select_topk_row(r, b_q, tau, O.DEFAULT_FLAGS)
            assert b_q in sel and len(sel) == min(tau, b_q + 1)
            assert (sel <= b_q).all()
            sel_nf = O.select_topk_row(r, b_q, tau, O.DEFAULT_FLAGS & ~O.FORCE_FIRST)
            others = [j for j in sel_nf if j != b_q]
            ref = np.argsort(-r[:b_q], kind="stable")[:max(0, min(tau, b_q + 1) - 1)]
            assert sorted(others) == sorted(ref.tolist())


def test_tau_from_density():
    assert O.tau_from_density(0.25, 16) == 4             # BASELINE.json cfg 1
    assert O.tau_from_density(0.20, 512) == 103
    assert O.tau_from_density(0.20, 2048) == 410
    assert O.tau_from_density(1.0, 16) == 16
    assert O.tau_from_density(0.001, 16) == 1


# --------------------------------------------------------------------- attention
def _sdpa_dense_causal(Q, K, V, scale, causal=True):
    """Library routine: torch scaled_dot_product_attention in fp64, GQA by repeat."""
    q = torch.from_numpy(Q).permute(1, 0, 2)[None]
    grp = Q.shape[1] // K.shape[1]
    k = torch.from_numpy(K).permute(1, 0, 2).repeat_interleave(grp, dim=0)[None]
    v = torch.from_numpy(V).permute(1, 0, 2).repeat_interleave(grp, dim=0)[None]
    o = torch.nn.functional.scaled_dot_product_attention(q, k, v, is_causal=causal, scale=scale)
    return o[0].permute(1, 0, 2).numpy()


@pytest.mark.parametrize("n,B", [(96, 16), (100, 16), (37, 64)])
def test_full_density_equals_dense_causal_attention(n, B):
    # north_star: at 100% density the sparse output equals brute-force dense softmax attention
    hq, hkv, d = 4, 2, 8
    Q, K, V = RNG.randn(n, hq, d), RNG.randn(n, hkv, d), RNG.randn(n, hkv, d)
    b = O.num_blocks(n, B)
    R = np.tril(RNG.rand(b, b))
    idx, cnt = O.select_topk(R, b, O.DEFAULT_FLAGS)
    assert (cnt == np.arange(1, b + 1)).all()
    scale = 1.0 / math.sqrt(d)
    out = O.sparse_attention(Q, K, V, idx, cnt, B, scale)
    assert np.allclose(out, _sdpa_dense_causal(Q, K, V, scale), atol=1e-12)


def test_full_density_noncausal():
    n, B, hq, hkv, d = 64, 16, 2, 1, 4
    Q, K, V = RNG.randn(n, hq, d), RNG.randn(n, hkv, d), RNG.randn(n, hkv, d)
    b = n // B
    idx, cnt = O.select_topk(RNG.rand(b, b), b, 0)
    out = O.sparse_attention(Q, K, V, idx, cnt, B, 0.5, flags=0)
    assert np.allclose(out, _sdpa_dense_causal(Q, K, V, 0.5, causal=False), atol=1e-12)


def test_sparse_attention_brute_force_per_token():
    # zero outside selected blocks, renormalised within -- token-by-token loops
    n, B, hq, hkv, d, tau = 80, 16, 2, 1, 4, 2
    Q, K, V = RNG.randn(n, hq, d), RNG.randn(n, hkv, d), RNG.randn(n, hkv, d)
    b = n // B
    idx, cnt = O.select_topk(np.tril(RNG.rand(b, b)), tau, O.DEFAULT_FLAGS)
    out = O.sparse_attention(Q, K, V, idx, cnt, B, 0.7)
    for t in range(n):
        i = t // B
        for u in range(hq):
            w, acc = [], []
            for j in idx[i, :cnt[i]]:
                for p in range(j * B, (j + 1) * B):
                    if p <= t:
                        w.append(math.exp(0.7 * float(Q[t, u] @ K[p, 0])))
                        acc.append(V[p, 0])
            w = np.asarray(w)
            ref = (w[:, None] * np.asarray(acc)).sum(0) / w.sum()
            assert np.allclose(out[t, u], ref, atol=1e-12)


def test_sparse_attention_probabilities_sum_to_one_and_order_invariance():
    n, B, hq, hkv, d, tau = 128, 16, 4, 2, 8, 3
    Q, K = RNG.randn(n, hq, d), RNG.randn(n, hkv, d)
    V1 = np.ones((n, hkv, d))
    b = n // B
    idx, cnt = O.select_topk(np.tril(RNG.rand(b, b)), tau, O.DEFAULT_FLAGS)
    out = O.sparse_attention(Q, K, V1, idx, cnt, B, 0.3)
    assert np.allclose(out, 1.0, atol=1e-13)              # sum_j P_ij = 1 over the selected keys
    V = RNG.randn(n, hkv, d)
    ref = O.sparse_attention(Q, K, V, idx, cnt, B, 0.3)
    idx_rev = idx.copy()
    for i in range(b):
        idx_rev[i, :cnt[i]] = idx[i, :cnt[i]][::-1]
    assert np.allclose(O.sparse_attention(Q, K, V, idx_rev, cnt, B, 0.3), ref, atol=1e-13)


def test_sparse_attention_lse_merge_of_disjoint_lists():
    n, B, hq, hkv, d = 128, 16, 2, 1, 8
    Q, K, V = RNG.randn(n, hq, d), RNG.randn(n, hkv, d), RNG.randn(n, hkv, d)
    b = n // B
    full_idx = np.tile(np.arange(b, dtype=np.int32), (b, 1)); full_cnt = np.full(b, b, np.int32)
    flags = 0                                              # bidirectional so both halves are non-empty
    ref = O.sparse_attention(Q, K, V, full_idx, full_cnt, B, 0.4, flags)
    ia = np.tile(np.arange(0, b // 2, dtype=np.int32), (b, 1)); ca = np.full(b, b // 2, np.int32)
    ib = np.tile(np.arange(b // 2, b, dtype=np.int32), (b, 1)); cb = np.full(b, b - b // 2, np.int32)
    oa, la = O.sparse_attention(Q, K, V, ia, ca, B, 0.4, flags, return_lse=True)
    ob, lb = O.sparse_attention(Q, K, V, ib, cb, B, 0.4, flags, return_lse=True)
    m = np.maximum(la, lb)
    wa, wb = np.exp(la - m), np.exp(lb - m)
    merged = (wa[..., None] * oa + wb[..., None] * ob) / (wa + wb)[..., None]
    assert np.allclose(merged, ref, atol=1e-12)


# --------------------------------------------------------------------- decode
def test_decode_attention_equals_prefill_row():
    n, B, hq, hkv, d, tau = 100, 16, 4, 2, 8, 3
    Q, K, V = RNG.randn(n, hq, d), RNG.randn(n, hkv, d), RNG.randn(n, hkv, d)
    b = O.num_blocks(n, B)
    idx, cnt = O.select_topk(np.tril(RNG.rand(b, b)), tau, O.DEFAULT_FLAGS)
    pre = O.sparse_attention(Q, K, V, idx, cnt, B, 0.35)
    t = n                                                   # last token
    sel = idx[b - 1, :cnt[b - 1]]
    dec = O.decode_attention(Q[t - 1], K[:t], V[:t], sel, B, 0.35)
    assert np.allclose(dec, pre[t - 1], atol=1e-12)


@pytest.mark.parametrize("t", [64 + 1, 64 + 9, 64 + 16, 5 * 16])
def test_decode_row_walk_equals_literal_alg2_row(t):
    # row b_q of the literal full-matrix Alg. 2 == the carried row vector r^k = r^{k-1} W^k
    B, hq, hkv, d, r, s, tau, L = 16, 4, 2, 8, 4, 2, 3, 3
    signs = RNG.randint(0, 2, d) * 2 - 1
    H = O.srht_matrix(d, signs, np.array([0, 2, 5, 7]), 1.0 / math.sqrt(r))
    flags = O.DEFAULT_FLAGS
    R_full, r_row = None, None
    b_q = (t - 1) // B
    for layer in range(L):
        Q = RNG.randn(t, hq, d); K = RNG.randn(t, hkv, d)
        pre = O.prefill_selection(Q[:t - 1], K[:t - 1], None, B=B, H_d=H, s=s, tau=tau, flags=flags)
        cache = O.DecodeCache(pre.qbar, pre.kbar, pre.S)
        sel, R_full, cache2 = O.decode_layer_literal(Q[t - 1], K[t - 1], cache, t, R_full,
                                                     B=B, H_d=H, s=s, tau=tau, flags=flags)
        # key rep of the current block equals the prefill definition over the first t tokens
        assert np.allclose(cache2.kbar, O.block_mean(O.head_mean(K[:t]), B), atol=1e-13)
        # row-vector form: rows < b_q come from the cached prefill scores, row b_q is the new row
        A = O.masked_softmax(cache2.S, flags)
        W = O.power(A, s, flags)
        r_row = O.decode_walk_row(r_row, W, b_q, flags)
        assert np.allclose(r_row, R_full[b_q], atol=1e-13)
        assert np.array_equal(O.select_topk_row(r_row, b_q, tau, flags), sel)
        assert b_q in sel
        # the new row really is the single-token estimate
        q_tilde = O.head_mean(Q[t - 1][None])[0] @ H
        a_new = (O.sketch(cache2.kbar, H) @ q_tilde) / math.sqrt(r)
        assert np.allclose(cache2.S[b_q, :b_q + 1], a_new[:b_q + 1], atol=1e-13)


@pytest.mark.parametrize("t", [3 * 16 + 1, 3 * 16 + 7, 4 * 16, 16 + 1])
@pytest.mark.parametrize("steps", [1, 3])
def test_decode_literal_column_update_and_running_query_mean(t, steps):
    """Alg. 2 Step 4(ii) ("update last column ... c_new = Q~ k~_{b_curr}") and the
    running mean of the decode-time q_avg (P11), pinned with CAUSAL off so that neither is masked out:
    after decoding tokens t .. t+steps-1 the cached score matrix must equal the block scores rebuilt from
    scratch over all tokens seen so far -- plain double loop S[i, j] = q~_i . k~_j / sqrt(r) on the block
    means of the raw tokens -- except row b_q, which holds the single-token row of the latest step
    (PAPER.md:814-821), and the cached query reps must equal the block means of Q."""
    B, hq, hkv, d, r, s, tau = 16, 4, 2, 8, 4, 2, 3
    rng = np.random.RandomState(100 * t + steps)
    signs = rng.randint(0, 2, d) * 2 - 1
    cols = np.array([1, 2, 4, 7])
    H = O.srht_matrix(d, signs, cols, 1.0 / math.sqrt(r))
    flags = O.SCORE_SOFTMAX | O.FORCE_FIRST | O.FORCE_LAST | O.ROWNORM       # CAUSAL off
    t_end = t + steps - 1
    Q, K = rng.randn(t_end, hq, d), rng.randn(t_end, hkv, d)
    pre = O.prefill_selection(Q[:t - 1], K[:t - 1], None, B=B, H_d=H, s=s, tau=tau, flags=flags)
    cache = O.DecodeCache(pre.qbar, pre.kbar, pre.S)
    for tt in range(t, t_end + 1):
        sel, R, cache = O.decode_layer_literal(Q[tt - 1], K[tt - 1], cache, tt, None, B=B, H_d=H, s=s, tau=tau,
                                               flags=flags)
        b = O.num_blocks(tt, B)
        b_q = (tt - 1) // B
        # from scratch, written out: head mean, block mean, explicit Hadamard sums, double loop
        qbar = np.zeros((b, d)); kbar = np.zeros((b, d))
        for i in range(b):
            lo, hi = i * B, min((i + 1) * B, tt)
            qbar[i] = Q[lo:hi].mean(axis=1).mean(axis=0)
            kbar[i] = K[lo:hi].mean(axis=1).mean(axis=0)
        assert np.allclose(cache.qbar, qbar, atol=1e-13)
        assert np.allclose(cache.kbar, kbar, atol=1e-13)

        def sk(v):
            return np.array([sum(v[x] * signs[x] * (-1) ** bin(x & c).count("1") for x in range(d)) for c in cols]) / math.sqrt(r)

        S = np.zeros((b, b))
        for i in range(b):
            for j in range(b):
                S[i, j] = sk(qbar[i]) @ sk(kbar[j]) / math.sqrt(r)
        # P11: a block that completed during decode keeps, left of and on the diagonal, the single-token row
        # of its last token (row b_q wins; the later column updates only write columns > i of that row)
        for i in range((t - 1) // B, b_q):
            q_last = Q[(i + 1) * B - 1].mean(axis=0)
            for j in range(i + 1):
                S[i, j] = sk(q_last) @ sk(kbar[j]) / math.sqrt(r)
        q_tok = Q[tt - 1].mean(axis=0)
        for j in range(b):
            S[b_q, j] = sk(q_tok) @ sk(kbar[j]) / math.sqrt(r)
        assert cache.S.shape == (b, b)
        assert np.allclose(cache.S, S, atol=1e-12), np.abs(cache.S - S).max()
        # the column really changed (the pin would be vacuous otherwise) unless the block has just started
        if b_q > 0 and (tt - 1) % B != 0:
            stale = sk(qbar[0]) @ sk(K[b_q * B:tt - 1].mean(axis=1).mean(axis=0)) / math.sqrt(r)
            assert abs(stale - S[0, b_q]) > 1e-9
        assert R.shape == (b, b) and b_q in sel


def test_prefill_layer_end_to_end_full_density_is_dense():
    n, B, hq, hkv, d, r = 128, 16, 4, 2, 8, 4
    Q, K, V = RNG.randn(n, hq, d), RNG.randn(n, hkv, d), RNG.randn(n, hkv, d)
    H = O.srht_matrix(d, np.ones(d), np.array([1, 2, 4, 6]), 0.5)
    out, sel = O.prefill_layer(Q, K, V, None, B=B, H_d=H, s=2, tau=n // B)
    assert np.allclose(out, _sdpa_dense_causal(Q, K, V, 1 / math.sqrt(d)), atol=1e-12)
    assert sel.R.shape == (8, 8)
