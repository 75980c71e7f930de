"""Sketch&Walk Attention -- plain CPU oracle (fp64, numpy).

TEST INFRASTRUCTURE ONLY.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this
module.  It shares no code with the CUDA path (``paper_2602_07397_b200/``) and
never imports it.  Everything is written out in the paper's order and notation
so that it can be checked against PAPER.md by eye; there is no blocking,
fusion or reordering beyond what the cited passage states.  All arithmetic is
fp64; inputs are the exact bf16/fp32 values handed to the GPU, widened.

Citations are ``PAPER.md:<line>`` of /root/reference/PAPER.md plus the section /
algorithm they fall in.  ``P<n>`` refers to the "readings" table in DESIGN.md
(points where the paper is silent, ambiguous or garbled).

Block indices are 0-based here (the paper is 1-based).

Pins (tests/test_oracle_pins.py; ``-m "not gpu"``):
  hadamard / srht_matrix ... H H^T = d I, scipy.linalg.hadamard,
                             butterfly FWHT, FWHT(FWHT(x)) = d x
  block_mean ............... bilinearity vs Def. A.1 brute force
  sketch / block_scores .... r = d  =>  sqrt(r) S == qbar.kbar exactly;
                             unbiasedness over all C(d,r) subsets;
                             Remark A.9 printed numbers (tests/golden/remark_a9.txt)
  masked_softmax ........... rows sum to 1 over j <= i, row 0 = e_0,
                             scipy.special.softmax
  power / walk_update ...... s=1,R_prev=None => R == A; path-sum enumeration
                             (PAPER.md:588,682); R^k == W^0...W^k
                             via numpy.linalg.multi_dot; triangularity
  select_topk .............. brute force np.lexsort; forced/unique/ascending/ties
  sparse_attention ......... 100% density == dense causal softmax attention
                             (torch SDPA fp64); rows of P sum to 1;
                             order invariance; LSE merge of disjoint lists
  decode_* ................. decode output == row t of prefill attention given the
                             same S; row-vector walk == row b_q of literal Alg. 2;
                             column update + running query mean of Alg. 2 Step 4
                              == block scores rebuilt from scratch
                             with CAUSAL off (explicit double loop)
  PARITY UNPINNED (no printed number / closed form in the paper): the choice of
  readings P4 (element-wise power), P5 (softmax on block scores), P7 (forced
  blocks inside the tau budget), P9 (row rescale), P11 (row b_q wins), P13
  (tau = ceil(density b)) and whole-pipeline numeric values.  Each is a flag.
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import List, Optional, Tuple

import numpy as np

F64 = np.float64

# flag bits -- same numeric values as include/sw.h (the values are part of the
# C ABI contract stated in SURVEY.md section 8(b); nothing is imported from the GPU side)
CAUSAL = 1
SCORE_SOFTMAX = 2
POW_MATRIX = 4
FORCE_FIRST = 8
FORCE_LAST = 16
ROWNORM = 32
DEFAULT_FLAGS = CAUSAL | SCORE_SOFTMAX | FORCE_FIRST | FORCE_LAST | ROWNORM


# --------------------------------------------------------------------------
# Feature-space sketch: Hadamard / SRHT   (sec 2.2)
# --------------------------------------------------------------------------
def hadamard(d: int) -> np.ndarray:
    """Unnormalised Walsh-Hadamard matrix W in natural (Sylvester) order,
    W[x, y] = (-1)^popcount(x & y), so that W W^T = d I.  (P2)"""
    assert d >= 1 and (d & (d - 1)) == 0, "d must be a power of two"
    W = np.empty((d, d), dtype=F64)
    for x in range(d):
        for y in range(d):
            W[x, y] = -1.0 if bin(x & y).count("1") & 1 else 1.0
    return W


def srht_matrix(d: int, signs: np.ndarray, cols: np.ndarray, scale: float) -> np.ndarray:
    """H_d = scale * D W S  in R^{d x r}  (Lemma A.6 Step 1).
    D = diag(signs) (Rademacher), W = hadamard(d), S picks the columns ``cols``.
    Reading P1: scale = 1/sqrt(r) with the unnormalised W makes
    (u^T H)(H^T v) an unbiased estimate of u^T v."""
    signs = np.asarray(signs, dtype=F64).reshape(d)
    cols = np.asarray(cols, dtype=np.int64)
    W = hadamard(d)
    return scale * (signs[:, None] * W)[:, cols]


# --------------------------------------------------------------------------
# Token-space sketch: head mean + block mean   (Alg. 1 Steps 1-3)
# --------------------------------------------------------------------------
def head_mean(X: np.ndarray) -> np.ndarray:
    """Step 1: X[T, h, d] -> X_avg[T, d] = (1/h) sum_u X[:, u, :]."""
    X = np.asarray(X, dtype=F64)
    return X.sum(axis=1) / X.shape[1]


def num_blocks(n: int, B: int) -> int:
    """b = ceil(n / B)."""
    return (n + B - 1) // B


def block_mean(X_avg: np.ndarray, B: int) -> np.ndarray:
    """Steps 2-3 (eq. PAPER.md:57): xbar_i = mean of the rows of
    block i.  Reading P12: a partial last block divides by its number of valid
    tokens (the count-based running mean of Alg. 2)."""
    X_avg = np.asarray(X_avg, dtype=F64)
    n, d = X_avg.shape
    b = num_blocks(n, B)
    out = np.zeros((b, d), dtype=F64)
    for i in range(b):
        lo, hi = i * B, min((i + 1) * B, n)
        out[i] = X_avg[lo:hi].sum(axis=0) / (hi - lo)
    return out


def sketch(xbar: np.ndarray, H_d: np.ndarray) -> np.ndarray:
    """Step 4: xtilde = xbar H_d in R^{b x r}."""
    return np.asarray(xbar, dtype=F64) @ np.asarray(H_d, dtype=F64)


# --------------------------------------------------------------------------
# Block scores   (Alg. 1 Step 5; eq. PAPER.md:69)
# --------------------------------------------------------------------------
def block_scores(qs: np.ndarray, ks: np.ndarray) -> np.ndarray:
    """S = Qtilde Ktilde^T / sqrt(r)   (divide by sqrt(r) once: reading P3)."""
    r = qs.shape[1]
    return (np.asarray(qs, F64) @ np.asarray(ks, F64).T) / math.sqrt(r)


def masked_softmax(S: np.ndarray, flags: int = DEFAULT_FLAGS) -> np.ndarray:
    """Readings P5, P6.  With CAUSAL, entries j > i are masked.  With
    SCORE_SOFTMAX, A[i, :] = softmax over the unmasked j of S[i, :] (masked -> 0);
    without it A = S with masked entries set to 0 (literal Alg. 1)."""
    S = np.asarray(S, dtype=F64)
    bq, bk = S.shape
    A = np.zeros_like(S)
    for i in range(bq):
        hi = min(i + 1, bk) if (flags & CAUSAL) else bk
        row = S[i, :hi]
        if flags & SCORE_SOFTMAX:
            e = np.exp(row - row.max())
            A[i, :hi] = e / e.sum()
        else:
            A[i, :hi] = row
    return A


def power(A: np.ndarray, s: int, flags: int = DEFAULT_FLAGS) -> np.ndarray:
    """Step 6a: W = (A)^s.  Reading P4: element-wise by default
    (PAPER.md:784); POW_MATRIX gives the s-fold matrix product
    (Fig. 2)."""
    assert s >= 1
    A = np.asarray(A, dtype=F64)
    if flags & POW_MATRIX:
        W = A.copy()
        for _ in range(s - 1):
            W = W @ A
        return W
    return A ** s


# --------------------------------------------------------------------------
# Sketch-Determined Walk   (sec 2.3 eq. PAPER.md:77; Lemma A.11 PAPER.md:571-576;
#                           Alg. 1 Step 6 PAPER.md:783-787)
# --------------------------------------------------------------------------
def row_rescale(R: np.ndarray) -> np.ndarray:
    """Reading P9: divide every row by its max-abs (all-zero rows untouched).
    A positive per-row scale never changes any later top-tau."""
    R = np.array(R, dtype=F64, copy=True)
    for i in range(R.shape[0]):
        m = np.abs(R[i]).max() if R.shape[1] else 0.0
        if m > 0:
            R[i] /= m
    return R


def walk_update(R_prev: Optional[np.ndarray], A: np.ndarray, s: int,
                flags: int = DEFAULT_FLAGS) -> np.ndarray:
    """R^k = R^{k-1} W^k with W^k = (A^k)^s; R_prev=None is the identity so that
    R^0 = W^0 (P10).  In POW_MATRIX mode the product is
    taken as R <- R A, s times (same value as R (A^s)).  ROWNORM applies
    ``row_rescale`` after the update (P9)."""
    A = np.asarray(A, dtype=F64)
    b = A.shape[0]
    R = np.eye(b, dtype=F64) if R_prev is None else np.asarray(R_prev, dtype=F64)
    if flags & POW_MATRIX:
        for _ in range(s):
            R = R @ A
    else:
        R = R @ power(A, s, flags)
    if flags & ROWNORM:
        R = row_rescale(R)
    return R


# --------------------------------------------------------------------------
# Top-tau selection   (Alg. 1 Step 7 PAPER.md:788-791; P7, P8)
# --------------------------------------------------------------------------
def tau_from_density(density: float, b: int) -> int:
    """Reading P13: tau = max(1, ceil(density * b))."""
    return max(1, int(math.ceil(density * b - 1e-12)))


def _select_row(scores: np.ndarray, cand_hi: int, forced: List[int], tau: int) -> List[int]:
    """forced (priority order, truncated to the budget) + top-(rest) of the
    remaining candidates [0, cand_hi) by (score desc, index asc); NaN = -inf.
    Returns ascending indices."""
    budget = min(tau, cand_hi)
    forced = [f for f in forced if 0 <= f < cand_hi]
    uniq: List[int] = []
    for f in forced:
        if f not in uniq:
            uniq.append(f)
    forced = uniq[:budget]
    rest = [j for j in range(cand_hi) if j not in forced]
    need = budget - len(forced)

    def key(j):
        v = scores[j]
        if np.isnan(v):
            v = -np.inf
        return (-v, j)

    rest.sort(key=key)
    return sorted(forced + rest[:need])


def select_topk(R: np.ndarray, tau: int, flags: int = DEFAULT_FLAGS
                ) -> Tuple[np.ndarray, np.ndarray]:
    """Step 7 for every query block i of a square R.
    Candidates: j <= i with CAUSAL (P6) else all j.  Forced blocks count inside
    the budget (P7): the diagonal ("last", FORCE_LAST) block first, then block 0
    (FORCE_FIRST).  Output idx[b, tau] ascending, padded with -1; count[b]."""
    R = np.asarray(R, dtype=F64)
    b = R.shape[0]
    idx = np.full((b, tau), -1, dtype=np.int32)
    cnt = np.zeros((b,), dtype=np.int32)
    for i in range(b):
        cand_hi = i + 1 if (flags & CAUSAL) else R.shape[1]
        forced = []
        if flags & FORCE_LAST:
            forced.append(i)
        if flags & FORCE_FIRST:
            forced.append(0)
        sel = _select_row(R[i], cand_hi, forced, tau)
        cnt[i] = len(sel)
        idx[i, :len(sel)] = sel
    return idx, cnt


def select_topk_row(r: np.ndarray, b_q: int, tau: int, flags: int = DEFAULT_FLAGS) -> np.ndarray:
    """Alg. 2 Step 6: S = TopK(R[b_q, 0:b_curr], tau-1) U {b_curr},
    with block 0 also forced under FORCE_FIRST (P7).  b_curr == b_q."""
    r = np.asarray(r, dtype=F64)
    cand_hi = b_q + 1 if (flags & CAUSAL) else r.shape[0]
    forced = [b_q]                       # the current block is always kept
    if flags & FORCE_FIRST:
        forced.append(0)
    return np.asarray(_select_row(r, cand_hi, forced, tau), dtype=np.int32)


# --------------------------------------------------------------------------
# Block-sparse attention   (Alg. 1 Step 8 PAPER.md:792)
# --------------------------------------------------------------------------
def sparse_attention(Q: np.ndarray, K: np.ndarray, V: np.ndarray, idx: np.ndarray,
                     count: np.ndarray, B: int, softmax_scale: float,
                     flags: int = DEFAULT_FLAGS,
                     q_blocks: Optional[List[int]] = None,
                     q_heads: Optional[List[int]] = None,
                     return_lse: bool = False):
    """Per-head softmax attention on the original Q/K/V restricted to the tokens
    of the selected key blocks S_i: "zero outside selected blocks, renormalized
    within".  With CAUSAL a query at position t sees keys at
    positions <= t (token-causal inside the diagonal block, P6).  GQA (P14):
    q-head u reads kv-head u // (h_q / h_kv).

    Q[n, h_q, d], K,V[n, h_kv, d].  Returns O[n, h_q, d] (rows of unlisted
    q_blocks / q_heads stay 0) and optionally LSE[n, h_q] (natural log)."""
    Q = np.asarray(Q, F64); K = np.asarray(K, F64); V = np.asarray(V, F64)
    n, hq, d = Q.shape
    hkv = K.shape[1]
    grp = hq // hkv
    b = num_blocks(n, B)
    O = np.zeros((n, hq, V.shape[2]), dtype=F64)
    L = np.full((n, hq), -np.inf, dtype=F64)
    for i in (range(b) if q_blocks is None else q_blocks):
        qlo, qhi = i * B, min((i + 1) * B, n)
        sel = [int(j) for j in idx[i, :count[i]]]
        kpos = np.concatenate([np.arange(j * B, min((j + 1) * B, n)) for j in sel]) \
            if sel else np.zeros((0,), dtype=np.int64)
        qpos = np.arange(qlo, qhi)
        if flags & CAUSAL:
            mask = kpos[None, :] <= qpos[:, None]
        else:
            mask = np.ones((qhi - qlo, kpos.shape[0]), dtype=bool)
        for u in (range(hq) if q_heads is None else q_heads):
            g = u // grp
            s = (Q[qlo:qhi, u, :] @ K[kpos, g, :].T) * softmax_scale
            s = np.where(mask, s, -np.inf)
            m = s.max(axis=1, keepdims=True)
            m = np.where(np.isfinite(m), m, 0.0)
            p = np.exp(s - m)
            l = p.sum(axis=1, keepdims=True)
            safe = np.where(l > 0, l, 1.0)
            O[qlo:qhi, u, :] = (p / safe) @ V[kpos, g, :]
            L[qlo:qhi, u] = np.where(l[:, 0] > 0, m[:, 0] + np.log(safe[:, 0]), -np.inf)
    return (O, L) if return_lse else O


def decode_attention(q_t: np.ndarray, Kc: np.ndarray, Vc: np.ndarray, sel: np.ndarray,
                     B: int, softmax_scale: float) -> np.ndarray:
    """Alg. 2 Step 7: the new query token (position t-1, the last
    row of the cache) against the tokens of the selected cache blocks.
    q_t[h_q, d], Kc/Vc[t, h_kv, d] (cache already holds the new token)."""
    q_t = np.asarray(q_t, F64); Kc = np.asarray(Kc, F64); Vc = np.asarray(Vc, F64)
    t = Kc.shape[0]
    hq = q_t.shape[0]
    grp = hq // Kc.shape[1]
    kpos = np.concatenate([np.arange(j * B, min((j + 1) * B, t)) for j in sel])
    out = np.zeros((hq, Vc.shape[2]), dtype=F64)
    for u in range(hq):
        g = u // grp
        s = (Kc[kpos, g, :] @ q_t[u]) * softmax_scale
        p = np.exp(s - s.max())
        out[u] = (p / p.sum()) @ Vc[kpos, g, :]
    return out


# --------------------------------------------------------------------------
# Whole prefill layer   (Alg. 1)
# --------------------------------------------------------------------------
@dataclass
class LayerSelection:
    qbar: np.ndarray      # [b, d] block representatives (Step 3)
    kbar: np.ndarray
    qs: np.ndarray        # [b, r] sketches (Step 4)
    ks: np.ndarray
    S: np.ndarray         # raw sketched scores (Step 5)
    A: np.ndarray         # masked (softmax) block attention estimate (P5, P6)
    W: np.ndarray         # (A)^s
    R: np.ndarray         # walk state after this layer
    idx: np.ndarray       # [b, tau] selected key blocks, ascending, -1 padded
    count: np.ndarray


def prefill_selection(Q: np.ndarray, K: np.ndarray, R_prev: Optional[np.ndarray], *, B: int,
                      H_d: np.ndarray, s: int, tau: int,
                      flags: int = DEFAULT_FLAGS) -> LayerSelection:
    """Alg. 1 Steps 1-7 for one sequence of one layer."""
    qbar = block_mean(head_mean(Q), B)            # Steps 1-3
    kbar = block_mean(head_mean(K), B)
    qs = sketch(qbar, H_d)                        # Step 4
    ks = sketch(kbar, H_d)
    S = block_scores(qs, ks)                      # Step 5
    A = masked_softmax(S, flags)                  # P5, P6
    W = power(A, s, flags)                        # Step 6a
    R = walk_update(R_prev, A, s, flags)          # Step 6b
    idx, cnt = select_topk(R, tau, flags)         # Step 7
    return LayerSelection(qbar, kbar, qs, ks, S, A, W, R, idx, cnt)


def prefill_layer(Q, K, V, R_prev, *, B, H_d, s, tau, softmax_scale=None,
                  flags: int = DEFAULT_FLAGS):
    """Alg. 1 end to end: returns (O, LayerSelection)."""
    sel = prefill_selection(Q, K, R_prev, B=B, H_d=H_d, s=s, tau=tau, flags=flags)
    if softmax_scale is None:
        softmax_scale = 1.0 / math.sqrt(Q.shape[2])
    O = sparse_attention(Q, K, V, sel.idx, sel.count, B, softmax_scale, flags)
    return O, sel


# --------------------------------------------------------------------------
# Decode, literal full-matrix form of Alg. 2
# --------------------------------------------------------------------------
@dataclass
class DecodeCache:
    """Per-layer caches Alg. 2 takes as input."""
    qbar: np.ndarray      # [b_q, d] cached query-block reps
    kbar: np.ndarray      # [b_k, d] cached key-block reps (last one may be partial)
    S: np.ndarray         # cached raw block scores from prefill, [b_q, b_k]


def decode_layer_literal(q_t: np.ndarray, k_t: np.ndarray, cache: DecodeCache, t: int,
                         R_prev: Optional[np.ndarray], *, B: int, H_d: np.ndarray, s: int,
                         tau: int, flags: int = DEFAULT_FLAGS):
    """Alg. 2 Steps 2-6 in the literal full-matrix form for the token that brings
    the sequence length to ``t`` (1-based count; the cache tensors describe the
    first t-1 tokens).  q_t[h_q, d], k_t[h_kv, d].

    Returns (sel, R, cache') where sel are the selected blocks for this token,
    R the full b x b walk state and cache' the updated caches.

    Readings (P11): new K/V are inputs; the running mean uses count (t-1) mod B;
    row b_q wins over the column update; the column update touches rows < b_q;
    row b_q always uses the single-token sketch; a running mean of the decode-time
    q_avg is kept so that a completed block's cached rep equals the prefill one."""
    r = H_d.shape[1]
    b_curr = (t - 1) // B                       # 0-based current key block
    b_q = b_curr
    c = (t - 1) % B                             # tokens already in block b_curr
    k_avg = np.asarray(k_t, F64).sum(axis=0) / k_t.shape[0]
    q_avg = np.asarray(q_t, F64).sum(axis=0) / q_t.shape[0]
    d = k_avg.shape[0]
    kbar = np.array(cache.kbar, F64, copy=True)
    qbar = np.array(cache.qbar, F64, copy=True)
    Sc = np.array(cache.S, F64, copy=True)
    if c == 0:                                  # t mod B == 1: a new block starts
        kbar = np.vstack([kbar[:b_curr], k_avg[None, :]])
        qbar = np.vstack([qbar[:b_q], q_avg[None, :]])
        S = np.zeros((b_q + 1, b_curr + 1), dtype=F64)
        S[:b_q, :b_curr] = Sc[:b_q, :b_curr]
    else:                                       # running mean
        kbar[b_curr] = (c * kbar[b_curr] + k_avg) / (c + 1)
        qbar[b_q] = (c * qbar[b_q] + q_avg) / (c + 1)
        S = Sc
    # Step 3: sketch the single query token and all key reps
    q_tilde = q_avg @ H_d
    K_tilde = kbar @ H_d
    a_new = (K_tilde @ q_tilde) / math.sqrt(r)
    # Step 4: column first for rows < b_q, then the row (row wins)
    Q_tilde = qbar @ H_d
    c_new = (Q_tilde @ K_tilde[b_curr]) / math.sqrt(r)
    S[:b_q, b_curr] = c_new[:b_q]
    S[b_q, :b_curr + 1] = a_new
    # Step 5 with the same rule as prefill (P4, P5, P9)
    A = masked_softmax(S, flags)
    R = walk_update(R_prev, A, s, flags)
    sel = select_topk_row(R[b_q], b_q, tau, flags)               # Step 6
    return sel, R, DecodeCache(qbar, kbar, S)


def decode_walk_row(r_prev: Optional[np.ndarray], W: np.ndarray, b_q: int,
                    flags: int = DEFAULT_FLAGS) -> np.ndarray:
    """Row-vector form of the decode walk: r^k = r^{k-1} W^k with r^{-1} = e_{b_q}
    (row b_q of R_prev W depends only on row b_q of R_prev).  Used by the tests to
    show it equals row b_q of ``decode_layer_literal``.  W is already (A)^s
    (``power``); ROWNORM rescales the vector by its max-abs."""
    b = W.shape[0]
    if r_prev is None:
        r_prev = np.zeros((b,), dtype=F64)
        r_prev[b_q] = 1.0
    rr = np.asarray(r_prev, F64) @ np.asarray(W, F64)
    if flags & ROWNORM:
        m = np.abs(rr).max()
        if m > 0:
            rr = rr / m
    return rr
