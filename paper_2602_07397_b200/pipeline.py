"""Per-layer driver of the Sketch&Walk hot path: owns the device buffers and issues the six
C-ABI calls in the order of Alg. 1 / Alg. 2.  No arithmetic happens here."""
from __future__ import annotations

import math
from typing import Optional, Sequence

import numpy as np
import torch

from . import binding as sw


class PrefillPipeline:
    """Alg. 1 for a packed batch of sequences; the walk state R is carried across layers.  ``taus``: the block
    budget tau of every sequence (Alg. 1 Step 7), chosen by the caller -- like the C ABI, the driver takes tau as
    given and derives nothing from a density."""

    def __init__(self, seqlens: Sequence[int], h_q: int, h_kv: int, d: int, B: int, r: int, s: int,
                 taus: Sequence[int], signs: np.ndarray, cols: np.ndarray, flags: int = sw.SW_DEFAULT_FLAGS,
                 dtype: torch.dtype = torch.bfloat16, device: str = "cuda", keep_A: bool = False,
                 softmax_scale: Optional[float] = None):
        self.L = sw.make_layout(seqlens, B, device)
        self.h_q, self.h_kv, self.d, self.B, self.r, self.s = h_q, h_kv, d, B, r, s
        self.flags, self.dtype, self.device = flags, dtype, device
        self.softmax_scale = 1.0 / math.sqrt(d) if softmax_scale is None else softmax_scale
        self.sketch_scale = 1.0 / math.sqrt(r)
        self.signs = torch.as_tensor(np.asarray(signs, dtype=np.int8), device=device)
        self.cols = torch.as_tensor(np.asarray(cols, dtype=np.int32), device=device)
        if isinstance(taus, (int, float)) or len(taus) != len(self.L.blocks):
            raise sw.SwError(sw.SW_ERR_INVALID_ARG, "taus: one block budget per sequence")
        taus = [int(t) for t in taus]
        self.tau_max = max(taus)
        self.tau = torch.tensor(taus, dtype=torch.int32, device=device)
        L = self.L
        f32 = dict(dtype=torch.float32, device=device)
        self.qs = torch.empty(L.total_blocks, r, **f32)
        self.ks = torch.empty(L.total_blocks, r, **f32)
        self.qbar = torch.empty(L.total_blocks, d, **f32)
        self.kbar = torch.empty(L.total_blocks, d, **f32)
        self.W = torch.empty(L.total_sq, **f32)
        self.A = torch.empty(L.total_sq, **f32) if keep_A else None
        self.R = [torch.empty(L.total_sq, **f32), torch.empty(L.total_sq, **f32)]
        self.cur = -1                                   # index of the live R buffer (-1: none yet)
        self.idx = torch.empty(L.total_blocks, self.tau_max, dtype=torch.int32, device=device)
        self.count = torch.empty(L.total_blocks, dtype=torch.int32, device=device)
        # ping-pong matrix of the matrix-power reading + operand images of the tcgen05 walk GEMM
        nb = sw.sw_workspace_bytes(sw.SW_OP_WALK_UPDATE, L)
        self.walk_ws = torch.empty(nb, dtype=torch.uint8, device=device) if nb else None
        nb = sw.sw_workspace_bytes(sw.SW_OP_ATTN_PREFILL, L, h_q, h_kv, d, self.tau_max,
                                   sw.SW_F32 if dtype == torch.float32 else sw.SW_BF16)
        self.attn_ws = torch.empty(nb, dtype=torch.uint8, device=device) if nb else None

    def reset(self) -> None:
        self.cur = -1

    @property
    def R_cur(self) -> Optional[torch.Tensor]:
        return None if self.cur < 0 else self.R[self.cur]

    def select(self, Q: torch.Tensor, K: torch.Tensor, stream=None, fused: bool = True) -> None:
        """Steps 1-7: sketch -> block scores -> walk -> top-tau (idx / count updated in place).
        ``fused`` = sw_sketch_qk + sw_prefill_select (four launches); otherwise the plain calls."""
        L = self.L
        if fused and Q.dtype == K.dtype:
            sw.sw_sketch_qk(L, Q, K, self.signs, self.cols, self.r, self.sketch_scale, self.qs, self.ks, self.qbar,
                            self.kbar, stream)
            nxt = 0 if self.cur < 0 else 1 - self.cur
            sw.sw_prefill_select(L, self.qs, self.ks, self.r, self.s, self.flags, self.R_cur, self.R[nxt], self.W,
                                 self.A, self.tau, self.tau_max, self.idx, self.count, self.walk_ws, stream)
            self.cur = nxt
            return
        if Q.dtype == K.dtype:
            sw.sw_sketch_qk(L, Q, K, self.signs, self.cols, self.r, self.sketch_scale, self.qs, self.ks, self.qbar,
                            self.kbar, stream)
        else:
            sw.sw_sketch(L, Q, self.signs, self.cols, self.r, self.sketch_scale, self.qs, self.qbar, stream)
            sw.sw_sketch(L, K, self.signs, self.cols, self.r, self.sketch_scale, self.ks, self.kbar, stream)
        sw.sw_block_scores(L, self.qs, self.ks, self.r, self.s, self.flags, self.W, self.A, stream)
        nxt = 0 if self.cur < 0 else 1 - self.cur
        sw.sw_walk_update(L, self.R_cur, self.W, self.s, self.flags, self.R[nxt], self.walk_ws, stream)
        self.cur = nxt
        sw.sw_select_topk(L, self.R[nxt], self.tau, self.tau_max, self.flags, self.idx, self.count, stream)

    def attend(self, Q, K, V, out: Optional[torch.Tensor] = None, lse=None, stream=None) -> torch.Tensor:
        """Step 8: block-sparse attention over the blocks chosen by the last ``select``."""
        if out is None:
            out = torch.empty(self.L.total_tokens, self.h_q, self.d, dtype=Q.dtype, device=Q.device)
        sw.sw_sparse_attn_prefill(self.L, Q, K, V, self.idx, self.count, self.tau_max, self.softmax_scale,
                                  self.flags, out, lse, self.attn_ws, stream)
        return out

    def layer(self, Q, K, V, out=None, stream=None, fused: bool = True) -> torch.Tensor:
        self.select(Q, K, stream, fused)
        return self.attend(Q, K, V, out, None, stream)


class DecodePipeline:
    """Alg. 2 for a batch of sequences, one new token each.  Per layer the caller provides the
    caches (K/V cache, key-block means and sketches, cached W of the prefill); the row vector of the
    walk is carried across layers and restarts at every decode step."""

    def __init__(self, batch: int, max_blocks: int, h_q: int, h_kv: int, d: int, B: int, r: int, s: int,
                 taus: Sequence[int], signs: np.ndarray, cols: np.ndarray, flags: int = sw.SW_DEFAULT_FLAGS,
                 device: str = "cuda", softmax_scale: Optional[float] = None):
        self.batch, self.max_blocks = batch, max_blocks
        self.h_q, self.h_kv, self.d, self.B, self.r, self.s = h_q, h_kv, d, B, r, s
        self.flags, self.device = flags, device
        self.softmax_scale = 1.0 / math.sqrt(d) if softmax_scale is None else softmax_scale
        self.sketch_scale = 1.0 / math.sqrt(r)
        self.signs = torch.as_tensor(np.asarray(signs, dtype=np.int8), device=device)
        self.cols = torch.as_tensor(np.asarray(cols, dtype=np.int32), device=device)
        self.tau_max = int(max(taus))
        self.tau = torch.tensor(list(taus), dtype=torch.int32, device=device)
        f32 = dict(dtype=torch.float32, device=device)
        self.q_tok = torch.empty(batch, r, **f32)
        self.w_row = torch.empty(batch, max_blocks, **f32)
        self.rvec = [torch.empty(batch, max_blocks, **f32), torch.empty(batch, max_blocks, **f32)]
        self.cur = -1
        self.idx = torch.empty(batch, self.tau_max, dtype=torch.int32, device=device)
        self.count = torch.empty(batch, dtype=torch.int32, device=device)
        nb = sw.sw_decode_workspace_bytes(batch, h_q, h_kv, d, self.tau_max)
        self.attn_ws = torch.empty(max(nb, 16), dtype=torch.uint8, device=device)
        # sw_decode_select scratch (score row + partial sums handed between its three kernels)
        self.select_ws = torch.empty(sw.sw_decode_select_workspace_bytes(batch, max_blocks), dtype=torch.uint8,
                                     device=device)

    def reset(self) -> None:
        self.cur = -1

    def select(self, q, k_new, seqlens, kbar, ks, W_cache, stream=None, fused: bool = True) -> None:
        """q [batch,h_q,d], k_new [batch,h_kv,d]; kbar [batch,max_blocks,d], ks [batch,max_blocks,r]
        (updated in place for block b_curr); W_cache [batch,max_blocks,max_blocks].
        ``fused`` = one sw_decode_select launch (default); otherwise the five row-mode calls."""
        b, B, mb = self.batch, self.B, self.max_blocks
        if fused:
            nxt = 0 if self.cur < 0 else 1 - self.cur
            r_prev = None if self.cur < 0 else self.rvec[self.cur]
            sw.sw_decode_select(b, B, mb, q, k_new, seqlens, self.signs, self.cols, self.r, self.sketch_scale,
                                self.s, self.flags, kbar, ks, W_cache, W_cache.stride(0), r_prev, self.rvec[nxt],
                                self.tau, self.tau_max, self.idx, self.count, self.select_ws, stream)
            self.cur = nxt
            return
        sw.sw_sketch_append(b, B, mb, k_new, seqlens, self.signs, self.cols, self.r, self.sketch_scale,
                            kbar, ks, None, stream)
        sw.sw_sketch_append(b, B, mb, q, seqlens, self.signs, self.cols, self.r, self.sketch_scale,
                            None, None, self.q_tok, stream)
        sw.sw_block_scores_row(b, B, mb, self.q_tok, ks, seqlens, self.r, self.s, self.flags, self.w_row, stream)
        nxt = 0 if self.cur < 0 else 1 - self.cur
        r_prev = None if self.cur < 0 else self.rvec[self.cur]
        sw.sw_walk_update_row(b, B, mb, r_prev, W_cache, W_cache.stride(0), self.w_row, seqlens, self.flags,
                              self.rvec[nxt], stream)
        self.cur = nxt
        sw.sw_select_topk_row(b, B, mb, self.rvec[nxt], seqlens, self.tau, self.tau_max, self.flags, self.idx,
                              self.count, stream)

    def attend(self, q, kcache, vcache, seqlens, out=None, lse=None, stream=None) -> torch.Tensor:
        if out is None:
            out = torch.empty(self.batch, self.h_q, self.d, dtype=torch.bfloat16, device=q.device)
        sw.sw_sparse_attn_decode(self.batch, self.B, q, kcache, vcache, seqlens, self.idx, self.count,
                                 self.tau_max, self.softmax_scale, out, lse, self.attn_ws, stream)
        return out

    def attend_paged(self, q, kpool, vpool, block_table, seqlens, out=None, lse=None, stream=None) -> torch.Tensor:
        """Step 7 on a paged KV cache: pools [num_pages, B, h_kv, d], block_table [batch, max_blocks] int32."""
        if out is None:
            out = torch.empty(self.batch, self.h_q, self.d, dtype=torch.bfloat16, device=q.device)
        sw.sw_sparse_attn_decode_paged(self.batch, self.B, q, kpool, vpool, block_table, seqlens, self.idx, self.count,
                                       self.tau_max, self.softmax_scale, out, lse, self.attn_ws, stream)
        return out
