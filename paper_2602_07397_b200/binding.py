"""Thin ctypes binding of libsw (include/sw.h).  Argument marshalling only: every step of the
path runs in the CUDA kernels behind the C ABI.  PyTorch is used for device memory and streams.

There is no CPU fallback: if ``libsw.so`` has not been built (``python -m
paper_2602_07397_b200.build`` or ``__graft_entry__.build()``) importing this module raises.
"""
from __future__ import annotations

import ctypes as C
import math
import os
from dataclasses import dataclass
from typing import Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsw.so")

# ---- constants (include/sw.h) --------------------------------------------------------------
SW_OK, SW_ERR_INVALID_ARG, SW_ERR_UNSUPPORTED, SW_ERR_WORKSPACE, SW_ERR_CUDA, SW_ERR_ARCH = 0, -1, -2, -3, -4, -5
SW_VERSION = 101
SW_BF16, SW_F32 = 0, 1
SW_CAUSAL, SW_SCORE_SOFTMAX, SW_POW_MATRIX, SW_FORCE_FIRST, SW_FORCE_LAST, SW_ROWNORM = 1, 2, 4, 8, 16, 32
SW_DEFAULT_FLAGS = SW_CAUSAL | SW_SCORE_SOFTMAX | SW_FORCE_FIRST | SW_FORCE_LAST | SW_ROWNORM
SW_PREFILL_AUTO, SW_PREFILL_GENERIC, SW_PREFILL_TCGEN05 = 0, 1, 2
SW_WALK_AUTO, SW_WALK_SIMT, SW_WALK_TCGEN05 = 0, 1, 2
SW_OP_SKETCH, SW_OP_BLOCK_SCORES, SW_OP_WALK_UPDATE, SW_OP_SELECT_TOPK, SW_OP_ATTN_PREFILL, SW_OP_ATTN_DECODE = range(6)

EXPORTS = [
    "sw_sketch", "sw_sketch_qk", "sw_sketch_from_pooled", "sw_copy_pool", "sw_sketch_append", "sw_block_scores", "sw_block_scores_row", "sw_walk_update",
    "sw_walk_update_row", "sw_select_topk", "sw_select_topk_row", "sw_prefill_select", "sw_decode_select", "sw_sparse_attn_prefill",
    "sw_sparse_attn_decode", "sw_sparse_attn_decode_paged", "sw_sparse_attn_decode_static", "sw_workspace_bytes", "sw_decode_workspace_bytes", "sw_decode_select_workspace_bytes", "sw_decode_num_splits",
    "sw_set_prefill_kernel", "sw_get_prefill_kernel_used", "sw_set_walk_kernel", "sw_get_walk_kernel_used",
    "sw_last_error", "sw_version", "sw_launch_count",
]


class SwError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libsw error {code}: {msg}")
        self.code = code


class _Tensor(C.Structure):
    _fields_ = [("ptr", C.c_void_p), ("dtype", C.c_int32), ("heads", C.c_int32), ("d", C.c_int32),
                ("stride_tok", C.c_int64), ("stride_head", C.c_int64)]


class _Layout(C.Structure):
    _fields_ = [("batch", C.c_int32), ("block", C.c_int32), ("total_tokens", C.c_int32),
                ("total_blocks", C.c_int32), ("max_blocks", C.c_int32), ("cu_seqlens", C.c_void_p),
                ("cu_blocks", C.c_void_p), ("cu_sq", C.c_void_p)]


def _load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2602_07397_b200.build` "
            "(libsw has no CPU or PyTorch fallback)")
    lib = C.CDLL(LIB_PATH)
    i32, i64, u32, f32, vp, sz = C.c_int32, C.c_int64, C.c_uint32, C.c_float, C.c_void_p, C.c_size_t
    LP, TP = C.POINTER(_Layout), C.POINTER(_Tensor)
    sig = {
        "sw_sketch": (i32, [LP, TP, vp, vp, i32, f32, vp, vp, vp]),
        "sw_sketch_qk": (i32, [LP, TP, TP, vp, vp, i32, f32, vp, vp, vp, vp, vp]),
        "sw_sketch_from_pooled": (i32, [LP, vp, i32, i32, vp, vp, i32, f32, vp, vp, vp]),
        "sw_copy_pool": (i32, [LP, TP, vp, vp, vp]),
        "sw_sketch_append": (i32, [i32, i32, i32, TP, vp, vp, vp, i32, f32, vp, vp, vp, vp]),
        "sw_block_scores": (i32, [LP, vp, vp, i32, i32, u32, vp, vp, vp]),
        "sw_block_scores_row": (i32, [i32, i32, i32, vp, vp, vp, i32, i32, u32, vp, vp]),
        "sw_walk_update": (i32, [LP, vp, vp, i32, u32, vp, vp, sz, vp]),
        "sw_walk_update_row": (i32, [i32, i32, i32, vp, vp, i64, vp, vp, u32, vp, vp]),
        "sw_select_topk": (i32, [LP, vp, vp, i32, u32, vp, vp, vp]),
        "sw_prefill_select": (i32, [LP, vp, vp, i32, i32, u32, vp, vp, vp, vp, vp, i32, vp, vp, vp, sz, vp]),
        "sw_select_topk_row": (i32, [i32, i32, i32, vp, vp, vp, i32, u32, vp, vp, vp]),
        "sw_decode_select": (i32, [i32, i32, i32, TP, TP, vp, vp, vp, i32, f32, i32, u32, vp, vp, vp, i64, vp, vp,
                                   vp, i32, vp, vp, vp, sz, vp]),
        "sw_sparse_attn_prefill": (i32, [LP, TP, TP, TP, vp, vp, i32, f32, u32, vp, vp, vp, sz, vp]),
        "sw_sparse_attn_decode": (i32, [i32, i32, TP, TP, TP, i64, vp, vp, vp, i32, f32, vp, vp, vp, sz, vp]),
        "sw_sparse_attn_decode_paged": (i32, [i32, i32, TP, TP, TP, i64, vp, i32, vp, vp, vp, i32, f32, vp, vp, vp, sz,
                                              vp]),
        "sw_sparse_attn_decode_static": (i32, [i32, i32, TP, TP, TP, i64, vp, vp, vp, i32, f32, vp, vp, vp]),
        "sw_workspace_bytes": (sz, [i32, LP, i32, i32, i32, i32, i32]),
        "sw_decode_workspace_bytes": (sz, [i32, i32, i32, i32, i32]),
        "sw_decode_select_workspace_bytes": (sz, [i32, i32]),
        "sw_decode_num_splits": (i32, [i32, i32, i32, i32]),
        "sw_set_prefill_kernel": (i32, [i32]),
        "sw_get_prefill_kernel_used": (i32, []),
        "sw_set_walk_kernel": (i32, [i32]),
        "sw_get_walk_kernel_used": (i32, []),
        "sw_last_error": (C.c_char_p, []),
        "sw_version": (i32, []),
        "sw_launch_count": (C.c_uint64, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    if lib.sw_version() != SW_VERSION:
        raise ImportError(f"{LIB_PATH} reports version {lib.sw_version()}, this binding is written for {SW_VERSION} "
                          "(include/sw.h): rebuild with `python -m paper_2602_07397_b200.build --force`")
    return lib


_lib = _load()


def _check(code: int) -> None:
    if code != SW_OK:
        raise SwError(code, _lib.sw_last_error().decode("utf-8", "replace"))


def _ptr(t: Optional[torch.Tensor]) -> Optional[int]:
    return None if t is None else t.data_ptr()


def _stream(stream: Optional[torch.cuda.Stream]) -> Optional[int]:
    if stream is not None:
        return stream.cuda_stream
    if torch.cuda.is_available():
        return torch.cuda.current_stream().cuda_stream
    return None


def _dtype_code(t: torch.Tensor) -> int:
    if t.dtype == torch.bfloat16:
        return SW_BF16
    if t.dtype == torch.float32:
        return SW_F32
    raise SwError(SW_ERR_UNSUPPORTED, f"dtype {t.dtype}")


def _tensor(t: torch.Tensor) -> _Tensor:
    """[tokens, heads, d] view with unit stride on d."""
    if t.dim() != 3 or t.stride(2) != 1:
        raise SwError(SW_ERR_INVALID_ARG, "expected a [tokens, heads, d] tensor with contiguous d")
    return _Tensor(t.data_ptr(), _dtype_code(t), t.shape[1], t.shape[2], t.stride(0), t.stride(1))


@dataclass
class Layout:
    """Packed varlen batch (host sizes + device offset arrays)."""
    batch: int
    block: int
    seqlens: Sequence[int]
    total_tokens: int
    total_blocks: int
    max_blocks: int
    total_sq: int
    cu_seqlens: torch.Tensor
    cu_blocks: torch.Tensor
    cu_sq: torch.Tensor
    blocks: Sequence[int]

    def c(self) -> _Layout:
        return _Layout(self.batch, self.block, self.total_tokens, self.total_blocks, self.max_blocks,
                       self.cu_seqlens.data_ptr(), self.cu_blocks.data_ptr(), self.cu_sq.data_ptr())


def make_layout(seqlens: Sequence[int], block: int, device="cuda") -> Layout:
    seqlens = [int(n) for n in seqlens]
    blocks = [(n + block - 1) // block for n in seqlens]
    cu_s, cu_b, cu_q = [0], [0], [0]
    for n, b in zip(seqlens, blocks):
        cu_s.append(cu_s[-1] + n)
        cu_b.append(cu_b[-1] + b)
        cu_q.append(cu_q[-1] + b * b)
    return Layout(len(seqlens), block, seqlens, cu_s[-1], cu_b[-1], max(blocks) if blocks else 0, cu_q[-1],
                  torch.tensor(cu_s, dtype=torch.int32, device=device),
                  torch.tensor(cu_b, dtype=torch.int32, device=device),
                  torch.tensor(cu_q, dtype=torch.int64, device=device), blocks)


# ---- the calls (same names as the C ABI) ------------------------------------------------------
def sw_version() -> int:
    return _lib.sw_version()


def sw_launch_count() -> int:
    """Kernels launched by libsw in this process so far."""
    return int(_lib.sw_launch_count())


def sw_set_prefill_kernel(which: int) -> int:
    prev = _lib.sw_set_prefill_kernel(which)
    if prev < 0:
        _check(prev)
    return prev


def sw_get_prefill_kernel_used() -> int:
    return _lib.sw_get_prefill_kernel_used()


def sw_set_walk_kernel(which: int) -> int:
    prev = _lib.sw_set_walk_kernel(which)
    if prev < 0:
        raise SwError(prev, _lib.sw_last_error().decode())
    return prev


def sw_get_walk_kernel_used() -> int:
    return _lib.sw_get_walk_kernel_used()


def sw_last_error() -> str:
    return _lib.sw_last_error().decode("utf-8", "replace")


def sw_sketch(L: Layout, x, signs, cols, r: int, scale: float, sketch, mean=None, stream=None) -> None:
    lay, xt = L.c(), _tensor(x)
    _check(_lib.sw_sketch(C.byref(lay), C.byref(xt), _ptr(signs), _ptr(cols), r, scale, _ptr(sketch),
                          _ptr(mean), _stream(stream)))


def sw_sketch_qk(L: Layout, q, k, signs, cols, r: int, scale: float, qs, ks, qbar=None, kbar=None, stream=None) -> None:
    lay, qt, kt = L.c(), _tensor(q), _tensor(k)
    _check(_lib.sw_sketch_qk(C.byref(lay), C.byref(qt), C.byref(kt), _ptr(signs), _ptr(cols), r, scale, _ptr(qs),
                             _ptr(ks), _ptr(qbar), _ptr(kbar), _stream(stream)))


def sw_sketch_from_pooled(L: Layout, sums, heads: int, signs, cols, r: int, scale: float, sketch, mean=None,
                          stream=None) -> None:
    """sums: fp32 [total_blocks, d] = per-block sums over heads and valid tokens (left behind by a producer)."""
    lay = L.c()
    _check(_lib.sw_sketch_from_pooled(C.byref(lay), _ptr(sums), heads, sums.shape[-1], _ptr(signs), _ptr(cols), r,
                                      scale, _ptr(sketch), _ptr(mean), _stream(stream)))


def sw_copy_pool(L: Layout, x, dst, sums, stream=None) -> None:
    """dst: bf16 [total_tokens, heads, d] contiguous copy of x; sums: fp32 [total_blocks, d] (written)."""
    lay, xt = L.c(), _tensor(x)
    if dst.dtype != torch.bfloat16 or not dst.is_contiguous() or dst.shape != x.shape:
        raise SwError(SW_ERR_INVALID_ARG, "dst must be a contiguous bf16 tensor of x's shape")
    _check(_lib.sw_copy_pool(C.byref(lay), C.byref(xt), _ptr(dst), _ptr(sums), _stream(stream)))


def sw_sketch_append(batch, block, max_blocks, x, seqlens, signs, cols, r, scale, mean, sketch, tok_sketch,
                     stream=None) -> None:
    xt = _tensor(x)
    _check(_lib.sw_sketch_append(batch, block, max_blocks, C.byref(xt), _ptr(seqlens), _ptr(signs), _ptr(cols),
                                 r, scale, _ptr(mean), _ptr(sketch), _ptr(tok_sketch), _stream(stream)))


def sw_block_scores(L: Layout, qs, ks, r, s, flags, W, A=None, stream=None) -> None:
    lay = L.c()
    _check(_lib.sw_block_scores(C.byref(lay), _ptr(qs), _ptr(ks), r, s, flags, _ptr(W), _ptr(A), _stream(stream)))


def sw_block_scores_row(batch, block, max_blocks, q_tok, ks, seqlens, r, s, flags, w_row, stream=None) -> None:
    _check(_lib.sw_block_scores_row(batch, block, max_blocks, _ptr(q_tok), _ptr(ks), _ptr(seqlens), r, s, flags,
                                    _ptr(w_row), _stream(stream)))


def sw_walk_update(L: Layout, R_prev, W, s, flags, R_out, ws=None, stream=None) -> None:
    lay = L.c()
    _check(_lib.sw_walk_update(C.byref(lay), _ptr(R_prev), _ptr(W), s, flags, _ptr(R_out), _ptr(ws),
                               0 if ws is None else ws.numel() * ws.element_size(), _stream(stream)))


def sw_walk_update_row(batch, block, max_blocks, r_prev, W_cache, stride_seq, w_row, seqlens, flags, r_out,
                       stream=None) -> None:
    _check(_lib.sw_walk_update_row(batch, block, max_blocks, _ptr(r_prev), _ptr(W_cache), stride_seq, _ptr(w_row),
                                   _ptr(seqlens), flags, _ptr(r_out), _stream(stream)))


def sw_select_topk(L: Layout, R, tau, tau_max, flags, idx, count, stream=None) -> None:
    lay = L.c()
    _check(_lib.sw_select_topk(C.byref(lay), _ptr(R), _ptr(tau), tau_max, flags, _ptr(idx), _ptr(count),
                               _stream(stream)))


def sw_prefill_select(L: Layout, qs, ks, r, s, flags, R_prev, R_out, W, A, tau, tau_max, idx, count, ws=None,
                      stream=None) -> None:
    lay = L.c()
    _check(_lib.sw_prefill_select(C.byref(lay), _ptr(qs), _ptr(ks), r, s, flags, _ptr(R_prev), _ptr(R_out), _ptr(W),
                                  _ptr(A), _ptr(tau), tau_max, _ptr(idx), _ptr(count), _ptr(ws),
                                  0 if ws is None else ws.numel() * ws.element_size(), _stream(stream)))


def sw_select_topk_row(batch, block, max_blocks, r, seqlens, tau, tau_max, flags, idx, count, stream=None) -> None:
    _check(_lib.sw_select_topk_row(batch, block, max_blocks, _ptr(r), _ptr(seqlens), _ptr(tau), tau_max, flags,
                                   _ptr(idx), _ptr(count), _stream(stream)))


def sw_decode_select(batch, block, max_blocks, q, k_new, seqlens, signs, cols, r, scale, s, flags, kbar, ks,
                     W_cache, stride_seq, r_prev, r_out, tau, tau_max, idx, count, ws, stream=None) -> None:
    """ws: uint8 tensor of sw_decode_select_workspace_bytes(batch, max_blocks) bytes."""
    qt, kt = _tensor(q), _tensor(k_new)
    _check(_lib.sw_decode_select(batch, block, max_blocks, C.byref(qt), C.byref(kt), _ptr(seqlens), _ptr(signs),
                                 _ptr(cols), r, scale, s, flags, _ptr(kbar), _ptr(ks), _ptr(W_cache), stride_seq,
                                 _ptr(r_prev), _ptr(r_out), _ptr(tau), tau_max, _ptr(idx), _ptr(count),
                                 _ptr(ws), 0 if ws is None else ws.numel() * ws.element_size(), _stream(stream)))


def sw_workspace_bytes(op, L: Optional[Layout], h_q=0, h_kv=0, d=0, tau_max=0, dtype=SW_BF16) -> int:
    lay = L.c() if L is not None else None
    return _lib.sw_workspace_bytes(op, C.byref(lay) if lay is not None else None, h_q, h_kv, d, tau_max, dtype)


def sw_decode_workspace_bytes(batch, h_q, h_kv, d, tau_max) -> int:
    return _lib.sw_decode_workspace_bytes(batch, h_q, h_kv, d, tau_max)


def sw_decode_select_workspace_bytes(batch, max_blocks) -> int:
    return _lib.sw_decode_select_workspace_bytes(batch, max_blocks)


def sw_decode_num_splits(batch, h_kv, d, tau_max) -> int:
    return _lib.sw_decode_num_splits(batch, h_kv, d, tau_max)


def sw_sparse_attn_prefill(L: Layout, q, k, v, idx, count, tau_max, softmax_scale, flags, out, lse=None,
                           ws=None, stream=None) -> None:
    lay, qt, kt, vt = L.c(), _tensor(q), _tensor(k), _tensor(v)
    _check(_lib.sw_sparse_attn_prefill(C.byref(lay), C.byref(qt), C.byref(kt), C.byref(vt), _ptr(idx), _ptr(count),
                                       tau_max, softmax_scale, flags, _ptr(out), _ptr(lse), _ptr(ws),
                                       0 if ws is None else ws.numel() * ws.element_size(), _stream(stream)))


def sw_sparse_attn_decode(batch, block, q, kcache, vcache, seqlens, idx, count, tau_max, softmax_scale, out,
                          lse=None, ws=None, stream=None) -> None:
    """q [batch, h_q, d]; kcache/vcache [batch, t_max, h_kv, d] (d contiguous)."""
    if kcache.dim() != 4 or vcache.dim() != 4 or kcache.stride(3) != 1 or vcache.stride(3) != 1:
        raise SwError(SW_ERR_INVALID_ARG, "caches must be [batch, t, h_kv, d] with contiguous d")
    if kcache.stride(0) != vcache.stride(0):
        raise SwError(SW_ERR_INVALID_ARG, "k and v caches must share the batch stride")
    qt = _tensor(q)
    kt = _Tensor(kcache.data_ptr(), _dtype_code(kcache), kcache.shape[2], kcache.shape[3], kcache.stride(1),
                 kcache.stride(2))
    vt = _Tensor(vcache.data_ptr(), _dtype_code(vcache), vcache.shape[2], vcache.shape[3], vcache.stride(1),
                 vcache.stride(2))
    _check(_lib.sw_sparse_attn_decode(batch, block, C.byref(qt), C.byref(kt), C.byref(vt), kcache.stride(0),
                                      _ptr(seqlens), _ptr(idx), _ptr(count), tau_max, softmax_scale, _ptr(out),
                                      _ptr(lse), _ptr(ws), 0 if ws is None else ws.numel() * ws.element_size(),
                                      _stream(stream)))


SW_STATIC_SCRATCH_BYTES = 4 << 20


def sw_sparse_attn_decode_static(batch, block, q, kcache, vcache, seqlens, idx, count, tau_max, softmax_scale, out,
                                 lse=None, stream=None) -> None:
    """sw_sparse_attn_decode without a workspace argument, for callers that cannot allocate device memory (a
    pre-partitioned serving pool, a plug-in without an allocator, a thread that must stay clear of cudaMalloc):
    the split-KV partials live in a fixed SW_STATIC_SCRATCH_BYTES array inside libsw.  Raises SwError
    (SW_ERR_WORKSPACE) when sw_decode_workspace_bytes(...) exceeds that size.  All calls on a device share the
    array, so calls that may overlap on the GPU (other streams / threads) race; the first call on each device
    does a one-time address lookup and belongs in start-up code, outside stream capture.  See include/sw.h."""
    if kcache.dim() != 4 or vcache.dim() != 4 or kcache.stride(3) != 1 or vcache.stride(3) != 1:
        raise SwError(SW_ERR_INVALID_ARG, "caches must be [batch, t, h_kv, d] with contiguous d")
    if kcache.stride(0) != vcache.stride(0):
        raise SwError(SW_ERR_INVALID_ARG, "k and v caches must share the batch stride")
    qt = _tensor(q)
    kt = _Tensor(kcache.data_ptr(), _dtype_code(kcache), kcache.shape[2], kcache.shape[3], kcache.stride(1),
                 kcache.stride(2))
    vt = _Tensor(vcache.data_ptr(), _dtype_code(vcache), vcache.shape[2], vcache.shape[3], vcache.stride(1),
                 vcache.stride(2))
    _check(_lib.sw_sparse_attn_decode_static(batch, block, C.byref(qt), C.byref(kt), C.byref(vt), kcache.stride(0),
                                             _ptr(seqlens), _ptr(idx), _ptr(count), tau_max, softmax_scale,
                                             _ptr(out), _ptr(lse), _stream(stream)))


def sw_sparse_attn_decode_paged(batch, block, q, kpool, vpool, block_table, seqlens, idx, count, tau_max,
                                softmax_scale, out, lse=None, ws=None, stream=None) -> None:
    """q [batch, h_q, d]; kpool/vpool [num_pages, block, h_kv, d] (or [num_pages*block, h_kv, d]) with contiguous
    pages; block_table [batch, max_blocks] int32: page of every logical block."""
    if kpool.dim() == 4:
        if kpool.shape[1] != block or not kpool.is_contiguous() or not vpool.is_contiguous():
            raise SwError(SW_ERR_INVALID_ARG, "pools must be contiguous [num_pages, block, h_kv, d]")
        kpool = kpool.view(-1, kpool.shape[2], kpool.shape[3]); vpool = vpool.view(-1, vpool.shape[2], vpool.shape[3])
    if block_table.dim() != 2 or block_table.stride(1) != 1 or block_table.dtype != torch.int32:
        raise SwError(SW_ERR_INVALID_ARG, "block_table must be int32 [batch, max_blocks] with unit stride")
    qt, kt, vt = _tensor(q), _tensor(kpool), _tensor(vpool)
    _check(_lib.sw_sparse_attn_decode_paged(batch, block, C.byref(qt), C.byref(kt), C.byref(vt),
                                            kpool.shape[0] // block, _ptr(block_table), block_table.stride(0),
                                            _ptr(seqlens), _ptr(idx), _ptr(count), tau_max, softmax_scale, _ptr(out),
                                            _ptr(lse), _ptr(ws), 0 if ws is None else ws.numel() * ws.element_size(),
                                            _stream(stream)))
