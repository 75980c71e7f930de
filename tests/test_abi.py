"""Host-side checks that need no GPU: libsw builds/loads, exports every symbol include/sw.h declares,
and validates arguments before touching the device."""
import ctypes as C
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pkg():
    from paper_2602_07397_b200 import build as b
    b.build()
    import paper_2602_07397_b200 as p
    return p


def header_symbols():
    text = open(os.path.join(ROOT, "include", "sw.h")).read()
    return sorted(set(re.findall(r"SW_API\s+[\w\s\*]+?\b(sw_\w+)\s*\(", text)))


def test_header_declares_the_six_calls():
    syms = header_symbols()
    for name in ["sw_sketch", "sw_block_scores", "sw_walk_update", "sw_select_topk", "sw_sparse_attn_prefill",
                 "sw_sparse_attn_decode"]:
        assert name in syms


def test_library_exports_every_declared_symbol(pkg):
    lib = C.CDLL(pkg.LIB_PATH)
    syms = header_symbols()
    assert len(syms) >= 15
    for name in syms:
        assert getattr(lib, name) is not None
    assert sorted(pkg.EXPORTS) == syms
    text = open(os.path.join(ROOT, "include", "sw.h")).read()
    assert pkg.sw_version() == pkg.SW_VERSION == int(re.search(r"#define SW_VERSION (\d+)", text).group(1))


def test_flag_values_match_header(pkg):
    text = open(os.path.join(ROOT, "include", "sw.h")).read()
    for name in ["SW_CAUSAL", "SW_SCORE_SOFTMAX", "SW_POW_MATRIX", "SW_FORCE_FIRST", "SW_FORCE_LAST", "SW_ROWNORM"]:
        val = int(re.search(name + r"\s*=\s*(\d+)", text).group(1))
        assert getattr(pkg, name) == val
    from oracle import sw_oracle as O        # the oracle restates the same contract values independently
    assert (O.CAUSAL, O.SCORE_SOFTMAX, O.POW_MATRIX, O.FORCE_FIRST, O.FORCE_LAST, O.ROWNORM) == (1, 2, 4, 8, 16, 32)


def test_validation_happens_before_any_device_work(pkg):
    lib = pkg.binding._lib
    # NULL layout -> INVALID_ARG regardless of the device
    assert lib.sw_sketch(None, None, None, None, 64, 0.125, None, None, None) == pkg.SW_ERR_INVALID_ARG
    assert b"layout" in lib.sw_last_error()
    lay = pkg.binding._Layout(1, 48, 10, 1, 1, 1, 1, 1)
    assert lib.sw_block_scores(C.byref(lay), 1, 1, 64, 2, 0, 1, None, None) == pkg.SW_ERR_UNSUPPORTED
    lay = pkg.binding._Layout(1, 64, 10, 1, 1, 16, 16, 16)
    assert lib.sw_block_scores(C.byref(lay), 16, 16, 64, 0, 0, 16, None, None) == pkg.SW_ERR_INVALID_ARG   # s = 0
    # sketches that are not 16-byte aligned are refused by both callers of the fused score kernel (cp.async / float4)
    assert lib.sw_block_scores(C.byref(lay), 16 + 4, 16, 64, 2, 0, 16, None, None) == pkg.SW_ERR_INVALID_ARG
    assert b"aligned" in lib.sw_last_error()
    assert lib.sw_prefill_select(C.byref(lay), 16, 16 + 8, 64, 2, 0, None, 16, 16, None, 16, 4, 16, 16, None, 0,
                                 None) == pkg.SW_ERR_INVALID_ARG
    assert b"aligned" in lib.sw_last_error()
    t = pkg.binding._Tensor(16, pkg.SW_BF16, 8, 96, 768, 96)
    assert lib.sw_sketch(C.byref(lay), C.byref(t), None, 16, 64, 0.125, 16, None, None) == pkg.SW_ERR_UNSUPPORTED
    t = pkg.binding._Tensor(16, pkg.SW_BF16, 8, 128, 1024, 128)
    assert lib.sw_sketch(C.byref(lay), C.byref(t), None, 16, 48, 0.125, 16, None, None) == pkg.SW_ERR_INVALID_ARG  # r
    t = pkg.binding._Tensor(8, pkg.SW_BF16, 8, 128, 1024, 128)     # misaligned pointer
    assert lib.sw_sketch(C.byref(lay), C.byref(t), None, 16, 64, 0.125, 16, None, None) == pkg.SW_ERR_INVALID_ARG


def test_decode_row_mode_rejects_non_causal(pkg):
    """Alg. 2 Step 4(ii) is not carried by the row-vector form: without SW_CAUSAL the three
    decode calls that depend on it return SW_ERR_UNSUPPORTED (before looking at the device)."""
    lib = pkg.binding._lib
    nc = pkg.SW_DEFAULT_FLAGS & ~pkg.SW_CAUSAL
    assert lib.sw_block_scores_row(1, 64, 4, 16, 16, 16, 64, 2, nc, 16, None) == pkg.SW_ERR_UNSUPPORTED
    assert b"SW_CAUSAL" in lib.sw_last_error()
    assert lib.sw_walk_update_row(1, 64, 4, 16, 32, 16, 16, 16, nc, 48, None) == pkg.SW_ERR_UNSUPPORTED
    t = pkg.binding._Tensor(16, pkg.SW_BF16, 8, 128, 1024, 128)
    assert lib.sw_decode_select(1, 64, 4, C.byref(t), C.byref(t), 16, None, 16, 64, 0.125, 2, nc, 16, 16, 16, 16, None,
                                16, 16, 2, 16, 16, 16, 4096, None) == pkg.SW_ERR_UNSUPPORTED


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback_without_gpu(pkg):
    """Valid arguments but no device: the call must fail loudly (SW_ERR_ARCH), never compute on the host."""
    lib = pkg.binding._lib
    lay = pkg.binding._Layout(1, 64, 10, 1, 1, 16, 16, 16)
    assert lib.sw_block_scores(C.byref(lay), 16, 16, 64, 2, 0, 16, None, None) == pkg.SW_ERR_ARCH
    with pytest.raises(pkg.SwError):
        pkg.binding._check(pkg.SW_ERR_ARCH)


def test_host_only_helpers(pkg):
    assert pkg.sw_decode_num_splits(8, 8, 128, 410) >= 1
    assert pkg.sw_decode_workspace_bytes(8, 32, 8, 128, 410) > 0
    assert not hasattr(pkg, "tau_from_density")      # the budget is the caller's: the package derives nothing from a density


def test_make_layout_offsets(pkg):
    L = pkg.make_layout([130, 64, 257], 64, device="cpu")
    assert L.blocks == [3, 1, 5] and L.total_blocks == 9 and L.max_blocks == 5 and L.total_tokens == 451
    assert L.cu_seqlens.tolist() == [0, 130, 194, 451] and L.cu_blocks.tolist() == [0, 3, 4, 9]
    assert L.cu_sq.tolist() == [0, 9, 10, 35] and L.total_sq == 35
