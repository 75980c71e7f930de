"""sw_sparse_attn_decode_static: decode attention for callers that cannot allocate device memory.

Some users of libsw run where cudaMalloc is not an option: a serving process that handed its whole memory pool out
at start-up, a plug-in that gets tensors from its host framework but no allocator, a latency-critical thread that
must not hit a call that synchronises the device.  For them the library carries one entry point whose scratch (the
split-KV partials) is a fixed array inside libsw itself instead of a caller-supplied workspace.  This file checks it
against the ordinary sw_sparse_attn_decode on the same inputs, on two different problems back to back (the array is
shared by all calls and keeps the previous call's contents, so the second call runs on a dirty array), and checks
that a problem too big for the array is refused before anything is launched.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It makes no assumption about what ran before it in the process (it passes alone as well).
"""
import math

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

ATT_MAX, ATT_MEAN = 2e-2, 2e-3      # the attention tolerances of tests/test_gpu_parity.py


@pytest.fixture(scope="module")
def sw():
    import paper_2602_07397_b200 as pkg
    return pkg


def _problem(seed, ts, h_q, h_kv, d, B, tau):
    """Random q / caches and, per sequence, a valid ascending block list that always holds the last block."""
    rng = np.random.RandomState(seed)
    g = torch.Generator().manual_seed(seed)
    batch, tmax = len(ts), max(ts)
    q = torch.randn(batch, h_q, d, generator=g).bfloat16().cuda()
    kc = torch.randn(batch, tmax, h_kv, d, generator=g).bfloat16().cuda()
    vc = torch.randn(batch, tmax, h_kv, d, generator=g).bfloat16().cuda()
    idx = np.full((batch, tau), -1, np.int32)
    cnt = np.zeros(batch, np.int32)
    for s, t in enumerate(ts):
        bq = (t - 1) // B
        others = rng.permutation(bq)[:max(0, min(tau, bq + 1) - 1)]
        sel = np.sort(np.append(others, bq)).astype(np.int32)
        idx[s, :len(sel)] = sel
        cnt[s] = len(sel)
    seqlens = torch.tensor(ts, dtype=torch.int32).cuda()
    return batch, q, kc, vc, seqlens, torch.from_numpy(idx).cuda(), torch.from_numpy(cnt).cuda()


def test_static_scratch_decode_matches_workspace_decode_twice_in_a_row(sw):
    # two problems of different shape: the second one finds the first one's partials (laid out with another
    # split count and head count) still in the array
    problems = [
        dict(seed=11, ts=(64 * 9 + 1, 64 * 12, 700, 64), h_q=32, h_kv=8, d=128, B=64, tau=6),
        dict(seed=12, ts=(1000, 513, 128 * 5 + 64), h_q=16, h_kv=2, d=64, B=128, tau=4),
    ]
    for p in problems:
        batch, q, kc, vc, seqlens, idx, cnt = _problem(**p)
        h_q, h_kv, d, B, tau = p["h_q"], p["h_kv"], p["d"], p["B"], p["tau"]
        need = sw.sw_decode_workspace_bytes(batch, h_q, h_kv, d, tau)
        assert 0 < need <= sw.SW_STATIC_SCRATCH_BYTES
        scale = 1 / math.sqrt(d)
        # the existing path, with a caller-owned workspace
        ws = torch.empty(need, dtype=torch.uint8, device="cuda")
        out_ref = torch.full((batch, h_q, d), float("nan"), dtype=torch.bfloat16, device="cuda")
        lse_ref = torch.full((batch, h_q), float("nan"), device="cuda")
        sw.sw_sparse_attn_decode(batch, B, q, kc, vc, seqlens, idx, cnt, tau, scale, out_ref, lse_ref, ws)
        # the entry point under test: no workspace argument at all
        out = torch.full((batch, h_q, d), float("nan"), dtype=torch.bfloat16, device="cuda")
        lse = torch.full((batch, h_q), float("nan"), device="cuda")
        sw.sw_sparse_attn_decode_static(batch, B, q, kc, vc, seqlens, idx, cnt, tau, scale, out, lse)
        torch.cuda.synchronize()
        assert torch.isfinite(out.float()).all() and torch.isfinite(lse).all()
        err = (out.float() - out_ref.float()).abs()
        assert err.max().item() <= ATT_MAX and err.mean().item() <= ATT_MEAN, (err.max().item(), err.mean().item())
        assert (lse - lse_ref).abs().max().item() <= 1e-3
        # same kernels, same split count, same summation order: the header promises identical bits
        assert torch.equal(out, out_ref) and torch.equal(lse, lse_ref)


def test_static_scratch_decode_refuses_what_does_not_fit(sw):
    """A problem whose partials exceed the fixed array is an error with a readable message, not a silent overrun:
    nothing is launched and the output keeps its contents."""
    batch, h_q, h_kv, d, B, tau = 512, 32, 8, 128, 64, 64
    assert sw.sw_decode_workspace_bytes(batch, h_q, h_kv, d, tau) > sw.SW_STATIC_SCRATCH_BYTES
    q = torch.zeros(batch, h_q, d, dtype=torch.bfloat16, device="cuda")
    kc = torch.zeros(batch, B, h_kv, d, dtype=torch.bfloat16, device="cuda")
    vc = torch.zeros_like(kc)
    seqlens = torch.ones(batch, dtype=torch.int32, device="cuda")
    idx = torch.zeros(batch, tau, dtype=torch.int32, device="cuda")
    cnt = torch.ones(batch, dtype=torch.int32, device="cuda")
    out = torch.full((batch, h_q, d), 3.0, dtype=torch.bfloat16, device="cuda")
    launches = sw.sw_launch_count()
    with pytest.raises(sw.SwError) as e:
        sw.sw_sparse_attn_decode_static(batch, B, q, kc, vc, seqlens, idx, cnt, tau, 1 / math.sqrt(d), out)
    assert e.value.code == sw.SW_ERR_WORKSPACE and "SW_STATIC_SCRATCH_BYTES" in str(e.value)
    torch.cuda.synchronize()
    assert sw.sw_launch_count() == launches
    assert (out == 3.0).all()
