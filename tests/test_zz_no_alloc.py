"""attn_bwd_static: the backward for callers that cannot allocate GPU memory.

Some host programs cannot let this library call cudaMalloc: a process whose own pool reserved the card at start-up (the
call fails or eats memory the pool has promised elsewhere), or a step loop with a latency budget (an allocation can stall
every stream of the device).  attn_bwd_static serves them: no plan, no allocation, its one intermediate (delta per query
row) in a fixed array inside the library (AJ_STATIC_SCRATCH_MAX_ROWS rows, shared by every call on a device).

The GPU tests hold its dq, dk, dv against what the existing, plan-based attn_bwd returns for the same inputs, at the
tolerances of tests/test_gpu_backward.py, on calls made back to back -- a second call of another shape and other data, so
that anything stale in the shared scratch would show -- and they run the same whether this file is the whole session or
comes after every other test (the file is named to be collected last, so a failure here hides nothing).
The CPU tests cover the argument checks that come before any CUDA call, the size limit first of all.
"""
import ctypes

import numpy as np
import pytest
import torch

from helpers import max_norm_err
from paper_2606_25473_b200 import binding as aj
from paper_2606_25473_b200 import build as aj_build
from paper_2606_25473_b200.workloads import Workload, make_inputs

TOL = {"bf16": 1e-2, "fp32": 1e-4}      # max|err| / max|ref| per tensor, as in test_gpu_backward.py
KIND = {"teacher_forcing": aj.AJ_MASK_TEACHER_FORCING, "block_causal": aj.AJ_MASK_BLOCK_CAUSAL, "full": aj.AJ_MASK_FULL}


@pytest.fixture(scope="module", autouse=True)
def _built():
    aj_build.build_library()


# ---- CPU: rejected before anything touches a device ----------------------------------------------------------------------
def _raw_call(prob, mask):
    """The C call with no tensors at all: only good for argument errors that are found before the tensors are looked at."""
    null_t = ctypes.POINTER(aj.aj_tensor)()
    return aj.lib().attn_bwd_static(ctypes.byref(prob), ctypes.byref(mask), null_t, null_t, null_t, null_t, None,
                                    null_t, null_t, null_t, null_t, None)


def test_rows_beyond_the_fixed_scratch_are_rejected_with_both_numbers():
    nq = aj.AJ_STATIC_SCRATCH_MAX_ROWS // 8 + 1                 # 8 heads of it: one row too many
    prob = aj.make_problem(2, 4, nq, 64, 128, aj.AJ_BF16)
    mask, _ = aj.make_mask(aj.AJ_MASK_FULL)
    assert _raw_call(prob, mask) == aj.AJ_ERR_INVALID_ARG
    msg = aj.attn_jvp_last_error()
    assert str(8 * nq) in msg and str(aj.AJ_STATIC_SCRATCH_MAX_ROWS) in msg and "scratch" in msg


def test_the_largest_allowed_size_passes_the_size_check():
    prob = aj.make_problem(2, 4, aj.AJ_STATIC_SCRATCH_MAX_ROWS // 8, 64, 128, aj.AJ_BF16)
    mask, _ = aj.make_mask(aj.AJ_MASK_FULL)
    assert _raw_call(prob, mask) == aj.AJ_ERR_INVALID_ARG       # gets as far as the (null) tensors
    assert "q is NULL" in aj.attn_jvp_last_error()


def test_range_masks_and_bad_descriptors_are_refused():
    prob = aj.make_problem(1, 1, 64, 64, 64, aj.AJ_FP32)
    mask, keep = aj.make_mask(aj.AJ_MASK_RANGES, groups=[(0, 64, [(0, 64)])])
    assert _raw_call(prob, mask) == aj.AJ_ERR_UNSUPPORTED
    assert "attn_bwd" in aj.attn_jvp_last_error()
    mask, _ = aj.make_mask(aj.AJ_MASK_TEACHER_FORCING, 16, 3, 1)          # needs Nq = Nk = 96
    assert _raw_call(prob, mask) == aj.AJ_ERR_INVALID_ARG
    mask, _ = aj.make_mask(aj.AJ_MASK_BLOCK_CAUSAL, 16, 4, 3)             # 4 frames are not k chunks of 3
    assert _raw_call(prob, mask) == aj.AJ_ERR_INVALID_ARG
    prob = aj.make_problem(1, 1, 64, 64, 96, aj.AJ_FP32)
    mask, _ = aj.make_mask(aj.AJ_MASK_FULL)
    assert _raw_call(prob, mask) == aj.AJ_ERR_UNSUPPORTED                 # d


# ---- GPU: against the plan-based attn_bwd ----------------------------------------------------------------------------------
def _case(w: Workload, first_chunk_frames: int = 0, kernel=aj.AJ_KERNEL_AUTO, dout_seed: int = 7):
    """Inputs of `w` on the GPU, the library's forward (O, lse) on them, and attn_bwd's gradients (the existing path)."""
    dtype = aj.AJ_BF16 if w.dtype == "bf16" else aj.AJ_FP32
    prob = aj.make_problem(w.B, w.H, w.num_queries, w.N, w.d, dtype)
    mask, keep = aj.make_mask(KIND[w.mask], w.frame_len, w.num_frames, w.chunk_frames, first_chunk_frames)
    q, k, v, tq, tk, tv = [t.cuda() for t in make_inputs(w)]
    g = torch.Generator().manual_seed(dout_seed)
    dout = torch.randn(q.shape, generator=g).to(q.dtype).cuda()
    plan = aj.attn_jvp_plan_create(prob, mask)
    if kernel != aj.AJ_KERNEL_AUTO:
        aj.attn_jvp_plan_set_kernel(plan, kernel)
    o, to = torch.empty_like(q), torch.empty_like(q)
    lse = torch.empty((w.B, w.H, w.num_queries), dtype=torch.float32, device="cuda")
    aj.attn_jvp_fwd(plan, q, k, v, tq, tk, tv, o, to, lse, 0)
    ref = [torch.full_like(q, float("nan")), torch.full_like(k, float("nan")), torch.full_like(k, float("nan"))]
    aj.attn_bwd(plan, q, k, v, o, lse, dout, *ref, 0)
    torch.cuda.synchronize()
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_destroy(plan)
    return dict(w=w, prob=prob, mask=mask, keep=keep, q=q, k=k, v=v, o=o, lse=lse, dout=dout, ref=ref)


def _static(c, stream: int = 0):
    """One attn_bwd_static call into NaN-filled outputs (an unwritten element fails the comparison)."""
    out = [torch.full_like(c["q"], float("nan")), torch.full_like(c["k"], float("nan")), torch.full_like(c["k"], float("nan"))]
    aj.attn_bwd_static(c["prob"], c["mask"], c["q"], c["k"], c["v"], c["o"], c["lse"], c["dout"], *out, stream)
    return out


def _agree(c, got, tol=None):
    tol = tol or TOL[c["w"].dtype]
    for name, g, r in zip(("dq", "dk", "dv"), got, c["ref"]):
        g, r = g.double().cpu().numpy(), r.double().cpu().numpy()
        assert np.all(np.isfinite(g)), f"{c['w'].name}: non-finite or unwritten {name}"
        err = max_norm_err(g, r)
        assert err <= tol, f"{c['w'].name}: {name} differs from attn_bwd by {err:.3e} > {tol:.1e}"


@pytest.mark.gpu
def test_two_calls_in_a_row_match_attn_bwd_fp32():
    """Teacher forcing with ragged tiles (37-token frames, chunks of 2 after a first chunk of 1), then at once a smaller
    block-causal problem on other data: both against attn_bwd on the plain-FMA kernels, then the first again."""
    big = _case(Workload("static_tf_fp32", 2, 2, 64, "teacher_forcing", 37, 5, 2, "fp32", 1.0, seed=3), first_chunk_frames=1)
    small = _case(Workload("static_bc_fp32", 1, 3, 128, "block_causal", 45, 3, 1, "fp32", 1.0, seed=4), dout_seed=8)
    a = _static(big)
    b = _static(small)          # enqueued behind `a` on the same stream, shares the scratch
    a2 = _static(big)
    torch.cuda.synchronize()
    _agree(big, a)
    _agree(small, b)
    _agree(big, a2)
    for x, y in zip(a, a2):     # same inputs, same launch: the same bits whatever ran in between
        assert torch.equal(x, y)


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_tcgen05_backward_bf16():
    """bf16: the existing path is the CTA-pair tcgen05 backward (d = 128) and the single-CTA one (d = 64)."""
    c128 = _case(Workload("static_tf_bf16", 1, 2, 128, "teacher_forcing", 200, 3, 1, "bf16", 0.1, seed=5))
    c64 = _case(Workload("static_tfc_bf16_d64", 1, 2, 64, "teacher_forcing", 100, 4, 2, "bf16", 0.1, seed=6), dout_seed=9)
    a = _static(c128)
    b = _static(c64)
    torch.cuda.synchronize()
    _agree(c128, a)
    _agree(c64, b)


@pytest.mark.gpu
def test_full_mask_current_chunk_against_a_longer_key_prefix():
    """Nq != Nk under the full mask, on a side stream; the repeat of the call changes neither the result nor free memory."""
    c = _case(Workload("static_full_fp32", 1, 2, 64, "full", 50, 9, 1, "fp32", 1.0, seed=7, Nq=70), kernel=aj.AJ_KERNEL_SIMT)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        a = _static(c, s.cuda_stream)
        outs = [torch.full_like(t, float("nan")) for t in a]
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        aj.attn_bwd_static(c["prob"], c["mask"], c["q"], c["k"], c["v"], c["o"], c["lse"], c["dout"], *outs, s.cuda_stream)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before, "a steady-state call changed the device's free memory"
    _agree(c, a)
    for x, y in zip(a, outs):
        assert torch.equal(x, y)
