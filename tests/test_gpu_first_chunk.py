"""`-m gpu`: masks whose first block differs from the rest (`first_chunk_frames > 0`, "one initial latent frame
and then ..."; R6) through every kernel family, forward + JVP and primal backward, every row against the oracle.

The host scheduler's lowering of such descriptors is rasterised on the CPU (tests/test_schedule_host.py); here the lowered
schedules meet the kernels: CTA-pair and single-CTA tcgen05 (bf16, d = 128 and 64) and the plain-FMA kernels (fp32).
"""
import numpy as np
import pytest
import torch

import oracle
from helpers import max_norm_err
from paper_2606_25473_b200 import binding as aj
from paper_2606_25473_b200 import build as aj_build

pytestmark = pytest.mark.gpu

# (frame_len, num_frames, chunk_frames, first_chunk_frames): 1 + 2 + 2 frames and 3 + 1 + 1 frames of 100 tokens
SHAPES = [(100, 5, 2, 1), (100, 5, 1, 3)]
KERNELS = [("pair", aj.AJ_BF16, 128, aj.AJ_KERNEL_UMMA_PAIR), ("umma", aj.AJ_BF16, 128, aj.AJ_KERNEL_UMMA),
           ("umma_d64", aj.AJ_BF16, 64, aj.AJ_KERNEL_UMMA), ("simt", aj.AJ_FP32, 64, aj.AJ_KERNEL_SIMT)]


@pytest.fixture(scope="module", autouse=True)
def _ready():
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    aj_build.build_library()
    oracle.build()


@pytest.mark.parametrize("kname,dtype,d,kernel", KERNELS, ids=[k[0] for k in KERNELS])
@pytest.mark.parametrize("kind", ["teacher_forcing", "block_causal"])
@pytest.mark.parametrize("L,F,chunk,first", SHAPES, ids=["1+2+2", "3+1+1"])
def test_first_chunk_of_its_own_size(L, F, chunk, first, kind, kname, dtype, d, kernel):
    tf = kind == "teacher_forcing"
    N = F * L * (2 if tf else 1)
    B, H = 1, 2
    tdt = torch.bfloat16 if dtype == aj.AJ_BF16 else torch.float32
    g = torch.Generator().manual_seed(L + F + chunk + first + d)
    x = [torch.randn((B, H, N, d), generator=g).mul_(1.0 if i < 3 or dtype == aj.AJ_FP32 else 0.1).to(tdt) for i in range(6)]
    dout = torch.randn((B, H, N, d), generator=g).to(tdt)
    prob = aj.make_problem(B, H, N, N, d, dtype)
    mask, keep = aj.make_mask(aj.AJ_MASK_TEACHER_FORCING if tf else aj.AJ_MASK_BLOCK_CAUSAL, L, F, chunk, first)
    plan = aj.attn_jvp_plan_create(prob, mask)
    aj.attn_jvp_plan_set_kernel(plan, kernel)
    dev = [t.cuda() for t in x]
    o, to = torch.full_like(dev[0], float("nan")), torch.full_like(dev[0], float("nan"))
    lse = torch.full((B, H, N), float("nan"), dtype=torch.float32, device="cuda")
    aj.attn_jvp_fwd(plan, *dev, o, to, lse, 0)
    grads = [torch.full_like(dev[0], float("nan")) for _ in range(3)]
    aj.attn_bwd(plan, dev[0], dev[1], dev[2], o, lse, dout.cuda(), *grads, 0)
    torch.cuda.synchronize()
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_destroy(plan)

    num_blocks = 1 + (F - first) // chunk
    om = (oracle.teacher_forcing_mask if tf else oracle.block_causal_mask)(chunk * L, num_blocks, first * L)
    tol, tol_lse = (1e-2, 1e-3) if dtype == aj.AJ_BF16 else (1e-4, 1e-4)
    scale = 1.0 / np.sqrt(d)
    for h in range(H):
        a = [t[0, h].float().numpy() for t in x]
        ro, rto, rlse = oracle.attn_jvp_head(om, *a, scale)
        rq, rk, rv = oracle.attn_bwd_head(om, a[0], a[1], a[2], dout[0, h].float().numpy(), scale)
        for name, got, ref, t in (("o", o, ro, tol), ("to", to, rto, tol), ("lse", lse, rlse, tol_lse),
                                  ("dq", grads[0], rq, tol), ("dk", grads[1], rk, tol), ("dv", grads[2], rv, tol)):
            gg = got[0, h].double().cpu().numpy()
            assert np.all(np.isfinite(gg)), f"{name}: non-finite or unwritten"
            err = max_norm_err(gg, ref)
            assert err <= t, f"{kname} {kind} {L}x({first}+{chunk}..): {name} error {err:.3e} > {t:.1e}"
