"""`-m gpu`: the race detector of this repo.  Every kernel writes each output element exactly once and uses no atomics on data,
so repeated launches on the same inputs must give the same BITS; a hand-over that is missing a fence or a barrier phase that
can alias shows up here as a flipped bit sooner than in a tolerance test.  (compute-sanitizer is not available on the pool.)"""
import pytest
import torch

from gpu_common import make_plan
from paper_2606_25473_b200 import binding as aj
from paper_2606_25473_b200 import build as aj_build
from paper_2606_25473_b200.workloads import Workload, make_inputs

pytestmark = pytest.mark.gpu

CASES = [
    Workload("stress_pair", 2, 4, 128, "teacher_forcing", 700, 4, 1, "bf16", 0.1, seed=1),             # CTA-pair forward + backward
    Workload("stress_pair_cleanzero", 2, 4, 128, "teacher_forcing", 700, 4, 1, "bf16", 0.1, 2, True),  # forward-only + general kernel
    Workload("stress_fwd_only", 2, 4, 128, "teacher_forcing", 700, 4, 1, "bf16", 0.0, 3, False, True), # forward-only kernel, setmaxnreg
    Workload("stress_d64", 2, 4, 64, "teacher_forcing", 700, 4, 1, "bf16", 0.1, seed=4),               # single-CTA kernels
    Workload("stress_block_causal", 2, 6, 128, "block_causal", 1000, 5, 1, "bf16", 0.1, seed=5),       # more tasks than SM pairs
]


@pytest.mark.parametrize("w", CASES, ids=lambda w: w.name)
def test_repeated_launches_are_bit_identical(w):
    assert torch.cuda.is_available()
    aj_build.build_library()
    x = [t.cuda() for t in make_inputs(w)]
    plan = make_plan(w)
    dout = torch.randn(x[0].shape, generator=torch.Generator().manual_seed(7)).to(x[0].dtype).cuda()
    ref = None
    for it in range(60):
        o, to = torch.full_like(x[0], float("nan")), torch.full_like(x[0], float("nan"))
        lse = torch.full((w.B, w.H, w.N), float("nan"), dtype=torch.float32, device="cuda")
        if w.no_tangents:
            aj.attn_fwd(plan, *x[:3], o, lse, 0)
            to.zero_()
        else:
            aj.attn_jvp_fwd(plan, *x, o, to, lse, 0)
        dq, dk, dv = [torch.full_like(x[0], float("nan")) for _ in range(3)]
        aj.attn_bwd(plan, x[0], x[1], x[2], o, lse, dout, dq, dk, dv, 0)
        cur = (o, to, lse, dq, dk, dv)
        if ref is None:
            ref = cur
        else:
            for name, a, b in zip(("o", "to", "lse", "dq", "dk", "dv"), ref, cur):
                assert torch.equal(a, b), f"{w.name}: {name} differs in launch {it}"
    torch.cuda.synchronize()
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_destroy(plan)
    for t in ref:
        assert torch.isfinite(t.float()).all()
