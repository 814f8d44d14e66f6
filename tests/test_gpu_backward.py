"""`-m gpu`: the primal backward (attn_bwd) against the fp64 oracle's plain VJP, element by element.

The forward that feeds it (O, lse) is the library's own forward on the same inputs.  Tolerances are the forward's
(BASELINE.json): bf16 path max|err|/max|ref| <= 1e-2, fp32 path <= 1e-4, per tensor.
"""
import numpy as np
import pytest
import torch

import oracle
from gpu_common import make_plan
from helpers import oracle_mask, widen, max_norm_err
from paper_2606_25473_b200 import binding as aj
from paper_2606_25473_b200 import build as aj_build
from paper_2606_25473_b200.workloads import WORKLOADS, Workload, make_inputs

pytestmark = pytest.mark.gpu
TOL = {"bf16": 1e-2, "fp32": 1e-4}


@pytest.fixture(scope="module", autouse=True)
def _ready():
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    aj_build.build_library()
    oracle.build()


def _dout(w: Workload, seed=99):
    g = torch.Generator().manual_seed(seed)
    return torch.randn((w.B, w.H, w.num_queries, w.d), generator=g).to(w.torch_dtype)


def run_fwd_bwd(w: Workload, x, dout, plan=None, kernel=aj.AJ_KERNEL_AUTO):
    """-> (dq, dk, dv) on the CPU; the gradients start as NaN so that an unwritten element fails the comparison.
    kernel = AJ_KERNEL_SIMT forces the plain-FMA forward and backward kernels on bf16 inputs."""
    own = plan is None
    if own:
        plan = make_plan(w, kernel)
    q, k, v, tq, tk, tv = [t.cuda() for t in x]
    o, to = torch.empty_like(q), torch.empty_like(q)
    lse = torch.empty((w.B, w.H, w.num_queries), dtype=torch.float32, device="cuda")
    aj.attn_jvp_fwd(plan, q, k, v, tq, tk, tv, o, to, lse, 0)
    dq = torch.full_like(q, float("nan"))
    dk, dv = torch.full_like(k, float("nan")), torch.full_like(k, float("nan"))
    aj.attn_bwd(plan, q, k, v, o, lse, dout.cuda(), dq, dk, dv, 0)
    torch.cuda.synchronize()
    assert aj.attn_jvp_plan_device_status(plan) == 0, "a backward kernel abandoned its launch (pipeline wait timed out)"
    if own:
        aj.attn_jvp_plan_destroy(plan)
    return dq.cpu(), dk.cpu(), dv.cpu()


def check(w, x, dout, got, heads=None, rows=None, keys=None):
    om = oracle_mask(w)
    errs = {"dq": [], "dk": [], "dv": []}
    refs = {"dq": [], "dk": [], "dv": []}
    for b in range(w.B):
        for h in range(w.H):
            if heads is not None and (b, h) not in heads:
                continue
            rq, rk, rv = oracle.attn_bwd_head(om, widen(x[0][b, h]), widen(x[1][b, h]), widen(x[2][b, h]), widen(dout[b, h]),
                                              1.0 / np.sqrt(w.d), rows, keys)
            rsel = slice(None) if rows is None else rows
            ksel = slice(None) if keys is None else keys
            for name, g, r, sel in (("dq", got[0], rq, rsel), ("dk", got[1], rk, ksel), ("dv", got[2], rv, ksel)):
                gg = g[b, h][sel].double().numpy()
                assert np.all(np.isfinite(gg)), f"{w.name}: non-finite or unwritten {name}"
                errs[name].append(gg)
                refs[name].append(r)
    out = {}
    for name in errs:
        out[name] = max_norm_err(np.concatenate(errs[name]), np.concatenate(refs[name]))
        assert out[name] <= TOL[w.dtype], f"{w.name}: {name} error {out[name]:.3e} (all: {out})"
    return out


SMALL = [
    Workload("bwd_tf_fp32", 1, 2, 64, "teacher_forcing", 16, 3, 1, "fp32", 1.0, seed=0),
    Workload("bwd_tf_chunk_fp32", 2, 2, 128, "teacher_forcing", 37, 4, 2, "fp32", 1.0, seed=1),
    Workload("bwd_bc_fp32", 1, 2, 128, "block_causal", 45, 3, 1, "fp32", 1.0, seed=2),
    Workload("bwd_full_fp32", 1, 2, 64, "full", 70, 2, 1, "fp32", 1.0, seed=3),
    Workload("bwd_tf_bf16", 1, 2, 128, "teacher_forcing", 200, 3, 1, "bf16", 0.1, seed=4),      # forward = CTA-pair tcgen05 kernel
    Workload("bwd_bc_bf16_B2", 2, 2, 128, "block_causal", 137, 4, 1, "bf16", 0.1, seed=5),
    Workload("bwd_tf_bf16_d64", 1, 2, 64, "teacher_forcing", 50, 3, 1, "bf16", 0.1, seed=6),
    # tcgen05 backward (bf16, d = 128): several 128-row stationary tiles and 64-row streamed tiles, ragged everywhere
    Workload("bwd_tf_chunk_bf16", 1, 2, 128, "teacher_forcing", 100, 6, 3, "bf16", 0.1, seed=7),
    Workload("bwd_full_bf16_N517", 1, 3, 128, "full", 517, 1, 1, "bf16", 0.1, seed=8),
    Workload("bwd_tf_bf16_L8", 1, 1, 128, "teacher_forcing", 8, 2, 1, "bf16", 0.1, seed=9),          # every tile partial
    Workload("bwd_tf_bf16_L64x5", 1, 1, 128, "teacher_forcing", 64, 5, 1, "bf16", 0.1, seed=10),     # exact streamed tiles
    Workload("bwd_tf_bf16_L1560_F2", 1, 1, 128, "teacher_forcing", 1560, 2, 1, "bf16", 0.1, seed=11),
    Workload("bwd_tf_bf16_unit", 1, 2, 128, "teacher_forcing", 300, 3, 1, "bf16", 1.0, seed=12),      # unit-variance dO-scale tangents irrelevant; peaked scores below
]


@pytest.mark.parametrize("w", SMALL, ids=lambda w: w.name)
def test_backward_small_every_element(w):
    x = make_inputs(w)
    dout = _dout(w)
    plan = make_plan(w)
    got = run_fwd_bwd(w, x, dout, plan)
    got2 = run_fwd_bwd(w, x, dout, plan)           # second call reuses the plan's backward schedules
    aj.attn_jvp_plan_destroy(plan)
    errs = check(w, x, dout, got)
    for a, b in zip(got, got2):
        assert torch.equal(a, b)
    if w.dtype == "fp32":
        assert max(errs.values()) < 2e-5


def test_backward_bf16_tcgen05_and_simt_paths_agree():
    w = SMALL[4]
    x = make_inputs(w)
    x[0] = (x[0].float() * 3.0).to(torch.bfloat16)          # peaked scores: p spans many orders of magnitude
    dout = _dout(w)
    a = run_fwd_bwd(w, x, dout)
    b = run_fwd_bwd(w, x, dout, kernel=aj.AJ_KERNEL_SIMT)
    check(w, x, dout, a)
    check(w, x, dout, b)
    for u, v in zip(a, b):
        assert max_norm_err(u.double().numpy(), v.double().numpy()) <= 1e-2


@pytest.mark.parametrize("dtype", ["fp32", "bf16"])
def test_backward_ranges_mask_unseen_keys_and_keyless_rows(dtype):
    Nq, Nk, d = 300, 421, 128
    groups = [(0, 130, [(3, 70), (70, 131), (200, 400)]), (150, 290, [(64, 65)]), (290, 300, [])]
    g = torch.Generator().manual_seed(9)
    tdt = torch.bfloat16 if dtype == "bf16" else torch.float32
    q, dout = [torch.randn((1, 2, Nq, d), generator=g).to(tdt) for _ in range(2)]
    k, v = [torch.randn((1, 2, Nk, d), generator=g).to(tdt) for _ in range(2)]
    prob = aj.make_problem(1, 2, Nq, Nk, d, aj.AJ_BF16 if dtype == "bf16" else aj.AJ_FP32)
    mask, keep = aj.make_mask(aj.AJ_MASK_RANGES, groups=groups)
    plan = aj.attn_jvp_plan_create(prob, mask)
    dev = [t.cuda() for t in (q, k, v)]
    zq, zk = torch.zeros_like(dev[0]), torch.zeros_like(dev[1])
    o, to = torch.empty_like(dev[0]), torch.empty_like(dev[0])
    lse = torch.empty((1, 2, Nq), dtype=torch.float32, device="cuda")
    aj.attn_jvp_fwd(plan, *dev, zq, zk, zk, o, to, lse, 0)
    dq = torch.full_like(dev[0], float("nan"))
    dk, dv = torch.full_like(dev[1], float("nan")), torch.full_like(dev[1], float("nan"))
    aj.attn_bwd(plan, *dev, o, lse, dout.cuda(), dq, dk, dv, 0)
    torch.cuda.synchronize()
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_destroy(plan)
    om = oracle.ranges_mask(groups)
    for h in range(2):
        rq, rk, rv = oracle.attn_bwd_head(om, widen(q[0, h]), widen(k[0, h]), widen(v[0, h]), widen(dout[0, h]), 1.0 / np.sqrt(d))
        assert max_norm_err(dq[0, h].cpu().double().numpy(), rq) <= TOL[dtype]
        assert max_norm_err(dk[0, h].cpu().double().numpy(), rk) <= TOL[dtype]
        assert max_norm_err(dv[0, h].cpu().double().numpy(), rv) <= TOL[dtype]
    unseen = np.r_[0:3, 131:200, 400:421]                    # keys no row sees: exact zeros, and written
    keyless = np.r_[130:150, 290:300]
    assert torch.count_nonzero(dk[0, :, unseen]) == 0 and torch.count_nonzero(dv[0, :, unseen]) == 0
    assert torch.count_nonzero(dq[0, :, keyless]) == 0


def test_forward_only_plan_feeds_the_backward():
    # the non-JVP stages: attn_fwd on an AJ_TANGENT_NONE plan, then attn_bwd on the same plan
    w = Workload("fwdbwd_bc", 1, 2, 128, "block_causal", 150, 4, 1, "bf16", 0.0, 21, False, True)
    x = make_inputs(w)
    dout = _dout(w)
    plan = make_plan(w)
    q, k, v = [t.cuda() for t in x[:3]]
    o = torch.empty_like(q)
    lse = torch.empty((w.B, w.H, w.N), dtype=torch.float32, device="cuda")
    aj.attn_fwd(plan, q, k, v, o, lse, 0)
    dq, dk, dv = torch.full_like(q, float("nan")), torch.full_like(q, float("nan")), torch.full_like(q, float("nan"))
    aj.attn_bwd(plan, q, k, v, o, lse, dout.cuda(), dq, dk, dv, 0)
    torch.cuda.synchronize()
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_destroy(plan)
    check(w, x, dout, (dq.cpu(), dk.cpu(), dv.cpu()))


def test_backward_strided_views_and_argument_errors():
    w = SMALL[4]
    x = make_inputs(w)
    dout = _dout(w)
    ref = run_fwd_bwd(w, x, dout)
    plan = make_plan(w)
    nd = lambda t: t.cuda().permute(0, 2, 1, 3).contiguous().permute(0, 2, 1, 3)       # [B, N, H, d] storage
    q, k, v, tq, tk, tv = [nd(t) for t in x]
    o, to = torch.empty_like(q), torch.empty_like(q)
    lse = torch.empty((w.B, w.H, w.N), dtype=torch.float32, device="cuda")
    aj.attn_jvp_fwd(plan, q, k, v, tq, tk, tv, o, to, lse, 0)
    dq, dk, dv = torch.empty_like(q), torch.empty_like(q), torch.empty_like(q)
    assert not dq.is_contiguous()
    aj.attn_bwd(plan, q, k, v, o, lse, nd(dout), dq, dk, dv, 0)
    torch.cuda.synchronize()
    for a, b in zip((dq, dk, dv), ref):
        assert torch.equal(a.cpu(), b)
    with pytest.raises(aj.AttnJvpError) as e:
        bad = torch.empty(q.numel() + 8, dtype=torch.bfloat16, device="cuda")[1:1 + q.numel()].view(q.shape)
        aj.attn_bwd(plan, bad, k, v, o, lse, nd(dout), dq, dk, dv, 0)
    assert e.value.status == aj.AJ_ERR_INVALID_ARG
    assert aj.lib().attn_bwd(plan, None, None, None, None, None, None, None, None, None, None) == aj.AJ_ERR_INVALID_ARG
    assert aj.lib().attn_bwd(None, None, None, None, None, None, None, None, None, None, None) == aj.AJ_ERR_INVALID_ARG
    aj.attn_jvp_plan_destroy(plan)


def test_backward_full_size_config2_one_head_sampled():
    """BASELINE.json configs[1] shape (H = 1 to keep the fp32 backward and the oracle to seconds): sampled query rows
    and keys of every block, against the oracle (whose pass over all rows supplies lse and delta)."""
    base = WORKLOADS["wan13b_tf_framewise"]
    w = Workload("wan13b_tf_framewise_H1", 1, 1, base.d, base.mask, base.frame_len, base.num_frames, base.chunk_frames,
                 base.dtype, base.tangent_std, base.seed)
    x = make_inputs(w)
    dout = _dout(w)
    got = run_fwd_bwd(w, x, dout)
    rng = np.random.default_rng(5)
    C, n = w.block_len, w.num_blocks
    idx = []
    for blk in range(2 * n):                                  # first, last and two random tokens of every block
        idx += [blk * C, (blk + 1) * C - 1] + list(rng.integers(blk * C, (blk + 1) * C, size=2))
    idx = np.unique(np.asarray(idx, dtype=np.int64))
    errs = check(w, x, dout, got, rows=idx, keys=idx)
    print(f"{w.name}: {len(idx)} rows/keys, errs={errs}")
    for t in got:
        assert torch.isfinite(t.float()).all()
    half = w.N // 2
    assert torch.count_nonzero(got[1][:, :, half + (n - 1) * C:]) > 0      # the last noisy block's keys are seen by itself
