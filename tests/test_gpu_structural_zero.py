"""`-m gpu`: structural-zero tangents and the tangent-free forward (N3) against the fp64 oracle.

N1 -- "The tangent of the clean context is zero": with AJ_TANGENT_CLEAN_ZERO the CTA-pair kernel skips the
contractions whose operand is zero.  The oracle is unchanged: it evaluates Eq. 42-44 on the same (zero-filled) data.
N3 -- AJ_TANGENT_NONE: O and lse only, also for Nq != Nk (current chunk x cached prefix).
"""
import numpy as np
import pytest
import torch

import oracle
from gpu_common import TOL, compare, make_plan, run_gpu, run_oracle, sample_rows
from helpers import widen, max_norm_err
from paper_2606_25473_b200 import binding as aj
from paper_2606_25473_b200 import build as aj_build
from paper_2606_25473_b200.workloads import EXTRA_WORKLOADS, Workload, make_inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _ready():
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    aj_build.build_library()
    oracle.build()


def _cz(name, B, H, mask, L, F, cf, seed, std=0.1):
    return Workload(name, B, H, 128, mask, L, F, cf, "bf16", std, seed, True)


CLEAN_ZERO = [
    _cz("cz_frame_L200", 1, 2, "teacher_forcing", 200, 3, 1, 0),      # clean/noisy boundary inside a 256-row tile
    _cz("cz_chunk_L100", 1, 2, "teacher_forcing", 100, 6, 3, 1),
    _cz("cz_L256x4_B2", 2, 1, "teacher_forcing", 256, 4, 1, 2),       # boundary on a tile edge: no straddling task
    _cz("cz_L8", 1, 1, "teacher_forcing", 8, 2, 1, 3),                # one task, all modes inside one pair-step
    _cz("cz_L64x5", 1, 1, "teacher_forcing", 64, 5, 1, 4),            # single-tile entries: mixed pair-steps
    _cz("cz_L1560_F2", 1, 1, "teacher_forcing", 1560, 2, 1, 5),       # the real frame length, long primal-only tasks
    _cz("cz_L700_F3_unit", 1, 2, "teacher_forcing", 700, 3, 1, 6, std=1.0),
]


@pytest.mark.parametrize("kernel", [aj.AJ_KERNEL_UMMA_PAIR, aj.AJ_KERNEL_UMMA_PAIR_ONE], ids=["split", "one"])
@pytest.mark.parametrize("w", CLEAN_ZERO, ids=lambda w: w.name)
def test_clean_zero_every_row(w, kernel):
    # "split" (default): the primal-only tasks run in the forward-only kernel (two softmax warpgroups), the rest in the general
    # CTA-pair kernel; "one": every task in the general kernel
    x = make_inputs(w)
    half = w.N // 2
    assert all(torch.count_nonzero(t[:, :, :half]) == 0 for t in x[3:]) and all(torch.count_nonzero(t[:, :, half:]) > 0 for t in x[3:])
    plan = make_plan(w, kernel)
    k_id, launches = aj.attn_jvp_plan_kernel(plan)
    assert k_id == kernel and launches == (1 if kernel == aj.AJ_KERNEL_UMMA_PAIR_ONE else 2 if w.N // 2 >= 256 else launches)
    classes = aj.attn_jvp_plan_pair_classes(plan)
    n, C = w.num_blocks, w.block_len
    assert classes == [n * (n + 1) // 2 * C * C, n * (n - 1) // 2 * C * C, n * C * C]
    gpu = run_gpu(w, x, plan=plan)
    gpu2 = run_gpu(w, x, plan=plan)
    aj.attn_jvp_plan_destroy(plan)
    compare(w, gpu, run_oracle(w, x))
    for a, b in zip(gpu, gpu2):
        assert torch.equal(a, b)
    assert torch.count_nonzero(gpu[1][:, :, :half]) == 0          # clean rows: tO = 0 exactly
    # the promise changes which contractions run, not the result: the dense plan on the same data agrees to rounding
    plan_d = make_plan(w, tangent_zero=aj.AJ_TANGENT_DENSE)
    dense = run_gpu(w, x, plan=plan_d)
    aj.attn_jvp_plan_destroy(plan_d)
    assert torch.equal(gpu[2][:, :, half:], dense[2][:, :, half:])   # S, P~ and l of the noisy rows are computed identically
    assert torch.equal(gpu[0][:, :, half:], dense[0][:, :, half:])
    assert max_norm_err(gpu[1].double().numpy(), dense[1].double().numpy()) <= 1e-2


def test_clean_zero_rescales_mid_stream():
    # growing key norms move the running max by more than the lazy threshold all along the stream, in primal-only tasks
    # (O alone is rescaled) and in key-zero pair-steps (O and T)
    w = _cz("cz_growing", 1, 2, "teacher_forcing", 550, 2, 1, 13, std=0.5)
    x = make_inputs(w)
    ramp = torch.linspace(0.2, 9.0, w.N // 2).repeat(2).view(1, 1, w.N, 1)
    x[1] = (x[1].float() * ramp).to(torch.bfloat16)
    x[0] = (x[0].float() * 3.0).to(torch.bfloat16)
    ref = run_oracle(w, x)
    compare(w, run_gpu(w, x), ref)
    compare(w, run_gpu(w, x, kernel=aj.AJ_KERNEL_UMMA_PAIR_ONE), ref)


def test_forward_only_kernel_rescales_across_the_two_warpgroups():
    # AJ_TANGENT_NONE, one long key stream per task (14 pair-steps and more): the reference max keeps moving by more than the
    # lazy threshold, so it is handed from one softmax warpgroup to the other again and again and both rescale their share of l
    Nq, Nk = 600, 1900
    g = torch.Generator().manual_seed(77)
    q = (torch.randn((1, 2, Nq, 128), generator=g) * 3.0).to(torch.bfloat16)
    k = (torch.randn((1, 2, Nk, 128), generator=g) * torch.linspace(0.2, 9.0, Nk).view(1, 1, Nk, 1)).to(torch.bfloat16)
    v = torch.randn((1, 2, Nk, 128), generator=g).to(torch.bfloat16)
    prob = aj.make_problem(1, 2, Nq, Nk, 128, aj.AJ_BF16)
    mask, keep = aj.make_mask(aj.AJ_MASK_FULL, tangent_zero=aj.AJ_TANGENT_NONE)
    outs = {}
    for kernel in (aj.AJ_KERNEL_UMMA_PAIR, aj.AJ_KERNEL_UMMA_PAIR_ONE):
        plan = aj.attn_jvp_plan_create(prob, mask)
        aj.attn_jvp_plan_set_kernel(plan, kernel)
        o = torch.full((1, 2, Nq, 128), float("nan"), dtype=torch.bfloat16, device="cuda")
        lse = torch.full((1, 2, Nq), float("nan"), dtype=torch.float32, device="cuda")
        aj.attn_fwd(plan, q.cuda(), k.cuda(), v.cuda(), o, lse, 0)
        torch.cuda.synchronize()
        assert aj.attn_jvp_plan_device_status(plan) == 0
        aj.attn_jvp_plan_destroy(plan)
        outs[kernel] = (o.cpu(), lse.cpu())
    zq, zk = np.zeros((Nq, 128), np.float32), np.zeros((Nk, 128), np.float32)
    for h in range(2):
        ro, _, rlse = oracle.attn_jvp_head(oracle.full_mask(), widen(q[0, h]), widen(k[0, h]), widen(v[0, h]), zq, zk, zk, 1.0 / np.sqrt(128))
        for o, lse in outs.values():
            assert max_norm_err(o[0, h].double().numpy(), ro) <= 1e-2
            assert max_norm_err(lse[0, h].double().numpy(), rlse) <= 1e-3


def test_ranges_mask_with_zero_flags_matches_oracle():
    # keys [0, 300) have zero tangents, rows [0, 260) have zero tQ; group 2 mixes flagged and unflagged ranges
    Nq, Nk, d = 600, 700, 128
    groups = [(0, 260, [(0, 130), (150, 300)]), (260, 400, [(0, 300)]), (400, 600, [(20, 300), (300, 450), (500, 700)])]
    qz, kz = [1, 0, 0], [1, 1, 1, 1, 0, 0]
    g = torch.Generator().manual_seed(21)
    q, tq = [torch.randn((1, 2, Nq, d), generator=g).to(torch.bfloat16) for _ in range(2)]
    k, v, tk, tv = [torch.randn((1, 2, Nk, d), generator=g).to(torch.bfloat16) for _ in range(4)]
    tq[:, :, :260] = 0
    tk[:, :, :300] = 0
    tv[:, :, :300] = 0
    prob = aj.make_problem(1, 2, Nq, Nk, d, aj.AJ_BF16)
    mask, keep = aj.make_mask(aj.AJ_MASK_RANGES, groups=groups, tangent_zero=aj.AJ_TANGENT_CLEAN_ZERO, q_tangent_zero=qz, k_tangent_zero=kz)
    plan = aj.attn_jvp_plan_create(prob, mask)
    o = torch.full((1, 2, Nq, d), float("nan"), dtype=torch.bfloat16, device="cuda")
    to = torch.full_like(o, float("nan"))
    lse = torch.full((1, 2, Nq), float("nan"), dtype=torch.float32, device="cuda")
    aj.attn_jvp_fwd(plan, q.cuda(), k.cuda(), v.cuda(), tq.cuda(), tk.cuda(), tv.cuda(), o, to, lse, 0)
    torch.cuda.synchronize()
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_destroy(plan)
    om = oracle.ranges_mask(groups)
    for h in range(2):
        ro, rto, rlse = oracle.attn_jvp_head(om, widen(q[0, h]), widen(k[0, h]), widen(v[0, h]), widen(tq[0, h]),
                                             widen(tk[0, h]), widen(tv[0, h]), 1.0 / np.sqrt(d))
        assert max_norm_err(o[0, h].cpu().double().numpy(), ro) <= 1e-2
        assert max_norm_err(to[0, h].cpu().double().numpy(), rto) <= 1e-2
        assert max_norm_err(lse[0, h].cpu().double().numpy(), rlse) <= 1e-3


# ---------------------------------------------------------------------------------------- N3: forward without tangents
def _fwd_only(Nq, Nk, kind, args, groups=None, B=1, H=2, seed=0, with_to=False):
    d = 128
    g = torch.Generator().manual_seed(seed)
    q = torch.randn((B, H, Nq, d), generator=g).to(torch.bfloat16)
    k, v = [torch.randn((B, H, Nk, d), generator=g).to(torch.bfloat16) for _ in range(2)]
    prob = aj.make_problem(B, H, Nq, Nk, d, aj.AJ_BF16)
    mask, keep = aj.make_mask(kind, *args, groups=groups, tangent_zero=aj.AJ_TANGENT_NONE)
    plan = aj.attn_jvp_plan_create(prob, mask)
    o = torch.full((B, H, Nq, d), float("nan"), dtype=torch.bfloat16, device="cuda")
    lse = torch.full((B, H, Nq), float("nan"), dtype=torch.float32, device="cuda")
    to = torch.full_like(o, float("nan")) if with_to else None
    if with_to:
        aj.attn_jvp_fwd(plan, q.cuda(), k.cuda(), v.cuda(), None, None, None, o, to, lse, 0)
    else:
        aj.attn_fwd(plan, q.cuda(), k.cuda(), v.cuda(), o, lse, 0)
    torch.cuda.synchronize()
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_destroy(plan)
    return q, k, v, o.cpu(), lse.cpu(), None if to is None else to.cpu()


@pytest.mark.parametrize("Nq,Nk", [(300, 300), (200, 1337), (1560, 4 * 1560), (77, 64)])
def test_forward_only_full_mask_current_chunk_against_cached_prefix(Nq, Nk):
    # the current chunk's queries against the committed prefix plus itself: one group, one range
    q, k, v, o, lse, _ = _fwd_only(Nq, Nk, aj.AJ_MASK_FULL, ())
    z = np.zeros((Nq, 128), np.float32), np.zeros((Nk, 128), np.float32)
    for h in range(2):
        ro, rto, rlse = oracle.attn_jvp_head(oracle.full_mask(), widen(q[0, h]), widen(k[0, h]), widen(v[0, h]), z[0], z[1], z[1],
                                             1.0 / np.sqrt(128))
        assert max_norm_err(o[0, h].double().numpy(), ro) <= 1e-2
        assert max_norm_err(lse[0, h].double().numpy(), rlse) <= 1e-3
        # independent library routine for the same thing
        ref = torch.nn.functional.scaled_dot_product_attention(q[0, h].double(), k[0, h].double(), v[0, h].double())
        assert max_norm_err(o[0, h].double().numpy(), ref.numpy()) <= 1e-2


def test_forward_only_block_causal_and_ranges_write_zero_tangent_output():
    Nq = Nk = 5 * 90
    q, k, v, o, lse, to = _fwd_only(Nq, Nk, aj.AJ_MASK_BLOCK_CAUSAL, (90, 5, 1), with_to=True)
    assert torch.count_nonzero(to) == 0                     # a non-NULL `to` is filled with zeros
    z = np.zeros((Nq, 128), np.float32)
    om = oracle.block_causal_mask(90, 5)
    for h in range(2):
        ro, _, rlse = oracle.attn_jvp_head(om, widen(q[0, h]), widen(k[0, h]), widen(v[0, h]), z, z, z, 1.0 / np.sqrt(128))
        assert max_norm_err(o[0, h].double().numpy(), ro) <= 1e-2
        assert max_norm_err(lse[0, h].double().numpy(), rlse) <= 1e-3
    groups = [(0, 100, [(0, 40), (64, 300)]), (130, 210, [(299, 300)])]     # uncovered rows 100..129
    q, k, v, o, lse, _ = _fwd_only(210, 300, aj.AJ_MASK_RANGES, (), groups=groups)
    zq, zk = np.zeros((210, 128), np.float32), np.zeros((300, 128), np.float32)
    rows = np.r_[0:100, 130:210]
    for h in range(2):
        ro, _, rlse = oracle.attn_jvp_head(oracle.ranges_mask(groups), widen(q[0, h]), widen(k[0, h]), widen(v[0, h]), zq, zk, zk,
                                           1.0 / np.sqrt(128), rows)
        assert max_norm_err(o[0, h, rows].double().numpy(), ro) <= 1e-2
        assert max_norm_err(lse[0, h, rows].double().numpy(), rlse) <= 1e-3
        assert torch.count_nonzero(o[0, h, 100:130]) == 0 and torch.all(torch.isneginf(lse[0, h, 100:130]))


def test_null_tangents_are_rejected_unless_the_plan_says_none():
    w = CLEAN_ZERO[3]
    x = [t.cuda() for t in make_inputs(w)]
    o = torch.empty_like(x[0])
    plan = make_plan(w)                                            # CLEAN_ZERO: tangents are still required
    with pytest.raises(aj.AttnJvpError) as e:
        aj.attn_jvp_fwd(plan, x[0], x[1], x[2], None, None, None, o, None, None, 0)
    assert e.value.status == aj.AJ_ERR_INVALID_ARG
    with pytest.raises(aj.AttnJvpError) as e:
        aj.attn_fwd(plan, x[0], x[1], x[2], o, None, 0)
    assert e.value.status == aj.AJ_ERR_INVALID_ARG
    aj.attn_jvp_plan_destroy(plan)
    torch.cuda.synchronize()


@pytest.mark.parametrize("dtype,d", [("fp32", 64), ("fp32", 128), ("bf16", 64), ("bf16", 128)])
def test_tangent_none_means_the_same_on_every_kernel(dtype, d):
    """AJ_TANGENT_NONE plans: tq, tk, tv are never read (NULL or garbage alike), a non-NULL `to` is zero-filled, O and lse
    are plain masked attention -- on the SIMT kernel (fp32), the single-CTA tcgen05 kernel (bf16 d = 64) and the CTA-pair
    kernel (bf16 d = 128) alike; then attn_bwd on the same plan (the non-JVP stages)."""
    w = Workload(f"none_{dtype}_{d}", 1, 2, d, "block_causal", 70, 3, 1, dtype, 0.0, 17, False, True)
    x = make_inputs(w)
    plan = make_plan(w)
    want = aj.AJ_KERNEL_SIMT if dtype == "fp32" else aj.AJ_KERNEL_UMMA_PAIR if d == 128 else aj.AJ_KERNEL_UMMA
    assert aj.attn_jvp_plan_kernel(plan)[0] == want
    q, k, v = [t.cuda() for t in x[:3]]
    junk = torch.full_like(q, float("nan"))
    o1, o2, to2 = torch.empty_like(q), torch.empty_like(q), torch.full_like(q, float("nan"))
    lse1, lse2 = [torch.empty((w.B, w.H, w.N), dtype=torch.float32, device="cuda") for _ in range(2)]
    tl = torch.full_like(lse1, float("nan"))
    aj.attn_fwd(plan, q, k, v, o1, lse1, 0)
    aj.attn_jvp_fwd(plan, q, k, v, junk, junk, junk, o2, to2, lse2, 0, tlse=tl)
    torch.cuda.synchronize()
    assert torch.equal(o1, o2) and torch.equal(lse1, lse2)
    assert torch.count_nonzero(to2) == 0 and torch.count_nonzero(tl) == 0
    om = oracle.block_causal_mask(w.block_len, w.num_blocks)
    z = np.zeros((w.N, d), np.float32)
    tol = 1e-2 if dtype == "bf16" else 1e-4
    g = torch.Generator().manual_seed(5)
    dout = torch.randn(q.shape, generator=g).to(q.dtype)
    dq, dk, dv = [torch.full_like(q, float("nan")) for _ in range(3)]
    aj.attn_bwd(plan, q, k, v, o1, lse1, dout.cuda(), dq, dk, dv, 0)
    torch.cuda.synchronize()
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_destroy(plan)
    for h in range(w.H):
        ro, _, rlse = oracle.attn_jvp_head(om, widen(x[0][0, h]), widen(x[1][0, h]), widen(x[2][0, h]), z, z, z, 1.0 / np.sqrt(d))
        assert max_norm_err(o1[0, h].cpu().double().numpy(), ro) <= tol
        assert max_norm_err(lse1[0, h].cpu().double().numpy(), rlse) <= (1e-3 if dtype == "bf16" else 1e-4)
        rq, rk, rv = oracle.attn_bwd_head(om, widen(x[0][0, h]), widen(x[1][0, h]), widen(x[2][0, h]), widen(dout[0, h]), 1.0 / np.sqrt(d))
        for got, ref in ((dq, rq), (dk, rk), (dv, rv)):
            assert max_norm_err(got[0, h].cpu().double().numpy(), ref) <= tol


# ---------------------------------------------------------------------------------------- full size (what bench.py times)
FORWARD_EXTRAS = [n for n, w in EXTRA_WORKLOADS.items() if not w.backward]


def test_backward_extras_are_covered_by_the_backward_tests():
    # a workload whose step is attn_bwd is compared through attn_bwd (tests/test_gpu_backward.py), never through the forward
    import test_gpu_backward
    assert {n for n, w in EXTRA_WORKLOADS.items() if w.backward} == set(test_gpu_backward.FULL_SIZE_BACKWARD)


@pytest.mark.parametrize("name", FORWARD_EXTRAS)
def test_extra_workloads_full_size_sampled_rows(name):
    """SURVEY.md 8(c) row protocol (every head, every query group) on the 8(f) forward workloads bench.py times."""
    w = EXTRA_WORKLOADS[name]
    x = make_inputs(w)
    plan = make_plan(w)
    gpu = run_gpu(w, x, plan=plan)
    aj.attn_jvp_plan_destroy(plan)
    rows = sample_rows(w)
    errs = compare(w, gpu, run_oracle(w, x, rows))
    nrows = sum(len(r) for r in rows.values())
    print(f"{name}: {nrows} rows = {100.0 * nrows / (w.B * w.H * w.num_queries):.2f} % of all rows, errs={errs}")
    if w.clean_tangent_zero:
        assert torch.count_nonzero(gpu[1][:, :, :w.N // 2]) == 0
    for t in gpu:
        assert torch.isfinite(t.float()).all()
