"""`-m gpu`: the CUDA path (through the C ABI) against the fp64 oracle, element by element.

Tolerances are BASELINE.json's: bf16 path max|err|/max|ref| <= 1e-2 on O and tO, <= 1e-3 on lse; fp32 path <= 1e-4.
Small cases compare every row of every head and span several query/key tiles with ragged tails; the
full-size configs (the launch configuration bench.py times) compare a deterministic row sample.
"""
import numpy as np
import pytest
import torch

import oracle
from gpu_common import TOL, compare, make_plan, run_gpu, run_oracle, sample_rows
from helpers import oracle_mask, widen, max_norm_err
from paper_2606_25473_b200 import binding as aj
from paper_2606_25473_b200 import build as aj_build
from paper_2606_25473_b200.workloads import WORKLOADS, Workload, make_inputs, scaled_down

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _ready():
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    aj_build.build_library()
    oracle.build()


# ---------------------------------------------------------------------------------------- config 1 (fp32 path)
def test_config1_tiny_tf_fp32_every_row():
    w = WORKLOADS["tiny_tf_fp32"]
    x = make_inputs(w)
    plan = make_plan(w)
    assert aj.attn_jvp_plan_kernel(plan) == (aj.AJ_KERNEL_SIMT, 1)
    assert aj.attn_jvp_plan_info(plan)[0] == 3072
    gpu = run_gpu(w, x, plan=plan)
    aj.attn_jvp_plan_destroy(plan)
    errs = compare(w, gpu, run_oracle(w, x))
    assert max(errs.values()) < 1e-5          # plain fp32 FMA lands ~3e-7 (R14)


@pytest.mark.parametrize("mask,L,F,cf,d", [
    ("teacher_forcing", 50, 3, 1, 64), ("teacher_forcing", 37, 4, 2, 128), ("block_causal", 45, 3, 1, 128),
    ("full", 70, 2, 1, 64)])
def test_simt_fp32_ragged(mask, L, F, cf, d):
    w = Workload(f"simt_{mask}", 2, 2, d, mask, L, F, cf, "fp32", 1.0, seed=3)
    x = make_inputs(w)
    compare(w, run_gpu(w, x), run_oracle(w, x))


def test_simt_runs_bf16_inputs():
    w = Workload("simt_bf16", 1, 2, 128, "teacher_forcing", 40, 3, 1, "bf16", 0.1, seed=5)
    x = make_inputs(w)
    compare(w, run_gpu(w, x, kernel=aj.AJ_KERNEL_SIMT), run_oracle(w, x))


# ---------------------------------------------------------------------------------------- tcgen05 path, small
SMALL_UMMA = [
    # several 128-row query tiles and 64-key tiles, every group and range with a ragged tail
    Workload("tf_frame_L200", 1, 2, 128, "teacher_forcing", 200, 3, 1, "bf16", 0.1, seed=0),
    Workload("tf_chunk_L100", 1, 2, 128, "teacher_forcing", 100, 6, 3, "bf16", 0.1, seed=1),
    Workload("bc_L137_B2", 2, 2, 128, "block_causal", 137, 4, 1, "bf16", 0.1, seed=2),
    Workload("full_N517", 1, 3, 128, "full", 517, 1, 1, "bf16", 0.1, seed=3),
    Workload("tf_L8", 1, 1, 128, "teacher_forcing", 8, 2, 1, "bf16", 0.1, seed=4),          # all tiles partial
    Workload("tf_L64x5", 1, 1, 128, "teacher_forcing", 64, 5, 1, "bf16", 0.1, seed=5),      # exact key tiles
    Workload("tf_L1560_F2", 1, 1, 128, "teacher_forcing", 1560, 2, 1, "bf16", 0.1, seed=6),  # the real frame length
]


UMMA_KERNELS = [aj.AJ_KERNEL_UMMA_PAIR, aj.AJ_KERNEL_UMMA]     # cta_group::2 pairs (the default) and the single-CTA kernel
KERNEL_IDS = {aj.AJ_KERNEL_UMMA_PAIR: "pair", aj.AJ_KERNEL_UMMA: "single"}


def test_default_kernel_for_bf16_d128_is_the_cta_pair_kernel():
    plan = make_plan(SMALL_UMMA[0])
    assert aj.attn_jvp_plan_kernel(plan) == (aj.AJ_KERNEL_UMMA_PAIR, 1)
    with pytest.raises(aj.AttnJvpError) as e:                      # 256-row pair tiles exist only on the packed grid
        aj.attn_jvp_plan_set_tiling(plan, aj.AJ_TILING_PER_GROUP)
    assert e.value.status == aj.AJ_ERR_UNSUPPORTED
    aj.attn_jvp_plan_destroy(plan)


@pytest.mark.parametrize("kernel", UMMA_KERNELS, ids=KERNEL_IDS.get)
@pytest.mark.parametrize("w", SMALL_UMMA, ids=lambda w: w.name)
def test_umma_small_every_row(w, kernel):
    x = make_inputs(w)
    plan = make_plan(w, kernel)
    assert aj.attn_jvp_plan_kernel(plan) == (kernel, 1)
    gpu = run_gpu(w, x, plan=plan)
    gpu2 = run_gpu(w, x, plan=plan)            # a second launch on the same plan must agree
    aj.attn_jvp_plan_destroy(plan)
    compare(w, gpu, run_oracle(w, x))
    for a, b in zip(gpu, gpu2):
        assert torch.equal(a, b)


@pytest.mark.parametrize("w", SMALL_UMMA[:4] + SMALL_UMMA[6:], ids=lambda w: w.name)
def test_umma_per_group_and_packed_tilings_agree(w):
    # PACKED (default: global 128-row grid, straddling tiles carry row intervals) vs PER_GROUP
    x = make_inputs(w)
    ref = run_oracle(w, x)
    plan = make_plan(w, aj.AJ_KERNEL_UMMA)
    packed = run_gpu(w, x, plan=plan)
    aj.attn_jvp_plan_set_tiling(plan, aj.AJ_TILING_PER_GROUP)
    per_group = run_gpu(w, x, plan=plan)
    aj.attn_jvp_plan_set_tiling(plan, aj.AJ_TILING_PACKED)
    packed2 = run_gpu(w, x, plan=plan)
    aj.attn_jvp_plan_destroy(plan)
    compare(w, packed, ref)
    compare(w, per_group, ref)
    for a, b in zip(packed, packed2):
        assert torch.equal(a, b)


@pytest.mark.parametrize("kernel", UMMA_KERNELS, ids=KERNEL_IDS.get)
def test_umma_large_unit_variance_tangents(kernel):
    # tangents as large as the primals, peaked scores (|s| up to ~4*sqrt(d)/sqrt(d)): exercises the lazy rescale
    w = Workload("tf_peaked", 1, 2, 128, "teacher_forcing", 300, 3, 1, "bf16", 1.0, seed=11)
    x = make_inputs(w)
    x[0] = (x[0].float() * 4.0).to(torch.bfloat16)
    compare(w, run_gpu(w, x, kernel=kernel), run_oracle(w, x))


@pytest.mark.parametrize("kernel", UMMA_KERNELS, ids=KERNEL_IDS.get)
def test_umma_growing_scores_force_rescales_late_in_the_stream(kernel):
    # key norms grow along the sequence, so the running max keeps moving by more than the lazy threshold (2^8) long
    # after the first tiles: the accumulator rescale must happen mid-stream, several times per row
    w = Workload("full_growing", 1, 2, 128, "full", 1100, 1, 1, "bf16", 0.5, seed=13)
    x = make_inputs(w)
    ramp = torch.linspace(0.2, 9.0, w.N).view(1, 1, w.N, 1)
    x[1] = (x[1].float() * ramp).to(torch.bfloat16)
    x[0] = (x[0].float() * 3.0).to(torch.bfloat16)
    compare(w, run_gpu(w, x, kernel=kernel), run_oracle(w, x))


# ---------------------------------------------------------------------------------------- tcgen05 path, bf16 with d = 64
SMALL_UMMA_D64 = [
    Workload("d64_tf_frame_L200", 1, 2, 64, "teacher_forcing", 200, 3, 1, "bf16", 0.1, seed=20),
    Workload("d64_tf_chunk_L100", 1, 2, 64, "teacher_forcing", 100, 6, 3, "bf16", 0.1, seed=21),
    Workload("d64_bc_L137_B2", 2, 2, 64, "block_causal", 137, 4, 1, "bf16", 0.1, seed=22),
    Workload("d64_full_N517", 1, 3, 64, "full", 517, 1, 1, "bf16", 0.1, seed=23),
    Workload("d64_tf_L8", 1, 1, 64, "teacher_forcing", 8, 2, 1, "bf16", 0.1, seed=24),          # all tiles partial
    Workload("d64_tf_L64x5", 1, 1, 64, "teacher_forcing", 64, 5, 1, "bf16", 0.1, seed=25),      # exact key tiles
    Workload("d64_tf_L1560_F2", 1, 1, 64, "teacher_forcing", 1560, 2, 1, "bf16", 0.1, seed=26),  # the real frame length
]


@pytest.mark.parametrize("w", SMALL_UMMA_D64, ids=lambda w: w.name)
def test_umma_d64_small_every_row(w):
    # bf16 with d = 64 runs the single-CTA tcgen05 kernel (one 64-column swizzle block per operand row) by default
    x = make_inputs(w)
    ref = run_oracle(w, x)
    plan = make_plan(w)
    assert aj.attn_jvp_plan_kernel(plan) == (aj.AJ_KERNEL_UMMA, 1)
    with pytest.raises(aj.AttnJvpError) as e:                      # the CTA-pair kernels take d = 128 only
        aj.attn_jvp_plan_set_kernel(plan, aj.AJ_KERNEL_UMMA_PAIR)
    assert e.value.status == aj.AJ_ERR_UNSUPPORTED
    packed = run_gpu(w, x, plan=plan)
    packed2 = run_gpu(w, x, plan=plan)
    aj.attn_jvp_plan_set_tiling(plan, aj.AJ_TILING_PER_GROUP)
    per_group = run_gpu(w, x, plan=plan)
    aj.attn_jvp_plan_set_kernel(plan, aj.AJ_KERNEL_SIMT)           # the plain-FMA kernel as an on-GPU cross-check
    simt = run_gpu(w, x, plan=plan)
    aj.attn_jvp_plan_destroy(plan)
    compare(w, packed, ref)
    compare(w, per_group, ref)
    compare(w, simt, ref)
    for a, b in zip(packed, packed2):
        assert torch.equal(a, b)


def test_umma_d64_peaked_and_growing_scores_rescale_mid_stream():
    w = Workload("d64_full_growing", 1, 2, 64, "full", 1100, 1, 1, "bf16", 0.5, seed=27)
    x = make_inputs(w)
    ramp = torch.linspace(0.2, 9.0, w.N).view(1, 1, w.N, 1)
    x[1] = (x[1].float() * ramp).to(torch.bfloat16)
    x[0] = (x[0].float() * 3.0).to(torch.bfloat16)
    compare(w, run_gpu(w, x), run_oracle(w, x))
    w = Workload("d64_tf_peaked", 1, 2, 64, "teacher_forcing", 300, 3, 1, "bf16", 1.0, seed=28)    # unit-variance tangents
    x = make_inputs(w)
    x[0] = (x[0].float() * 4.0).to(torch.bfloat16)
    compare(w, run_gpu(w, x), run_oracle(w, x))


@pytest.mark.parametrize("d", [64, 128])
def test_single_cta_kernel_tangent_free_mode(d):
    # AJ_TANGENT_NONE on the single-CTA tcgen05 kernel (the default for bf16 d = 64; forced for d = 128): S and P~ V only
    for w in (Workload(f"fwd_only_tf_d{d}", 1, 2, d, "teacher_forcing", 200, 3, 1, "bf16", 0.0, 30, False, True),
              Workload(f"fwd_only_prefix_d{d}", 2, 2, d, "full", 150, 4, 1, "bf16", 0.0, 31, False, True, 150)):   # Nq != Nk
        plan = make_plan(w, aj.AJ_KERNEL_UMMA)
        assert aj.attn_jvp_plan_kernel(plan) == (aj.AJ_KERNEL_UMMA, 1)
        x = make_inputs(w)
        got = run_gpu(w, x, plan=plan)
        aj.attn_jvp_plan_destroy(plan)
        compare(w, got, run_oracle(w, x))
        if d == 64:
            plan = make_plan(w)
            assert aj.attn_jvp_plan_kernel(plan)[0] == aj.AJ_KERNEL_UMMA
            aj.attn_jvp_plan_destroy(plan)


@pytest.mark.parametrize("kernel", UMMA_KERNELS, ids=KERNEL_IDS.get)
def test_one_plan_on_two_streams_at_once(kernel):
    # the forward keeps no per-call device state in the plan (task lists are read-only): two launches of the same plan in flight
    # on two streams, on different inputs, give the bits of the same launches run one after the other
    w = Workload("two_streams", 1, 4, 128, "teacher_forcing", 700, 3, 1, "bf16", 0.1, seed=41)
    w2 = Workload("two_streams_b", 1, 4, 128, "teacher_forcing", 700, 3, 1, "bf16", 0.1, seed=42)
    xa, xb = [t.cuda() for t in make_inputs(w)], [t.cuda() for t in make_inputs(w2)]
    plan = make_plan(w, kernel)
    outs = []
    for x in (xa, xb):                                   # sequential reference
        o, to = torch.empty_like(x[0]), torch.empty_like(x[0])
        lse = torch.empty((w.B, w.H, w.N), dtype=torch.float32, device="cuda")
        aj.attn_jvp_fwd(plan, *x, o, to, lse, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        outs.append((o, to, lse))
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    conc = []
    for x, st in ((xa, s1), (xb, s2)):
        o, to = torch.full_like(x[0], float("nan")), torch.full_like(x[0], float("nan"))
        lse = torch.full((w.B, w.H, w.N), float("nan"), dtype=torch.float32, device="cuda")
        conc.append((o, to, lse))
    torch.cuda.synchronize()
    for rep in range(3):
        for (x, st), out in zip(((xa, s1), (xb, s2)), conc):
            aj.attn_jvp_fwd(plan, *x, *out, st.cuda_stream)
    torch.cuda.synchronize()
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_destroy(plan)
    for ref, got in zip(outs, conc):
        for a, b in zip(ref, got):
            assert torch.equal(a, b)


@pytest.mark.parametrize("mode", ["per_head", "per_slot"])
def test_rendezvous_forced_on_a_small_problem(mode):
    # Long-sequence launches make the SM pairs meet -- before every head when their tasks differ in cost (configs[4] turns that
    # on by itself), at every task slot when they cost the same (its full-mask control).  attn_jvp_plan_set_rendezvous forces
    # either mode on a problem the oracle finishes in seconds: more tasks than pairs, eight heads, same results as without it.
    w = Workload("head_sync", 2, 4, 128, "block_causal", 1000, 5, 1, "bf16", 0.1, seed=51)
    x = make_inputs(w)
    plan = make_plan(w)
    assert aj.attn_jvp_plan_rendezvous(plan) == aj.AJ_RENDEZVOUS_OFF          # AUTO leaves it off on short key streams
    plain = run_gpu(w, x, plan=plan)
    want = aj.AJ_RENDEZVOUS_PER_HEAD if mode == "per_head" else aj.AJ_RENDEZVOUS_PER_SLOT
    aj.attn_jvp_plan_set_rendezvous(plan, want)
    assert aj.attn_jvp_plan_rendezvous(plan) == want
    synced = run_gpu(w, x, plan=plan)
    synced2 = run_gpu(w, x, plan=plan)
    # two launches of the plan in flight at once share the counters: allowed to be slow, not to be wrong (attn_jvp.h)
    dev = [t.cuda() for t in x]
    streams = [torch.cuda.Stream() for _ in range(2)]
    conc = [[torch.full_like(dev[0], float("nan")), torch.full_like(dev[0], float("nan")),
             torch.full((w.B, w.H, w.N), float("nan"), dtype=torch.float32, device="cuda")] for _ in streams]
    torch.cuda.synchronize()
    for st, out in zip(streams, conc):
        aj.attn_jvp_fwd(plan, *dev, *out, st.cuda_stream)
    torch.cuda.synchronize()
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_set_rendezvous(plan, aj.AJ_RENDEZVOUS_OFF)
    assert aj.attn_jvp_plan_rendezvous(plan) == aj.AJ_RENDEZVOUS_OFF
    off = run_gpu(w, x, plan=plan)
    aj.attn_jvp_plan_destroy(plan)
    rows = {(0, 0): np.arange(0, w.N, 7), (1, 3): np.arange(3, w.N, 11)}
    compare(w, synced, run_oracle(w, x, rows))
    for other in (synced2, plain, off, [t.cpu() for t in conc[0]], [t.cpu() for t in conc[1]]):
        for a, b in zip(synced, other):                   # the lists may differ (levelled at every head), the arithmetic per task does not
            assert torch.equal(a, b)


def test_worker_budget_leaves_sm_pairs_free_and_keeps_the_bits():
    # attn_jvp_plan_set_workers: task lists for fewer SM pairs (room for a collective's kernels beside the persistent grid).
    # Forward + JVP (general and forward-only kernel of a clean-zero plan) and the backward: same bits under every budget.
    w = Workload("budget", 1, 4, 128, "teacher_forcing", 700, 4, 1, "bf16", 0.1, seed=61, clean_tangent_zero=True)
    x = make_inputs(w)
    g = torch.Generator().manual_seed(62)
    dout = torch.randn(x[0].shape, generator=g).to(torch.bfloat16).cuda()
    plan = make_plan(w)
    full_pairs = aj.attn_jvp_plan_workers(plan)
    assert full_pairs[0] > 8 and full_pairs[1] > 8

    def run():
        o, to, lse = [t.cuda() for t in run_gpu(w, x, plan=plan)]
        dev = [t.cuda() for t in x]
        grads = [torch.full_like(dev[0], float("nan")) for _ in range(3)]
        aj.attn_bwd(plan, dev[0], dev[1], dev[2], o, lse, dout, *grads, 0)
        torch.cuda.synchronize()
        assert aj.attn_jvp_plan_device_status(plan) == 0
        return [o, to, lse] + grads

    ref = run()
    for budget in (8, 1, 66):
        aj.attn_jvp_plan_set_workers(plan, budget)
        pairs = aj.attn_jvp_plan_workers(plan)
        assert pairs[0] == min(budget, full_pairs[0]) and pairs[1] == min(budget, full_pairs[1])
        for a, b in zip(run(), ref):
            assert torch.equal(a, b)
    aj.attn_jvp_plan_set_workers(plan, 0)
    assert aj.attn_jvp_plan_workers(plan) == full_pairs
    aj.attn_jvp_plan_destroy(plan)
    rows = {(0, h): np.arange(h, w.N, 13) for h in range(w.H)}
    compare(w, [t.cpu() for t in ref[:3]], run_oracle(w, x, rows))


def test_umma_zero_tangents_give_exact_zero():
    w = SMALL_UMMA[0]
    x = make_inputs(w)
    for i in (3, 4, 5):
        x[i].zero_()
    o, to, lse = run_gpu(w, x)
    assert torch.count_nonzero(to) == 0
    ref = run_oracle(w, x)
    compare(w, (o, to, lse), ref, tol=dict(o=1e-2, to=1e-2, lse=1e-3))


def test_umma_masked_keys_have_no_effect():
    w = SMALL_UMMA[0]                       # TF: the first noisy block sees only itself
    x = make_inputs(w)
    base = run_gpu(w, x)
    half, C = w.N // 2, w.block_len
    y = [t.clone() for t in x]
    for i in (1, 2, 4, 5):                  # K, V, tK, tV of every key the first noisy block may not see
        y[i][:, :, :half] = 7.0
        y[i][:, :, half + C:] = -3.0
    pert = run_gpu(w, y)
    rows = slice(half, half + C)
    for a, b in zip(base, pert):
        assert torch.equal(a[:, :, rows], b[:, :, rows])


def test_umma_strided_views():
    # [B, N, H, d] storage viewed as [B, H, N, d] (what a projection layer produces), outputs likewise
    w = SMALL_UMMA[0]
    x = make_inputs(w)
    dev = [t.cuda().permute(0, 2, 1, 3).contiguous().permute(0, 2, 1, 3) for t in x]
    assert not dev[0].is_contiguous()
    o = torch.full((w.B, w.N, w.H, w.d), float("nan"), dtype=torch.bfloat16, device="cuda").permute(0, 2, 1, 3)
    to = torch.full_like(o, float("nan"))
    lse = torch.empty((w.B, w.H, w.N), dtype=torch.float32, device="cuda")
    plan = make_plan(w)
    aj.attn_jvp_fwd(plan, *dev, o, to, lse, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    aj.attn_jvp_plan_destroy(plan)
    ref = run_gpu(w, x)
    assert torch.equal(o.cpu(), ref[0]) and torch.equal(to.cpu(), ref[1]) and torch.equal(lse.cpu(), ref[2])


@pytest.mark.parametrize("kernel", UMMA_KERNELS, ids=KERNEL_IDS.get)
def test_umma_matches_simt_kernel_on_bf16(kernel):
    w = SMALL_UMMA[1]
    x = make_inputs(w)
    a = run_gpu(w, x, kernel=kernel)
    b = run_gpu(w, x, kernel=aj.AJ_KERNEL_SIMT)
    for u, v, tol in zip(a, b, (1e-2, 1e-2, 1e-3)):
        assert max_norm_err(u.double().numpy(), v.double().numpy()) <= tol


# ---------------------------------------------------------------------------------------- generic ranges, edge cases
@pytest.mark.parametrize("dtype,d", [("fp32", 64), ("bf16", 128)])
def test_ranges_mask_uncovered_rows_and_nq_ne_nk(dtype, d):
    Nq, Nk = 300, 421
    groups = [(0, 130, [(3, 70), (70, 131), (200, 421)]), (150, 290, [(64, 65)]), (290, 300, [])]
    tdt = torch.bfloat16 if dtype == "bf16" else torch.float32
    g = torch.Generator().manual_seed(9)
    q, tq = [torch.randn((1, 2, Nq, d), generator=g).to(tdt) for _ in range(2)]
    k, v, tk, tv = [torch.randn((1, 2, Nk, d), generator=g).to(tdt) for _ in range(4)]
    prob = aj.make_problem(1, 2, Nq, Nk, d, aj.AJ_BF16 if dtype == "bf16" else aj.AJ_FP32)
    mask, keep = aj.make_mask(aj.AJ_MASK_RANGES, groups=groups)
    plan = aj.attn_jvp_plan_create(prob, mask)
    o = torch.full((1, 2, Nq, d), float("nan"), dtype=tdt, device="cuda")
    to = torch.full_like(o, float("nan"))
    lse = torch.full((1, 2, Nq), float("nan"), dtype=torch.float32, device="cuda")
    aj.attn_jvp_fwd(plan, q.cuda(), k.cuda(), v.cuda(), tq.cuda(), tk.cuda(), tv.cuda(), o, to, lse, 0)
    torch.cuda.synchronize()
    aj.attn_jvp_plan_destroy(plan)
    o, to, lse = o.cpu(), to.cpu(), lse.cpu()
    om = oracle.ranges_mask(groups)
    covered = np.r_[0:130, 150:290]
    empty = np.r_[130:150, 290:300]
    tol = TOL[dtype]
    for h in range(2):
        ro, rto, rlse = oracle.attn_jvp_head(om, widen(q[0, h]), widen(k[0, h]), widen(v[0, h]), widen(tq[0, h]),
                                             widen(tk[0, h]), widen(tv[0, h]), 1.0 / np.sqrt(d), covered)
        assert max_norm_err(o[0, h, covered].double().numpy(), ro) <= tol["o"]
        assert max_norm_err(to[0, h, covered].double().numpy(), rto) <= tol["to"]
        assert max_norm_err(lse[0, h, covered].double().numpy(), rlse) <= tol["lse"]
        # rows in no group or with no key: O = 0, tO = 0, lse = -inf (R9)
        assert torch.count_nonzero(o[0, h, empty]) == 0 and torch.count_nonzero(to[0, h, empty]) == 0
        assert torch.all(torch.isneginf(lse[0, h, empty]))


def test_lse_may_be_null_and_custom_scale():
    w = SMALL_UMMA[4]
    x = make_inputs(w)
    plan = make_plan(w, scale=0.05)
    dev = [t.cuda() for t in x]
    o, to = torch.empty_like(dev[0]), torch.empty_like(dev[0])
    aj.attn_jvp_fwd(plan, *dev, o, to, None, 0)
    torch.cuda.synchronize()
    aj.attn_jvp_plan_destroy(plan)
    om = oracle.teacher_forcing_mask(w.block_len, w.num_blocks)
    ro, rto, _ = oracle.attn_jvp_head(om, *[widen(t[0, 0]) for t in x], 0.05)
    assert max_norm_err(o.cpu()[0, 0].double().numpy(), ro) <= 1e-2
    assert max_norm_err(to.cpu()[0, 0].double().numpy(), rto) <= 1e-2


@pytest.mark.parametrize("w", [SMALL_UMMA[0], SMALL_UMMA[2], WORKLOADS["tiny_tf_fp32"]], ids=lambda w: w.name)
def test_fwd_host_matches_device_path(w):
    # attn_jvp_fwd_host launches head by head (copies of the neighbouring heads in flight): same bits as one launch
    x = make_inputs(w, pin=True)
    plan = make_plan(w)
    o = torch.full_like(x[0], float("nan")).pin_memory()
    to = torch.full_like(x[0], float("nan")).pin_memory()
    lse = torch.full((w.B, w.H, w.N), float("nan"), dtype=torch.float32).pin_memory()
    ref = run_gpu(w, x, plan=plan)
    for _ in range(2):                                  # the second call reuses the staging buffers and events
        aj.attn_jvp_fwd_host(plan, *x, o, to, lse, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert torch.equal(o, ref[0]) and torch.equal(to, ref[1]) and torch.equal(lse, ref[2])
        o.fill_(float("nan")); to.fill_(float("nan")); lse.fill_(float("nan"))
    aj.attn_jvp_fwd_host(plan, *x, o, to, None, 0)      # default stream, no lse
    torch.cuda.synchronize()
    assert torch.equal(o, ref[0]) and torch.equal(to, ref[1]) and torch.isnan(lse).all()
    if w.dtype == "bf16":                               # switching the kernel rebuilds the per-head schedule too
        aj.attn_jvp_plan_set_kernel(plan, aj.AJ_KERNEL_UMMA)
        ref1 = run_gpu(w, x, plan=plan)
        aj.attn_jvp_fwd_host(plan, *x, o, to, lse, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert torch.equal(o, ref1[0]) and torch.equal(to, ref1[1]) and torch.equal(lse, ref1[2])
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_destroy(plan)


def test_broadcast_heads_zero_stride():
    """A K/V shared by all heads (`expand` over H: stride_h = 0).  The SIMT kernels honour it; the tcgen05 kernels cannot
    express it in a TMA tensor map and say so (AJ_ERR_UNSUPPORTED) instead of reading heads 16 bytes apart; an output with
    aliased heads is always an error."""
    w = Workload("bcast", 1, 3, 128, "block_causal", 80, 3, 1, "bf16", 0.1, seed=8)
    x = make_inputs(w)
    for i in (1, 2, 4, 5):
        x[i] = x[i][:, :1].expand(-1, w.H, -1, -1)             # every head sees head 0's K, V, tK, tV
    dev = [t.cuda() for t in x]
    dev = [dev[0], dev[1][:, :1].expand(-1, w.H, -1, -1), dev[2][:, :1].expand(-1, w.H, -1, -1), dev[3],
           dev[4][:, :1].expand(-1, w.H, -1, -1), dev[5][:, :1].expand(-1, w.H, -1, -1)]
    assert dev[1].stride(1) == 0
    o, to = torch.full_like(dev[0], float("nan")), torch.full_like(dev[0], float("nan"))
    lse = torch.empty((w.B, w.H, w.N), dtype=torch.float32, device="cuda")
    plan = make_plan(w)
    with pytest.raises(aj.AttnJvpError) as e:
        aj.attn_jvp_fwd(plan, *dev, o, to, lse, 0)
    assert e.value.status == aj.AJ_ERR_UNSUPPORTED
    aj.attn_jvp_plan_set_kernel(plan, aj.AJ_KERNEL_SIMT)
    aj.attn_jvp_fwd(plan, *dev, o, to, lse, 0)
    torch.cuda.synchronize()
    compare(w, (o.cpu(), to.cpu(), lse.cpu()), run_oracle(w, [t.contiguous() for t in x]))
    with pytest.raises(aj.AttnJvpError) as e:                      # aliased output heads
        aj.attn_jvp_fwd(plan, *dev, o[:, :1].expand(-1, w.H, -1, -1), to, lse, 0)
    assert e.value.status == aj.AJ_ERR_INVALID_ARG
    aj.attn_jvp_plan_destroy(plan)


def test_binding_rejects_tensors_that_do_not_match_the_plan():
    w = SMALL_UMMA[4]
    plan = make_plan(w)
    dev = [t.cuda() for t in make_inputs(w)]
    o, to = torch.empty_like(dev[0]), torch.empty_like(dev[0])
    lse = torch.empty((w.B, w.H, w.N), dtype=torch.float32, device="cuda")
    with pytest.raises(ValueError):                                # wrong N
        aj.attn_jvp_fwd(plan, dev[0][:, :, :-8], *dev[1:], o, to, lse, 0)
    with pytest.raises(ValueError):                                # wrong dtype
        aj.attn_jvp_fwd(plan, dev[0].float(), *dev[1:], o, to, lse, 0)
    with pytest.raises(ValueError):                                # host tensor on the device call
        aj.attn_jvp_fwd(plan, dev[0].cpu(), *dev[1:], o, to, lse, 0)
    with pytest.raises(ValueError):                                # lse of the wrong dtype
        aj.attn_jvp_fwd(plan, *dev, o, to, lse.double(), 0)
    with pytest.raises(ValueError):                                # lse too short
        aj.attn_jvp_fwd(plan, *dev, o, to, lse[:, :, :-1].contiguous(), 0)
    aj.attn_jvp_fwd(plan, *dev, o, to, lse, 0)
    torch.cuda.synchronize()
    aj.attn_jvp_plan_destroy(plan)


def test_tensor_maps_are_cached_by_the_plan():
    w = SMALL_UMMA[0]
    plan = make_plan(w)
    dev = [t.cuda() for t in make_inputs(w)]
    o, to = torch.empty_like(dev[0]), torch.empty_like(dev[0])
    assert aj.attn_jvp_plan_tensor_map_stats(plan) == (0, 0)
    aj.attn_jvp_fwd(plan, *dev, o, to, None, 0)
    assert aj.attn_jvp_plan_tensor_map_stats(plan) == (6, 0)
    aj.attn_jvp_fwd(plan, *dev, o, to, None, 0)
    assert aj.attn_jvp_plan_tensor_map_stats(plan) == (6, 6)
    q2 = dev[0].clone()                                             # one argument moves: one map is re-encoded
    aj.attn_jvp_fwd(plan, q2, *dev[1:], o, to, None, 0)
    assert aj.attn_jvp_plan_tensor_map_stats(plan) == (7, 11)
    torch.cuda.synchronize()
    aj.attn_jvp_plan_destroy(plan)


def test_fwd_argument_errors():
    w = SMALL_UMMA[4]
    plan = make_plan(w)
    dev = [t.cuda() for t in make_inputs(w)]
    o, to = torch.empty_like(dev[0]), torch.empty_like(dev[0])
    with pytest.raises(aj.AttnJvpError) as e:                      # misaligned pointer
        bad = torch.empty(dev[0].numel() + 8, dtype=torch.bfloat16, device="cuda")[1:1 + dev[0].numel()].view_as(dev[0])
        aj.attn_jvp_fwd(plan, bad, *dev[1:], o, to, None, 0)
    assert e.value.status == aj.AJ_ERR_INVALID_ARG
    with pytest.raises(aj.AttnJvpError) as e:                      # stride_n < d
        aj.attn_jvp_fwd(plan, dev[0].as_strided(dev[0].shape, (w.N * 64, w.N * 64, 64, 1)), *dev[1:], o, to, None, 0)
    assert e.value.status == aj.AJ_ERR_INVALID_ARG
    assert aj.lib().attn_jvp_fwd(plan, None, None, None, None, None, None, None, None, None, None) == aj.AJ_ERR_INVALID_ARG
    with pytest.raises(aj.AttnJvpError) as e:                      # the tcgen05 kernel does not cover fp32
        p32 = make_plan(WORKLOADS["tiny_tf_fp32"])
        try:
            aj.attn_jvp_plan_set_kernel(p32, aj.AJ_KERNEL_UMMA)
        finally:
            aj.attn_jvp_plan_destroy(p32)
    assert e.value.status == aj.AJ_ERR_UNSUPPORTED
    aj.attn_jvp_plan_destroy(plan)
    torch.cuda.synchronize()


# ---------------------------------------------------------------------------------------- configs 2-5 at full size
FULL = ["wan13b_tf_framewise", "wan13b_tf_chunkwise", "block_causal_b2", "dit_large_tf_chunkwise", "dit_large_full"]


@pytest.mark.parametrize("name,kernel", [(n, aj.AJ_KERNEL_AUTO) for n in FULL] + [("wan13b_tf_framewise", aj.AJ_KERNEL_UMMA)],
                         ids=lambda v: v if isinstance(v, str) else {0: "default", 2: "single"}[v])
def test_full_size_config_sampled_rows(name, kernel):
    """The launch configuration bench.py times, against the oracle on the SURVEY.md 8(c) row protocol: every head, every
    query group (first / last row, both sides of every tile boundary, 16 random rows)."""
    w = WORKLOADS[name]
    x = make_inputs(w)
    plan = make_plan(w, kernel)
    assert aj.attn_jvp_plan_kernel(plan)[0] == (aj.AJ_KERNEL_UMMA_PAIR if kernel == aj.AJ_KERNEL_AUTO else kernel)
    pairs, ntasks = aj.attn_jvp_plan_info(plan)
    assert pairs == w.unmasked_pairs_per_head
    gpu = run_gpu(w, x, plan=plan)
    aj.attn_jvp_plan_destroy(plan)
    rows = sample_rows(w)
    assert set(rows) == {(b, h) for b in range(w.B) for h in range(w.H)}
    errs = compare(w, gpu, run_oracle(w, x, rows))
    nrows = sum(len(r) for r in rows.values())
    print(f"{name}: {nrows} rows = {100.0 * nrows / (w.B * w.H * w.num_queries):.2f} % of all rows, errs={errs}")
    # properties that hold at any size: every output written and finite
    for t in gpu:
        assert torch.isfinite(t.float()).all()


def test_config2_one_full_head_every_row():
    """one full head of config 2 -- all 65,520 rows of head (0, 5) of the 12-head launch bench.py times,
    O, tO, lse and the lse tangent, element by element."""
    w = WORKLOADS["wan13b_tf_framewise"]
    x = make_inputs(w)
    plan = make_plan(w)
    dev = [t.cuda() for t in x]
    o, to = torch.full_like(dev[0], float("nan")), torch.full_like(dev[0], float("nan"))
    lse = torch.full((w.B, w.H, w.N), float("nan"), dtype=torch.float32, device="cuda")
    tlse = torch.full_like(lse, float("nan"))
    aj.attn_jvp_fwd(plan, *dev, o, to, lse, torch.cuda.current_stream().cuda_stream, tlse=tlse)
    torch.cuda.synchronize()
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_destroy(plan)
    h = 5
    ro, rto, rlse, rtl = oracle.attn_jvp_head(oracle.teacher_forcing_mask(w.block_len, w.num_blocks),
                                              *[widen(t[0, h]) for t in x], 1.0 / np.sqrt(w.d), with_tlse=True)
    errs = dict(o=max_norm_err(o[0, h].cpu().double().numpy(), ro), to=max_norm_err(to[0, h].cpu().double().numpy(), rto),
                lse=max_norm_err(lse[0, h].cpu().double().numpy(), rlse), tlse=max_norm_err(tlse[0, h].cpu().double().numpy(), rtl))
    print(f"config 2, head {h}, all {w.N} rows: {errs}")
    assert errs["o"] <= 1e-2 and errs["to"] <= 1e-2 and errs["lse"] <= 1e-3 and errs["tlse"] <= 1e-2, errs


# ---------------------------------------------------------------------------------------- the lse tangent (attn_jvp_fwd_tl)
@pytest.mark.parametrize("kernel", [aj.AJ_KERNEL_UMMA_PAIR, aj.AJ_KERNEL_UMMA, aj.AJ_KERNEL_SIMT], ids=["pair", "single", "simt"])
@pytest.mark.parametrize("w", [SMALL_UMMA[0], SMALL_UMMA[2], SMALL_UMMA[3]], ids=lambda w: w.name)
def test_lse_tangent_every_row(w, kernel):
    # tlse = sum_b p_ab tS_ab = r / l, unit-variance tangents so that it is not small
    w = Workload(w.name, w.B, w.H, w.d, w.mask, w.frame_len, w.num_frames, w.chunk_frames, w.dtype, 1.0, w.seed)
    x = make_inputs(w)
    plan = make_plan(w, kernel)
    dev = [t.cuda() for t in x]
    o, to = torch.empty_like(dev[0]), torch.empty_like(dev[0])
    lse = torch.empty((w.B, w.H, w.N), dtype=torch.float32, device="cuda")
    tlse = torch.full_like(lse, float("nan"))
    aj.attn_jvp_fwd(plan, *dev, o, to, lse, 0, tlse=tlse)
    o2, to2, lse2 = torch.empty_like(o), torch.empty_like(o), torch.empty_like(lse)
    aj.attn_jvp_fwd(plan, *dev, o2, to2, lse2, 0)                   # without tlse: the same bits everywhere else
    torch.cuda.synchronize()
    aj.attn_jvp_plan_destroy(plan)
    assert torch.equal(o, o2) and torch.equal(to, to2) and torch.equal(lse, lse2)
    om = oracle_mask(w)
    got, want = [], []
    for b in range(w.B):
        for h in range(w.H):
            want.append(oracle.attn_jvp_head(om, *[widen(t[b, h]) for t in x], 1.0 / np.sqrt(w.d), with_tlse=True)[3])
            got.append(tlse[b, h].cpu().double().numpy())
    err = max_norm_err(np.concatenate(got), np.concatenate(want))
    assert err <= (1e-2 if w.dtype == "bf16" else 1e-4), err


def test_lse_tangent_is_zero_where_tangents_are_structurally_zero():
    w = Workload("tl_cleanzero", 1, 2, 128, "teacher_forcing", 300, 3, 1, "bf16", 1.0, 3, True)
    x = make_inputs(w)
    plan = make_plan(w)                                             # AJ_TANGENT_CLEAN_ZERO from the workload
    dev = [t.cuda() for t in x]
    o, to = torch.empty_like(dev[0]), torch.empty_like(dev[0])
    lse = torch.empty((w.B, w.H, w.N), dtype=torch.float32, device="cuda")
    tlse = torch.full_like(lse, float("nan"))
    aj.attn_jvp_fwd(plan, *dev, o, to, lse, 0, tlse=tlse)
    torch.cuda.synchronize()
    aj.attn_jvp_plan_destroy(plan)
    assert torch.count_nonzero(tlse[:, :, :w.N // 2]) == 0          # clean rows: primal-only tasks
    om = oracle_mask(w)
    for h in range(w.H):
        rtl = oracle.attn_jvp_head(om, *[widen(t[0, h]) for t in x], 1.0 / np.sqrt(w.d), with_tlse=True)[3]
        assert max_norm_err(tlse[0, h].cpu().double().numpy(), rtl) <= 1e-2


# ---------------------------------------------------------------------------------------- Ulysses
@pytest.mark.parametrize("P,G", [(2, 1), (2, 2), (4, 1)])
def test_ulysses_sequence_shards_with_the_cuda_local_op_against_the_oracle(P, G):
    """P virtual ranks in one process, each holding the token shard [B, H, N/P, d]: the production pack / unpack index
    arithmetic with the all-to-all replaced by its definition, the CUDA call as the local op on every head shard (forward
    + JVP, then the primal backward), and the reassembled result against the UNDISTRIBUTED oracle."""
    from paper_2606_25473_b200 import ulysses
    w = Workload("uly_tf", 1, 4, 128, "teacher_forcing", 120, 2, 1, "bf16", 0.1, seed=21)      # N = 480, H = 4
    x = make_inputs(w)
    g = torch.Generator().manual_seed(22)
    dout = torch.randn(x[0].shape, generator=g).to(torch.bfloat16)
    hg = w.H // (P * G)
    wl = Workload("uly_local", w.B, hg, w.d, w.mask, w.frame_len, w.num_frames, w.chunk_frames, w.dtype, w.tangent_std)
    plan = make_plan(wl)                                       # one plan for every head group: (B, H / (P G) heads, N, N)
    fwd, bwd = ulysses.local_attn_jvp(plan), ulysses.local_attn_bwd(plan)
    n = w.N // P
    dev = [t.cuda() for t in x] + [dout.cuda()]
    shards = [[t[:, :, r * n:(r + 1) * n].contiguous() for t in dev] for r in range(P)]
    saved = {}

    def fwd_op(r, grp, q, k, v, tq, tk, tv):
        o, to, lse = fwd(grp, q, k, v, tq, tk, tv)
        saved[(r, grp)] = (q, k, v, o, lse)
        return o, to

    outs = ulysses.emulate_ranks(P, [s[:6] for s in shards], 2, fwd_op, G)
    grads = ulysses.emulate_ranks(P, [s[6:] for s in shards], 3, lambda r, grp, do: bwd(grp, *saved[(r, grp)], do), G)
    torch.cuda.synchronize()
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_destroy(plan)
    o = torch.cat([outs[r][0] for r in range(P)], dim=2).cpu()
    to = torch.cat([outs[r][1] for r in range(P)], dim=2).cpu()
    lse = torch.empty((w.B, w.H, w.N), dtype=torch.float32)
    h = w.H // P
    for (r, grp), sv in saved.items():
        lse[:, r * h + grp * hg:r * h + (grp + 1) * hg] = sv[4].cpu()
    compare(w, (o, to, lse), run_oracle(w, x))
    om = oracle_mask(w)
    for i, name in enumerate(("dq", "dk", "dv")):
        got = torch.cat([grads[r][i] for r in range(P)], dim=2).cpu()
        for hh in range(w.H):
            ref = oracle.attn_bwd_head(om, widen(x[0][0, hh]), widen(x[1][0, hh]), widen(x[2][0, hh]), widen(dout[0, hh]),
                                       1.0 / np.sqrt(w.d))[i]
            assert max_norm_err(got[0, hh].double().numpy(), ref) <= 1e-2, (name, hh)


def test_ulysses_local_ops_follow_torchs_current_stream():
    """local_attn_jvp / local_attn_bwd without a stream argument launch on torch's current stream AT CALL TIME: under
    `with torch.cuda.stream(s)` the inputs are produced on s (here behind a long sleep), so a kernel on the legacy default
    stream would read them before they exist.  Same bits as the synchronous run."""
    from paper_2606_25473_b200 import ulysses
    w = SMALL_UMMA[0]
    x = make_inputs(w)
    g = torch.Generator().manual_seed(23)
    dout = torch.randn(x[0].shape, generator=g).to(w.torch_dtype)
    plan = make_plan(w)
    fwd, bwd = ulysses.local_attn_jvp(plan), ulysses.local_attn_bwd(plan)
    dev = [t.cuda() for t in x] + [dout.cuda()]
    o, to, lse = fwd(0, *dev[:6])
    ref = (o, to, lse) + bwd(0, dev[0], dev[1], dev[2], o, lse, dev[6])
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        torch.cuda._sleep(200_000_000)                       # ~0.1 s: everything below on s is still pending when enqueued
        late = [torch.zeros_like(t).copy_(t, non_blocking=True) for t in dev]
        o, to, lse = fwd(0, *late[:6])
        got = (o, to, lse) + bwd(0, late[0], late[1], late[2], o, lse, late[6])
    torch.cuda.synchronize()
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_destroy(plan)
    for a, b in zip(got, ref):
        assert torch.equal(a, b)


def test_ulysses_pipeline_with_nccl_world_size_1():
    """The production pipeline (async all_to_all_single per head group on NCCL, here one rank = one GPU, so the exchanges
    are identities): same bits as the direct call on all heads."""
    import torch.distributed as dist
    from paper_2606_25473_b200 import ulysses
    w = SMALL_UMMA[0]
    x = make_inputs(w)
    plan = make_plan(w)
    ref = run_gpu(w, x, plan=plan)
    aj.attn_jvp_plan_destroy(plan)
    wl = Workload("uly_local1", w.B, 1, w.d, w.mask, w.frame_len, w.num_frames, w.chunk_frames, w.dtype, w.tangent_std)
    plan = make_plan(wl)
    own = not dist.is_initialized()
    if own:
        dist.init_process_group("nccl", init_method="tcp://127.0.0.1:29517", rank=0, world_size=1)
    try:
        o, to, saved = ulysses.ulysses_attn_jvp(ulysses.local_attn_jvp(plan, torch.cuda.current_stream().cuda_stream),
                                                *[t.cuda() for t in x], head_groups=w.H)
        torch.cuda.synchronize()
    finally:
        if own:
            dist.destroy_process_group()
    aj.attn_jvp_plan_destroy(plan)
    lse = torch.cat([s[4] for s in saved], dim=1)
    assert torch.equal(o.cpu(), ref[0]) and torch.equal(to.cpu(), ref[1]) and torch.equal(lse.cpu(), ref[2])
