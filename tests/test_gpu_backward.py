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


BF16_D128 = [w for w in SMALL if w.dtype == "bf16" and w.d == 128]


@pytest.mark.parametrize("w", BF16_D128, ids=lambda w: w.name)
def test_backward_single_cta_tcgen05_kernel_every_element(w):
    # a plan forced to AJ_KERNEL_UMMA runs the single-CTA backward (128 stationary rows per CTA, per-group tiling); the default
    # (test_backward_small_every_element) is the CTA-pair backward (256 rows per SM pair, packed tiling)
    x = make_inputs(w)
    dout = _dout(w)
    got = run_fwd_bwd(w, x, dout, kernel=aj.AJ_KERNEL_UMMA)
    check(w, x, dout, got)
    pair = run_fwd_bwd(w, x, dout)
    for u, v in zip(got, pair):
        assert max_norm_err(u.double().numpy(), v.double().numpy()) <= 1e-2


BF16_D64 = [
    Workload("bwd_d64_tf_L200", 1, 2, 64, "teacher_forcing", 200, 3, 1, "bf16", 0.1, seed=40),
    Workload("bwd_d64_tf_chunk_L100", 1, 2, 64, "teacher_forcing", 100, 6, 3, "bf16", 0.1, seed=41),
    Workload("bwd_d64_bc_L137_B2", 2, 2, 64, "block_causal", 137, 4, 1, "bf16", 0.1, seed=42),
    Workload("bwd_d64_full_N517", 1, 3, 64, "full", 517, 1, 1, "bf16", 0.1, seed=43),
    Workload("bwd_d64_tf_L8", 1, 1, 64, "teacher_forcing", 8, 2, 1, "bf16", 0.1, seed=44),
    Workload("bwd_d64_tf_L1560_F2", 1, 1, 64, "teacher_forcing", 1560, 2, 1, "bf16", 0.1, seed=45),
    Workload("bwd_d64_tf_unit", 1, 2, 64, "teacher_forcing", 300, 3, 1, "bf16", 1.0, seed=46),
]


@pytest.mark.parametrize("w", BF16_D64, ids=lambda w: w.name)
def test_backward_bf16_d64_runs_the_single_cta_tcgen05_kernels_every_element(w):
    # bf16 with d = 64: forward and backward on the single-CTA tcgen05 kernels (one 64-column swizzle block per operand row);
    # the plain-FMA kernels on the same plan as an on-GPU cross-check
    x = make_inputs(w)
    dout = _dout(w)
    plan = make_plan(w)
    assert aj.attn_jvp_plan_kernel(plan)[0] == aj.AJ_KERNEL_UMMA
    got = run_fwd_bwd(w, x, dout, plan)
    got2 = run_fwd_bwd(w, x, dout, plan)
    aj.attn_jvp_plan_set_kernel(plan, aj.AJ_KERNEL_SIMT)
    simt = run_fwd_bwd(w, x, dout, plan)
    aj.attn_jvp_plan_destroy(plan)
    check(w, x, dout, got)
    check(w, x, dout, simt)
    for a, b in zip(got, got2):
        assert torch.equal(a, b)
    assert any(not torch.equal(a, b) for a, b in zip(got, simt)), "the forced plain-FMA run must be a different kernel"


def test_backward_pair_kernel_many_tasks_per_pair_and_long_streams():
    # more 256-row tasks than SM pairs (148 + tasks on 74 pairs: every pair runs several tasks back to back, with the
    # accumulators, the TMEM A operands and the {lse, delta} stages reused), long streams with odd tile counts
    w = Workload("bwd_bc_bf16_many", 2, 4, 128, "block_causal", 1000, 5, 1, "bf16", 0.1, seed=31)
    x = make_inputs(w)
    dout = _dout(w)
    got = run_fwd_bwd(w, x, dout)
    check(w, x, dout, got, heads=[(0, 0), (1, 3)])
    for t in got:
        assert torch.isfinite(t.float()).all()


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


# ---------------------------------------------------------------------------------------- full size (what bench.py times)
FULL_SIZE_BACKWARD = ["wan13b_tf_framewise_bwd", "wan13b_tf_framewise_d64_bwd"]     # EXTRA_WORKLOADS whose step is attn_bwd


def _block_samples(w, rng, per_block=6):
    """first, last, both sides of the 128- / 256-row tile boundaries next to the block's ends, and random tokens of every block"""
    C, n = w.block_len, w.num_blocks
    idx = []
    for blk in range(2 * n if w.mask == "teacher_forcing" else n):
        q0, q1 = blk * C, (blk + 1) * C
        first256, last256 = (q0 // 256 + 1) * 256, ((q1 - 1) // 256) * 256
        cand = [q0, q1 - 1, first256 - 1, first256, last256 - 1, last256, q0 + 127, q0 + 128]
        cand += list(rng.integers(q0, q1, size=per_block))
        idx += [int(r) for r in cand if q0 <= r < q1]
    return np.unique(np.asarray(idx, dtype=np.int64))


@pytest.mark.parametrize("name", FULL_SIZE_BACKWARD)
def test_backward_full_size_all_heads_launch_sampled(name):
    """The launch bench.py times for the backward workload: all heads in one attn_bwd call (host-assigned head-major
    task lists), compared on three heads -- the first, a middle one and the LAST one the lists schedule -- at sampled query
    rows and keys of every block (the oracle's pass over all rows of a head supplies lse and delta)."""
    from paper_2606_25473_b200.workloads import EXTRA_WORKLOADS
    w = EXTRA_WORKLOADS[name]
    assert w.backward and w.H >= 12
    x = make_inputs(w)
    dout = _dout(w)
    got = run_fwd_bwd(w, x, dout)
    for t in got:
        assert torch.isfinite(t.float()).all()
    heads = [(0, 0), (0, w.H // 2 - 1), (0, w.H - 1)]
    for i, bh in enumerate(heads):
        idx = _block_samples(w, np.random.default_rng(50 + i))
        errs = check(w, x, dout, got, heads=[bh], rows=idx, keys=idx)
        print(f"{w.name} head {bh}: {len(idx)} rows and keys, errs={errs}")
    half, C, n = w.N // 2, w.block_len, w.num_blocks
    assert torch.count_nonzero(got[1][:, :, half + (n - 1) * C:]) > 0      # the last noisy block's keys are seen by itself


@pytest.mark.parametrize("name", ["wan13b_tf_chunkwise", "block_causal_b2"])
def test_backward_full_size_other_masks_sampled(name):
    """The transposed packed schedules of the chunk-wise mask (4680-row blocks) and of B = 2 block-causal at full size, all heads
    in one attn_bwd call: two heads (the first, and the last head of the last batch) at sampled rows and keys of every block."""
    import dataclasses
    from paper_2606_25473_b200.workloads import WORKLOADS
    w = dataclasses.replace(WORKLOADS[name], name=name + "_bwd", backward=True)
    x = make_inputs(w)
    dout = _dout(w)
    got = run_fwd_bwd(w, x, dout)
    for t in got:
        assert torch.isfinite(t.float()).all()
    for i, bh in enumerate([(0, 0), (w.B - 1, w.H - 1)]):
        idx = _block_samples(w, np.random.default_rng(60 + i), per_block=4)
        errs = check(w, x, dout, got, heads=[bh], rows=idx, keys=idx)
        print(f"{w.name} head {bh}: {len(idx)} rows and keys, errs={errs}")


def test_backward_config2_one_full_head_every_element():
    """One full head of config 2 through the 12-head launch: every row of dQ and every key of dK, dV of head (0, 11)."""
    from paper_2606_25473_b200.workloads import EXTRA_WORKLOADS
    w = EXTRA_WORKLOADS["wan13b_tf_framewise_bwd"]
    x = make_inputs(w)
    dout = _dout(w)
    got = run_fwd_bwd(w, x, dout)
    errs = check(w, x, dout, got, heads=[(0, w.H - 1)])
    print(f"{w.name} head (0, {w.H - 1}), every element: {errs}")


@pytest.mark.parametrize("w", [SMALL[4], SMALL[0]], ids=lambda w: w.name)
def test_bwd_host_matches_device_path(w):
    # attn_bwd_host: per-head copies and launches on three streams; same bits as the one-launch device path
    x = make_inputs(w, pin=True)
    dout = _dout(w).pin_memory()
    plan = make_plan(w)
    q, k, v, tq, tk, tv = [t.cuda() for t in x]
    o, to = torch.empty_like(q), torch.empty_like(q)
    lse = torch.empty((w.B, w.H, w.N), dtype=torch.float32, device="cuda")
    aj.attn_jvp_fwd(plan, q, k, v, tq, tk, tv, o, to, lse, 0)
    dq, dk, dv = torch.empty_like(q), torch.empty_like(k), torch.empty_like(k)
    aj.attn_bwd(plan, q, k, v, o, lse, dout.cuda(), dq, dk, dv, 0)
    torch.cuda.synchronize()
    h_o, h_lse = o.cpu().pin_memory(), lse.cpu().pin_memory()
    h = [torch.full_like(x[0], float("nan")).pin_memory(), torch.full_like(x[1], float("nan")).pin_memory(),
         torch.full_like(x[1], float("nan")).pin_memory()]
    encodes = []
    for _ in range(3):                                  # later calls reuse staging buffers, schedules and tensor maps
        aj.attn_bwd_host(plan, x[0], x[1], x[2], h_o, h_lse, dout, *h, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        for a, b in zip(h, (dq, dk, dv)):
            assert torch.equal(a, b.cpu())
        for t in h:
            t.fill_(float("nan"))
        encodes.append(aj.attn_jvp_plan_tensor_map_stats(plan)[0])
        aj.attn_bwd(plan, q, k, v, o, lse, dout.cuda(), dq, dk, dv, 0)     # alternating with the device call evicts nothing either
        torch.cuda.synchronize()
    # steady state encodes nothing, including the per-head augmentation-row maps of the CTA-pair dK/dV pass
    assert encodes[1] == encodes[0] and encodes[2] == encodes[0] == aj.attn_jvp_plan_tensor_map_stats(plan)[0], encodes
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_destroy(plan)


def test_forward_and_backward_replay_from_a_cuda_graph():
    """SURVEY.md 8(b) "no hidden stream sync" / PAPER.md:534 (CUDA Graphs): after one eager call (attn_bwd builds its
    schedules on first use) attn_jvp_fwd + attn_bwd are captured into a graph; two replays on fresh inputs give the bits of
    the eager calls; the plan's tensor-map cache encodes nothing in steady state."""
    w = SMALL[4]
    x = make_inputs(w)
    dout = _dout(w)
    plan = make_plan(w)
    q, k, v, tq, tk, tv = [t.cuda() for t in x]
    dO = dout.cuda()
    o, to = torch.empty_like(q), torch.empty_like(q)
    lse = torch.empty((w.B, w.H, w.N), dtype=torch.float32, device="cuda")
    dq, dk, dv = torch.empty_like(q), torch.empty_like(k), torch.empty_like(k)
    side = torch.cuda.Stream()

    def step(stream):
        aj.attn_jvp_fwd(plan, q, k, v, tq, tk, tv, o, to, lse, stream)
        aj.attn_bwd(plan, q, k, v, o, lse, dO, dq, dk, dv, stream)

    with torch.cuda.stream(side):
        step(side.cuda_stream)
    side.synchronize()
    eager = [t.clone() for t in (o, to, lse, dq, dk, dv)]
    enc0, hits0 = aj.attn_jvp_plan_tensor_map_stats(plan)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        step(side.cuda_stream)
    enc1, hits1 = aj.attn_jvp_plan_tensor_map_stats(plan)
    assert enc1 == enc0 and hits1 >= hits0 + 13          # 6 forward + 7 backward maps (CTA-pair passes), all from the plan's cache
    for _ in range(2):
        for t in (o, to, lse, dq, dk, dv):
            t.fill_(float("nan"))
        graph.replay()
        torch.cuda.synchronize()
        for a, b in zip((o, to, lse, dq, dk, dv), eager):
            assert torch.equal(a, b)
    # new data in the same buffers: the replay follows it
    q.copy_((x[0].float() * 0.5).to(q.dtype))
    graph.replay()
    torch.cuda.synchronize()
    ref = [t.clone() for t in (o, dq)]
    step(0)
    torch.cuda.synchronize()
    assert torch.equal(ref[0], o) and torch.equal(ref[1], dq)
    assert aj.attn_jvp_plan_device_status(plan) == 0
    aj.attn_jvp_plan_destroy(plan)
