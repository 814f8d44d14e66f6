"""Shared by the `-m gpu` tests: run a workload through the C ABI, run the oracle, pick rows to compare."""
import numpy as np
import torch

import oracle
from helpers import oracle_mask, widen, max_norm_err
from paper_2606_25473_b200 import binding as aj
from paper_2606_25473_b200.workloads import Workload, make_inputs

# BASELINE.json north_star tolerances, max|err| / max|ref| per tensor
TOL = {"bf16": dict(o=1e-2, to=1e-2, lse=1e-3), "fp32": dict(o=1e-4, to=1e-4, lse=1e-4)}


def mask_kind(w: Workload) -> int:
    return {"teacher_forcing": aj.AJ_MASK_TEACHER_FORCING, "block_causal": aj.AJ_MASK_BLOCK_CAUSAL,
            "full": aj.AJ_MASK_FULL}[w.mask]


def make_plan(w: Workload, kernel: int = aj.AJ_KERNEL_AUTO, scale: float = 0.0, tangent_zero=None):
    """tangent_zero: an aj_tangent_zero promise; default = what the workload's data guarantees."""
    prob = aj.make_problem(w.B, w.H, w.num_queries, w.N, w.d, aj.AJ_BF16 if w.dtype == "bf16" else aj.AJ_FP32, scale)
    if tangent_zero is None:
        tangent_zero = (aj.AJ_TANGENT_NONE if w.no_tangents else
                        aj.AJ_TANGENT_CLEAN_ZERO if w.clean_tangent_zero else aj.AJ_TANGENT_DENSE)
    mask, keep = aj.make_mask(mask_kind(w), w.frame_len, w.num_frames, w.chunk_frames, tangent_zero=tangent_zero)
    plan = aj.attn_jvp_plan_create(prob, mask)
    if kernel != aj.AJ_KERNEL_AUTO:
        aj.attn_jvp_plan_set_kernel(plan, kernel)
    return plan


def run_gpu(w: Workload, inputs_cpu, kernel: int = aj.AJ_KERNEL_AUTO, plan=None):
    """-> (o, to, lse) on the CPU.  Outputs start as NaN so that an unwritten row fails the comparison."""
    own = plan is None
    if own:
        plan = make_plan(w, kernel)
    dev = [x.cuda() for x in inputs_cpu]
    o = torch.full_like(dev[0], float("nan"))
    to = torch.full_like(dev[0], float("nan"))
    lse = torch.full((w.B, w.H, w.num_queries), float("nan"), dtype=torch.float32, device="cuda")
    if w.no_tangents:                      # forward only: no tangent goes in, none comes out (tO = 0 by definition)
        aj.attn_fwd(plan, *dev[:3], o, lse, torch.cuda.current_stream().cuda_stream)
        to.zero_()
    else:
        aj.attn_jvp_fwd(plan, *dev, o, to, lse, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert aj.attn_jvp_plan_device_status(plan) == 0, "the kernel abandoned a launch (pipeline wait timed out)"
    if own:
        aj.attn_jvp_plan_destroy(plan)
    return o.cpu(), to.cpu(), lse.cpu()


def run_oracle(w: Workload, inputs_cpu, rows_by_head=None):
    """rows_by_head: {(b, h): int64 rows} or None for every row of every head.
    -> {(b, h): (rows, o, to, lse)} in fp64."""
    om = oracle_mask(w)
    scale = 1.0 / np.sqrt(w.d)
    out = {}
    for b in range(w.B):
        for h in range(w.H):
            if rows_by_head is not None and (b, h) not in rows_by_head:
                continue
            rows = None if rows_by_head is None else np.asarray(rows_by_head[(b, h)], dtype=np.int64)
            args = [widen(x[b, h]) for x in inputs_cpu]
            o, to, lse = oracle.attn_jvp_head(om, *args, scale, rows)
            out[(b, h)] = (np.arange(w.num_queries) if rows is None else rows, o, to, lse)
    return out


def compare(w: Workload, gpu, ref, tol=None):
    """Max-normalised error per tensor over all compared rows (R11)."""
    tol = tol or TOL[w.dtype]
    o, to, lse = gpu
    got = {"o": [], "to": [], "lse": []}
    want = {"o": [], "to": [], "lse": []}
    for (b, h), (rows, ro, rto, rlse) in ref.items():
        got["o"].append(o[b, h, rows].double().numpy()); want["o"].append(ro)
        got["to"].append(to[b, h, rows].double().numpy()); want["to"].append(rto)
        got["lse"].append(lse[b, h, rows].double().numpy()); want["lse"].append(rlse)
    errs = {}
    for key in got:
        g, r = np.concatenate(got[key]), np.concatenate(want[key])
        assert np.all(np.isfinite(g)), f"{w.name}: non-finite or unwritten {key}"
        errs[key] = max_norm_err(g, r)
    for key in errs:
        assert errs[key] <= tol[key], f"{w.name}: {key} error {errs[key]:.3e} > {tol[key]:.1e} (all: {errs})"
    return errs


def query_groups(w: Workload):
    """The mask's query groups as [(q_begin, q_end)] from the block structure (test-side accounting)."""
    C, n = w.block_len, w.num_blocks
    if w.mask == "full":
        return [(0, w.num_queries)]
    if w.mask == "block_causal":
        return [(i * C, (i + 1) * C) for i in range(n)]
    return [(i * C, (i + 1) * C) for i in range(2 * n)]


def sample_rows(w: Workload, random_per_group: int = 16, max_boundaries: int = 64, heads=None, seed: int = 1234):
    """SURVEY.md 8(c) "GPU-vs-oracle protocol" for the full-size configs: for EVERY (b, h) (or those in `heads`) and EVERY
    query group -- its first and last row, the rows on both sides of every query-tile boundary that falls inside it (the
    global 256- and 128-row grids of the packed tilings and the group-relative 128-row grid of per-group tiling; at most
    `max_boundaries` of them per group and grid, seeded choice, when a group holds more), and `random_per_group` seeded
    random rows.  -> {(b, h): sorted unique int64 rows}.  Asserts that every group is hit on every head."""
    groups = query_groups(w)
    out = {}
    for b in range(w.B):
        for h in range(w.H):
            if heads is not None and (b, h) not in heads:
                continue
            rng = np.random.default_rng([seed, b, h])
            rows, hit = [], set()
            for g, (q0, q1) in enumerate(groups):
                cand = [q0, q1 - 1]
                for grid, origin in ((256, 0), (128, 0), (128, q0)):
                    first = origin + ((q0 - origin) // grid + 1) * grid
                    bnd = np.arange(first, q1, grid)
                    if len(bnd) > max_boundaries:
                        bnd = rng.choice(bnd, size=max_boundaries, replace=False)
                    for t in bnd:
                        cand += [int(t) - 1, int(t)]
                # at least `random_per_group` random rows, and enough of them that about 2 % of a large group is compared
                n_rand = max(random_per_group, min(1024, int(0.02 * (q1 - q0)) - len(cand)))
                cand += [int(r) for r in rng.integers(q0, q1, size=n_rand)]
                cand = [r for r in cand if q0 <= r < q1]
                assert len(cand) >= min(random_per_group, q1 - q0)
                rows += cand
                hit.add(g)
            assert hit == set(range(len(groups))), "every query group must be sampled on every head"
            out[(b, h)] = np.unique(np.asarray(rows, dtype=np.int64))
    return out
