#!/usr/bin/env python
"""Benchmark of the fused attention-JVP hot path (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl reference]

A step = one pass of the whole hot path (schedule already planned; one `attn_jvp_fwd` call = one kernel launch)
over one batch of synthetic input of the BASELINE.json configs[1] shape (Wan2.1-1.3B-shaped frame-wise
teacher-forcing JVP).  Prints ONE JSON line (rank 0).  FLOP convention: 12*d flop per unmasked (query, key)
pair (six length-d contractions); padded tile area, masked pairs and the softmax are
not counted.  N > 1: every rank runs its own head shard (B, H heads each; Ulysses-style head sharding,
PAPER.md:318) with no data-path collective -> "scaling": "weak".

`--ulysses`: the ranks hold SEQUENCE shards [B, H, N/P, d] of ONE problem; a step = packed all-to-all
in per head group, the kernel on the rank's head shard, packed all-to-all out (paper_2606_25473_b200/ulysses.py), timed
whole and in parts -> "scaling": "strong".  On a box without CUDA it is a dry run of the exchange (gloo, no kernel).

`--impl reference` times the fp64 CPU oracle (oracle/, as it stands) on the host cores on a bounded row sample
of the same workload; rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

from paper_2606_25473_b200.workloads import EXTRA_WORKLOADS, WORKLOADS, Workload, make_inputs

METRIC = "attention-JVP TFLOPS (unmasked pairs)"
UNIT = "TFLOP/s"
DEFAULT_WORKLOAD = "wan13b_tf_framewise"
FALLBACK_PEAKS = {"bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "hbm_gbs": 6650.0}   # B200_PROFILING.md


def pair_classes(w: Workload):
    """Unmasked pairs per head needing 2 / 4 / 6 length-d contractions (accounting only).  Dense tangents: all 6.
    Zero clean tangents: clean x clean pairs need S and P V only, noisy x clean pairs also tQ K^T and H V."""
    if w.no_tangents:
        return [w.unmasked_pairs_per_head, 0, 0]
    if not w.clean_tangent_zero:
        return [0, 0, w.unmasked_pairs_per_head]
    n, C = w.num_blocks, w.block_len
    return [n * (n + 1) // 2 * C * C, n * (n - 1) // 2 * C * C, n * C * C]


def flops_per_call(w: Workload) -> float:
    """2*d flop per contraction per unmasked pair: 12*d per pair with dense tangents (the BASELINE.json convention)."""
    if w.backward:      # five contractions per pair: S recomputed, dP = dO V^T, dV += P^T dO, dK += dS^T Q, dQ += dS K
        return 10.0 * w.d * w.unmasked_pairs_per_head * w.B * w.H
    c = pair_classes(w)
    return 2.0 * w.d * (2 * c[0] + 4 * c[1] + 6 * c[2]) * w.B * w.H


def allowed_keys_per_row(w: Workload, rows: np.ndarray) -> np.ndarray:
    """Size of a row's allowed key set from the block structure (accounting only, for the CPU sample)."""
    C, n = w.block_len, w.num_blocks
    if w.mask == "full":
        return np.full(rows.shape, w.N, dtype=np.int64)
    blk = (rows // C) % n          # clean block i and noisy block i both see (i + 1) * C keys
    return (blk + 1) * C


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return dict(FALLBACK_PEAKS), "fallback"


def recorded_traffic(workload: str):
    """DRAM bytes per launch of the dominant kernel from the committed ncu --set full capture, if any, and where the figure
    comes from (rows of profiles/dram_traffic.csv: workload, kernel / capture name, bytes): -> (bytes, source) or (None, None).
    The last matching row wins; the source names it so that a capture older than the kernel is visible in the line."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    if not os.path.exists(path):
        return None, None
    best, src = None, None
    with open(path) as f:
        for line in f:
            parts = [p.strip() for p in line.split(",")]
            if len(parts) >= 3 and parts[0] == workload:
                try:
                    best, src = float(parts[2]), f"profiles/dram_traffic.csv: {parts[1]}"
                except ValueError:
                    pass
    return best, src


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")
    REASONS = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu_index = gpu_index
        self.proc = None
        self.out = None

    def start(self):
        try:
            self.out = tempfile.TemporaryFile(mode="w+")
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.gpu_index), f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=self.out, stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self):
        res = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return res
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.out.seek(0)
        sm, smax, power, reasons = [], [], [], set()
        for line in self.out.read().splitlines():
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for name, val in zip(self.REASONS, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        self.out.close()
        if sm:
            # "under load" = samples in the upper half of the power range (skips idle samples at the edges)
            thr = 0.5 * (max(power) + min(power))
            loaded = [c for c, p in zip(sm, power) if p >= thr] or sm
            loaded_p = [p for p in power if p >= thr] or power
            res.update(sm_mhz=statistics.median(loaded), sm_max_mhz=max(smax), reasons=sorted(reasons),
                       samples=len(sm), power_w_max=max(power), power_w_loaded=sum(loaded_p) / len(loaded_p))
        return res


# ----------------------------------------------------------------------------------------------- CPU oracle legs
def time_oracle_sample(w: Workload, inputs, budget_s: float, seed: int = 0):
    """Runs the oracle as it stands on a seeded uniform row sample of head (0, 0) sized to ~budget_s seconds.
    -> (TFLOP/s under the 12*d convention, seconds, number of rows, cores, (rows, o, to, lse) of the sample)."""
    import oracle
    oracle.build()
    om = {"teacher_forcing": oracle.teacher_forcing_mask, "block_causal": oracle.block_causal_mask}.get(w.mask)
    om = om(w.block_len, w.num_blocks) if om else oracle.full_mask()
    args = [x[0, 0].float().numpy() for x in inputs]
    scale = 1.0 / float(np.sqrt(w.d))
    rng = np.random.default_rng(seed)
    pilot = np.sort(rng.integers(0, w.num_queries, size=64))
    t0 = time.perf_counter()
    oracle.attn_jvp_head(om, *args, scale, pilot)
    dt = max(time.perf_counter() - t0, 1e-6)
    nrows = int(min(max(64, budget_s / dt * 64), 4 * w.num_queries))
    rows = np.sort(rng.integers(0, w.num_queries, size=nrows))
    t0 = time.perf_counter()
    ref = oracle.attn_jvp_head(om, *args, scale, rows)
    dt = time.perf_counter() - t0
    flops = 12.0 * w.d * float(allowed_keys_per_row(w, rows).sum())
    return flops / dt / 1e12, dt, nrows, oracle.num_threads(), (rows,) + tuple(ref)


def rows_seeing_key(w: Workload, keys: np.ndarray) -> np.ndarray:
    """How many query rows see each key, from the block structure (accounting only, for the CPU backward sample)."""
    C, n = w.block_len, w.num_blocks
    if w.mask == "full":
        return np.full(keys.shape, w.num_queries, dtype=np.int64)
    if w.mask == "block_causal":
        return (n - keys // C) * C
    half = w.N // 2
    j = (keys % half) // C
    return np.where(keys < half, (n - j) * C + (n - 1 - j) * C, C)   # clean key: clean blocks >= j and noisy blocks > j


def time_oracle_bwd_sample(w: Workload, q, k, v, dout, n_sample: int, seed: int = 0):
    """The backward oracle as it stands on head (0, 0): its pass over ALL query rows (lse and delta, which every key needs)
    plus dQ of `n_sample` seeded rows and dK, dV of `n_sample` seeded keys.
    -> (TFLOP/s over the contractions the oracle executed, seconds, cores, (rows, keys, dq, dk, dv))."""
    import oracle
    oracle.build()
    om = {"teacher_forcing": oracle.teacher_forcing_mask, "block_causal": oracle.block_causal_mask}.get(w.mask)
    om = om(w.block_len, w.num_blocks) if om else oracle.full_mask()
    rng = np.random.default_rng(seed)
    rows = np.unique(rng.integers(0, w.num_queries, size=n_sample))
    keys = np.unique(rng.integers(0, w.N, size=n_sample))
    args = [x[0, 0].float().numpy() for x in (q, k, v, dout)]
    t0 = time.perf_counter()
    dq, dk, dv = oracle.attn_bwd_head(om, *args, 1.0 / float(np.sqrt(w.d)), rows, keys)
    dt = time.perf_counter() - t0
    # executed: S and dP for every pair of the head (2 contractions), dQ for the sampled rows (1), S, dP, dK, dV for the sampled keys (4)
    flops = 2.0 * w.d * (2.0 * w.unmasked_pairs_per_head + float(allowed_keys_per_row(w, rows).sum()) +
                         4.0 * float(rows_seeing_key(w, keys).sum()))
    return flops / dt / 1e12, dt, oracle.num_threads(), (rows, keys, dq, dk, dv)


def run_reference(args, w: Workload):
    """--impl reference: the oracle on the host cores; each step is a bounded row sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    inputs = make_inputs(w)
    steps, warmup = args.steps, args.warmup
    budget = min(6.0, 150.0 / (steps + warmup))
    for i in range(warmup):
        time_oracle_sample(w, inputs, budget, seed=100 + i)
    tot_flops, tot_s, tot_rows, cores = 0.0, 0.0, 0, 1
    for i in range(steps):
        tf, dt, nrows, cores, _ = time_oracle_sample(w, inputs, budget, seed=i)
        tot_flops += tf * 1e12 * dt
        tot_s += dt
        tot_rows += nrows
    value = tot_flops / tot_s / 1e12
    sample = f"{tot_rows // steps} uniformly sampled query rows of head (0,0) per step, all their allowed keys"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": warmup, "ms_per_step": 1e3 * tot_s / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(w),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "tokens_per_s": tot_rows / tot_s, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(w: Workload):
    return {"workload": w.name, "B": w.B, "H": w.H, "d": w.d, "N": w.N, "mask": w.mask, "frame_len": w.frame_len,
            "num_frames": w.num_frames, "chunk_frames": w.chunk_frames, "input_dtype": w.dtype,
            "unmasked_pairs_per_head": w.unmasked_pairs_per_head,
            "Nq": w.num_queries,
            "tangents": "none (forward only)" if w.no_tangents else "zero on the clean half" if w.clean_tangent_zero else "dense",
            "pass": "primal backward (attn_bwd)" if w.backward else "forward",
            "flop_convention": ("10*d per unmasked pair (S, dP, dV, dK, dQ)" if w.backward else
                                "4*d per unmasked pair (S and P V only)" if w.no_tangents else
                                "2*d per contraction actually needed per unmasked pair (2, 4 or 6 of them: zero clean tangents)"
                                if w.clean_tangent_zero else "12*d per unmasked pair"),
            "l2": ("no flush: the inputs (%.2f GB) are larger than the 126 MB L2" % (input_bytes(w) / 1e9) if not needs_l2_flush(w) else
                   "flushed: a 256 MB buffer is overwritten between timed launches (the inputs, %.3f GB, would stay in the 126 MB L2); "
                   "every launch is timed by its own event pair" % (input_bytes(w) / 1e9))}


def input_bytes(w: Workload) -> int:
    eb = 2 if w.dtype == "bf16" else 4
    per_q, per_k = w.B * w.H * w.num_queries * w.d * eb, w.B * w.H * w.N * w.d * eb
    return (1 if w.no_tangents else 2) * (per_q + 2 * per_k)


def needs_l2_flush(w: Workload) -> bool:
    return input_bytes(w) < 2 * 126e6


# ----------------------------------------------------------------------------------------------- distributed glue
def dist_setup(n_gpus: int):
    """One process per GPU (torchrun env).  -> (rank, world, local_rank, initialised)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        backend = "nccl" if torch.cuda.is_available() else "gloo"
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
        return rank, world, local, True
    if n_gpus > 1:
        raise SystemExit("bench.py --gpus N > 1 must be launched with torch.distributed.run (one rank per GPU)")
    return 0, 1, 0, False


def aggregate(elapsed_ms: float, units: float, initialised: bool, device: str = "cpu"):
    """Whole-job numbers: time = max over ranks, units = sum over ranks (no data-path collective anywhere else)."""
    if not initialised:
        return elapsed_ms, units
    import torch.distributed as dist
    t = torch.tensor([elapsed_ms], dtype=torch.float64, device=device)
    u = torch.tensor([units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def barrier(initialised: bool):
    if initialised:
        import torch.distributed as dist
        dist.barrier()


# ----------------------------------------------------------------------------------------------- the CUDA arm
def run_cuda(args, w: Workload):
    from paper_2606_25473_b200 import binding as aj

    rank, world, local, inited = dist_setup(args.gpus)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the attention-JVP path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    stream = torch.cuda.current_stream()
    kind = {"teacher_forcing": aj.AJ_MASK_TEACHER_FORCING, "block_causal": aj.AJ_MASK_BLOCK_CAUSAL,
            "full": aj.AJ_MASK_FULL}[w.mask]
    prob = aj.make_problem(w.B, w.H, w.num_queries, w.N, w.d, aj.AJ_BF16 if w.dtype == "bf16" else aj.AJ_FP32)
    tz = aj.AJ_TANGENT_NONE if w.no_tangents else aj.AJ_TANGENT_CLEAN_ZERO if w.clean_tangent_zero else aj.AJ_TANGENT_DENSE
    mask, keep = aj.make_mask(kind, w.frame_len, w.num_frames, w.chunk_frames, tangent_zero=tz)
    t0 = time.perf_counter()
    plan = aj.attn_jvp_plan_create(prob, mask)
    plan_ms = 1e3 * (time.perf_counter() - t0)
    kernel, launches_per_call = aj.attn_jvp_plan_kernel(plan)
    pairs, num_tasks = aj.attn_jvp_plan_info(plan)
    assert pairs == w.unmasked_pairs_per_head and aj.attn_jvp_plan_pair_classes(plan) == pair_classes(w)

    # every rank draws its own head shard (seed + rank): weak scaling, no exchange
    wr = Workload(w.name, w.B, w.H, w.d, w.mask, w.frame_len, w.num_frames, w.chunk_frames, w.dtype, w.tangent_std,
                  w.seed + rank, w.clean_tangent_zero, w.no_tangents, w.Nq, w.backward)
    host_all = make_inputs(wr, pin=True)
    host = host_all[:3] + [None, None, None] if w.no_tangents else host_all   # the forward-only call takes no tangents
    devin = [None if x is None else x.to(dev, non_blocking=True) for x in host]
    o = torch.empty_like(devin[0])
    to = None if w.no_tangents else torch.empty_like(devin[0])
    lse = torch.empty((w.B, w.H, w.num_queries), dtype=torch.float32, device=dev)
    h_o = torch.empty_like(host[0]).pin_memory()
    h_to = None if w.no_tangents else torch.empty_like(host[0]).pin_memory()
    h_lse = torch.empty((w.B, w.H, w.num_queries), dtype=torch.float32).pin_memory()
    torch.cuda.synchronize()
    flops = flops_per_call(w)
    K, W = args.steps, args.warmup

    def step_device():
        aj.attn_jvp_fwd(plan, *devin, o, to, lse, stream.cuda_stream)

    def step_host():
        aj.attn_jvp_fwd_host(plan, *host, h_o, h_to, h_lse, stream.cuda_stream)
        stream.synchronize()                  # the user reads the result after every step

    if w.backward:
        # the step is attn_bwd on the forward's O and lse (computed once, outside the timed region); end to end = the
        # six device inputs of attn_bwd copied up from pinned host memory, the call, dQ, dK, dV copied back
        step_device()
        g = torch.Generator().manual_seed(1000 + rank)
        h_bwd = [host[0], host[1], host[2], o.cpu().pin_memory(),
                 torch.randn(host[0].shape, generator=g).to(host[0].dtype).pin_memory()]
        h_lse_in = lse.cpu().pin_memory()
        d_bwd = [x.to(dev) for x in h_bwd]
        dq, dk, dv = torch.empty_like(devin[0]), torch.empty_like(devin[1]), torch.empty_like(devin[1])
        h_grads = [torch.empty_like(host[0]).pin_memory(), torch.empty_like(host[1]).pin_memory(), torch.empty_like(host[1]).pin_memory()]

        def step_device():
            aj.attn_bwd(plan, d_bwd[0], d_bwd[1], d_bwd[2], d_bwd[3], lse, d_bwd[4], dq, dk, dv, stream.cuda_stream)

        def step_host():
            aj.attn_bwd_host(plan, h_bwd[0], h_bwd[1], h_bwd[2], h_bwd[3], h_lse_in, h_bwd[4], *h_grads, stream.cuda_stream)
            stream.synchronize()

    # ---- device-resident timing: events on the launching stream, barrier + synchronize on both sides
    for _ in range(W):
        step_device()
    torch.cuda.synchronize()
    barrier(inited)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if needs_l2_flush(w) else None
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
    ev_b = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
    torch.cuda.synchronize()
    ev[0].record(stream)
    for i in range(K):
        if flush is not None:          # small inputs: evict them from L2, then time this launch alone
            flush.zero_()
        ev_b[i].record(stream)
        step_device()
        ev[i + 1].record(stream)
    torch.cuda.synchronize()
    barrier(inited)
    clocks = sampler.stop() if rank == 0 else None
    per_launch = [ev_b[i].elapsed_time(ev[i + 1]) for i in range(K)]
    total_ms = ev[0].elapsed_time(ev[K]) if flush is None else sum(per_launch)
    del flush

    # ---- energy per launch: board power (nvidia-smi, 100 ms samples) over a loop of at least 2.5 s of back-to-back launches
    energy = None
    if rank == 0 and world == 1 and not args.no_energy:
        n_loop = max(K, int(2.5e3 / max(total_ms / K, 1e-3)) + 1)
        ps = ClockSampler(local)
        ps.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(n_loop):
            step_device()
        e1.record(stream)
        torch.cuda.synchronize()
        pw = ps.stop()
        loop_ms = e0.elapsed_time(e1)
        if pw.get("power_w_loaded"):
            joule = pw["power_w_loaded"] * loop_ms * 1e-3 / n_loop
            energy = {"energy_j_per_launch": joule, "pj_per_counted_flop": joule / flops * 1e12, "mean_board_power_w": pw["power_w_loaded"],
                      "sm_mhz": pw["sm_mhz"], "launches": n_loop, "loop_s": loop_ms * 1e-3, "ms_per_launch": loop_ms / n_loop,
                      "how": "mean of nvidia-smi power.draw samples in the upper half of the power range x loop time / launches"}
    total_ms_all, flops_all = aggregate(total_ms, flops * K, inited, dev)

    # ---- end to end through the C ABI with HOST buffers: H2D of the six inputs + kernel + D2H of O, tO, lse
    for _ in range(min(W, 3)):
        step_host()
    torch.cuda.synchronize()
    barrier(inited)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(K):
        step_host()
    e1.record(stream)
    torch.cuda.synchronize()
    barrier(inited)
    e2e_ms_all, e2e_flops_all = aggregate(e0.elapsed_time(e1), flops * K, inited, dev)
    h2d = sum(x.numel() * x.element_size() for x in host if x is not None)
    d2h = h_o.numel() * h_o.element_size() * (1 if w.no_tangents else 2) + h_lse.numel() * 4
    if w.backward:
        h2d = sum(x.numel() * x.element_size() for x in h_bwd) + h_lse_in.numel() * 4
        d2h = sum(x.numel() * x.element_size() for x in h_grads)
        launches_per_call = 3               # delta, dQ, dK/dV kernels

    # ---- host cost of one enqueue: the time attn_jvp_fwd (attn_bwd) takes to return, median of 1000 calls on a SMALL problem
    # of the same kernel family (so that the device drains faster than the host enqueues and the launch queue never blocks)
    overhead_us = None
    if rank == 0 and w.dtype == "bf16" and w.d == 128:
        sw = Workload("overhead_probe", 1, 2, 128, "teacher_forcing", 128, 2, 1, "bf16", 0.1)
        sp = aj.attn_jvp_plan_create(aj.make_problem(sw.B, sw.H, sw.N, sw.N, sw.d, aj.AJ_BF16),
                                     aj.make_mask(aj.AJ_MASK_TEACHER_FORCING, sw.frame_len, sw.num_frames, 1)[0])
        sx = [t.to(dev) for t in make_inputs(sw)]
        so, sto = torch.empty_like(sx[0]), torch.empty_like(sx[0])
        sl = torch.empty((sw.B, sw.H, sw.N), dtype=torch.float32, device=dev)
        sg = [torch.empty_like(sx[0]) for _ in range(3)]
        aj.attn_jvp_fwd(sp, *sx, so, sto, sl, stream.cuda_stream)
        aj.attn_bwd(sp, sx[0], sx[1], sx[2], so, sl, sx[3], *sg, stream.cuda_stream)
        torch.cuda.synchronize()
        import ctypes
        ts_f, ts_b, ts_c = [], [], []
        for i in range(1000):
            t0 = time.perf_counter_ns()
            aj.attn_jvp_fwd(sp, *sx, so, sto, sl, stream.cuda_stream)
            t1 = time.perf_counter_ns()
            aj.attn_bwd(sp, sx[0], sx[1], sx[2], so, sl, sx[3], *sg, stream.cuda_stream)
            t2 = time.perf_counter_ns()
            ts_f.append((t1 - t0) / 1e3); ts_b.append((t2 - t1) / 1e3)
            if i % 100 == 99:
                torch.cuda.synchronize()
        # the C ABI alone: arguments marshalled once, 1000 calls of the exported function itself
        views = [aj.aj_tensor(t.data_ptr(), t.stride(0), t.stride(1), t.stride(2)) for t in (*sx, so, sto)]
        refs = [ctypes.byref(v) for v in views]
        fn, lse_p, st_p = aj.lib().attn_jvp_fwd, ctypes.c_void_p(sl.data_ptr()), ctypes.c_void_p(stream.cuda_stream)
        for i in range(1000):
            t0 = time.perf_counter_ns()
            fn(sp, *refs, lse_p, st_p)
            ts_c.append((time.perf_counter_ns() - t0) / 1e3)
            if i % 100 == 99:
                torch.cuda.synchronize()
        enc, hits = aj.attn_jvp_plan_tensor_map_stats(sp)
        aj.attn_jvp_plan_destroy(sp)
        overhead_us = {"attn_jvp_fwd_c_abi": statistics.median(ts_c), "attn_jvp_fwd_python_binding": statistics.median(ts_f),
                       "attn_bwd_python_binding": statistics.median(ts_b),
                       "how": "median host time of 1000 calls on a 2-head, 512-token problem of the same kernels: the exported C "
                              "function with arguments marshalled once (ctypes foreign-call cost included), and the Python "
                              "binding (argument checks and marshalling per call)",
                       "tensor_maps_encoded": enc, "tensor_map_cache_hits": hits}

    # ---- parity of what was just timed: the device outputs of head (0, 0) against the oracle rows of the cpu_baseline leg
    parity = None
    cpu_leg = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and not w.backward:
        step_device()
        torch.cuda.synchronize()
        tf, dt, nrows, cores, (rows, ro, rto, rlse) = time_oracle_sample(w, host_all, args.cpu_budget_s)
        cpu_leg = (tf, dt, nrows, cores)
        rsel = torch.from_numpy(rows).to(dev)

        def nerr(got, ref):
            den = float(np.max(np.abs(ref)))
            return float(np.max(np.abs(got.double().cpu().numpy() - ref)) / (den if den > 0 else 1.0))

        parity = {"rows": int(len(rows)), "head": [0, 0], "o": nerr(o[0, 0][rsel], ro), "lse": nerr(lse[0, 0][rsel], rlse),
                  "to": None if w.no_tangents else nerr(to[0, 0][rsel], rto), "metric": "max|gpu - oracle| / max|oracle|",
                  "tolerance": {"o": 1e-2, "to": 1e-2, "lse": 1e-3} if w.dtype == "bf16" else {"o": 1e-4, "to": 1e-4, "lse": 1e-4}}
        parity["ok"] = all(parity[k] is None or parity[k] <= parity["tolerance"][k] for k in ("o", "to", "lse"))
    bwd_leg = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and w.backward:
        # the gradients that were just timed, head (0, 0), against the backward oracle on sampled rows and keys
        step_device()
        torch.cuda.synchronize()
        tf, dt, cores, (rows, keys, rdq, rdk, rdv) = time_oracle_bwd_sample(w, h_bwd[0], h_bwd[1], h_bwd[2], h_bwd[4], args.bwd_parity_samples)
        bwd_leg = (tf, dt, cores, len(rows), len(keys))
        rsel, ksel = torch.from_numpy(rows).to(dev), torch.from_numpy(keys).to(dev)

        def nerr(got, ref):
            den = float(np.max(np.abs(ref)))
            return float(np.max(np.abs(got.double().cpu().numpy() - ref)) / (den if den > 0 else 1.0))

        tol = 1e-2 if w.dtype == "bf16" else 1e-4
        parity = {"rows": int(len(rows)), "keys": int(len(keys)), "head": [0, 0], "dq": nerr(dq[0, 0][rsel], rdq),
                  "dk": nerr(dk[0, 0][ksel], rdk), "dv": nerr(dv[0, 0][ksel], rdv), "metric": "max|gpu - oracle| / max|oracle|",
                  "tolerance": {"dq": tol, "dk": tol, "dv": tol}}
        parity["ok"] = all(parity[k] <= tol for k in ("dq", "dk", "dv"))

    aj.attn_jvp_plan_destroy(plan)
    if rank != 0:
        return
    peaks, peak_src = load_peaks()
    traffic, traffic_src = recorded_traffic(w.name)
    value = flops_all / (total_ms_all * 1e-3) / 1e12
    avg_launch_ms = total_ms / K
    achieved = flops / (avg_launch_ms * 1e-3) / 1e12
    peak = float(peaks.get("bf16_tflops", FALLBACK_PEAKS["bf16_tflops"]))
    sustained = float(peaks.get("bf16_tflops_sustained", FALLBACK_PEAKS["bf16_tflops_sustained"]))
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": total_ms_all / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16" if w.dtype == "bf16" else "f32", "data": "synthetic", "config": workload_config(w),
        "tokens_per_s": world * w.B * w.num_queries / (total_ms_all / K * 1e-3),
        "kernel": {1: "simt_fp32", 2: "tcgen05_umma", 3: "tcgen05_umma_cta_pair", 4: "tcgen05_umma_cta_pair_one_launch"}[kernel], "num_tasks": num_tasks, "plan_create_ms": plan_ms,
        "ms_per_launch": {"mean": avg_launch_ms, "median": statistics.median(per_launch), "min": min(per_launch)},
        "e2e": {"value": e2e_flops_all / (e2e_ms_all * 1e-3) / 1e12, "unit": UNIT, "ms_per_step": e2e_ms_all / K,
                "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "api": ("attn_bwd_host (pinned host buffers, copies inside the timed region)" if w.backward
                        else "attn_jvp_fwd_host (pinned host buffers, copies inside the timed region)")},
        "gpu_launches": K * launches_per_call,
        "clocks": clocks,
        "roofline": {"bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                     "traffic": traffic, "traffic_source": traffic_src, "peak_source": f"{peak_src} bf16_tflops (burst cuBLAS GEMM)",
                     "frac_of_sustained": achieved / sustained, "frac_of_nominal_2250": achieved / 2250.0,
                     "kernel": {1: "attn_jvp_simt_kernel", 2: "attn_jvp_umma_kernel", 4: "attn_jvp_umma_pair_kernel",
                                3: ("attn_fwd_umma_pair_kernel" if w.no_tangents else
                                    "attn_fwd_umma_pair_kernel (primal-only tasks) + attn_jvp_umma_pair_kernel" if w.clean_tangent_zero
                                    else "attn_jvp_umma_pair_kernel")}[kernel],
                     "flops_per_launch": flops},
    }
    if kernel == 1:
        # plain-FMA kernels (fp32 inputs, or bf16 with d = 64): bound by fp32 FMA issue, not by the tensor pipe.  Peak from the
        # unit counts and the maximum SM clock: SMs x 128 fp32 lanes x 2 flop x f.
        props = torch.cuda.get_device_properties(local)
        f_max = (clocks or {}).get("sm_max_mhz") or 1965.0
        alu_peak = props.multi_processor_count * 128 * 2 * f_max * 1e6 / 1e12
        line["roofline"].update(bound="alu", peak=alu_peak, frac=achieved / alu_peak,
                                peak_source=f"derived: {props.multi_processor_count} SMs x 128 fp32 lanes x 2 flop x {f_max:.0f} MHz",
                                note="counted flop are the six length-d contractions only; the kernel also spends FMA issue slots "
                                     "on the softmax and on shared-memory address arithmetic")
        del line["roofline"]["frac_of_sustained"], line["roofline"]["frac_of_nominal_2250"]
    if w.backward:
        # three kernels per step, timed together: delta (HBM-bound, small), the dQ pass and the dK/dV pass of the tcgen05
        # backward kernel (bf16, d = 128).  The 10*d convention counts the minimal five contractions;
        # the two-pass kernel executes seven (S and dP are recomputed in the second pass).
        pair = w.dtype == "bf16" and w.d == 128
        line["kernel"] = ("tcgen05_backward_two_pass_cta_pairs" if pair else
                          "tcgen05_backward_two_pass_single_cta" if kernel == 2 else "simt_fp32_backward")
        line["roofline"].update(kernel=("attn_bwd_dq_pair_kernel (dQ) + attn_bwd_umma_pair_kernel<true> (dK, dV) + attn_bwd_delta_kernel" if pair else
                                        "attn_bwd_umma_kernel<false> (dQ) + attn_bwd_umma_kernel<true> (dK, dV) + attn_bwd_delta_kernel" if kernel == 2
                                        else "attn_bwd_simt_kernel + attn_bwd_delta_kernel"),
                                executed_over_counted_contractions=7.0 / 5.0)
    if w.clean_tangent_zero and not w.no_tangents:     # what the same call would be credited under the dense 12*d convention (speed-up over dense)
        line["equivalent_dense_tflops"] = 12.0 * w.d * w.unmasked_pairs_per_head * w.B * w.H / (avg_launch_ms * 1e-3) / 1e12
    if overhead_us is not None:
        line["launch_overhead_us"] = overhead_us
    if energy is not None:
        line["energy"] = energy
    if parity is not None:
        line["parity"] = parity
    if cpu_leg is not None:                                          # (the timed oracle leg is the forward oracle)
        tf, dt, nrows, cores = cpu_leg
        line["cpu_baseline"] = {"value": tf, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"{nrows} uniformly sampled query rows of head (0,0), all their allowed "
                                          f"keys, {dt:.1f} s", "extrapolated_full_config_s": flops / (tf * 1e12)}
    if bwd_leg is not None:
        tf, dt, cores, nr, nk_s = bwd_leg
        line["cpu_baseline"] = {"value": tf, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"head (0,0): the backward oracle's pass over all {w.num_queries} query rows (lse, delta), dQ of "
                                          f"{nr} sampled rows, dK and dV of {nk_s} sampled keys, {dt:.1f} s",
                                "flop_convention": "2*d per contraction the oracle executed (S and dP per pair of the head; dQ per "
                                                   "sampled row; S, dP, dK, dV per sampled key)",
                                "extrapolated_full_config_s": 14.0 * w.d * w.unmasked_pairs_per_head * w.B * w.H / (tf * 1e12)}
    if parity is not None and not parity["ok"]:
        # a fast wrong kernel must not score: no value, and a failing exit status
        line["value"] = None
        line["invalid"] = "the timed outputs are outside the tolerance against the oracle (see parity)"
        print(json.dumps(line), flush=True)
        raise SystemExit(3)
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------- the Ulysses arm (8(f) N4)
def run_ulysses(args, w: Workload):
    """ONE problem of the workload's shape, sequence-sharded over the ranks: a step = per head group one
    packed all-to-all in, the kernel on the rank's head shard, one packed all-to-all out.  Strong scaling: the whole job's
    FLOPs over the max-over-ranks time.  Also timed in parts (exchange alone with a no-op local op; kernel alone on the
    head shard).  Without CUDA: a dry run of the exchange on gloo with a no-op local op (no throughput is reported)."""
    from paper_2606_25473_b200 import ulysses
    import torch.distributed as dist

    rank, world, local, inited = dist_setup(args.gpus)
    cuda = torch.cuda.is_available()
    if not inited:                                       # world size 1 still goes through the collective
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29531")
        dist.init_process_group("nccl" if cuda else "gloo", rank=0, world_size=1)
    P, G = world, args.head_groups
    if w.H % (P * G) or w.N % P or w.backward or w.Nq:
        raise SystemExit(f"--ulysses needs H = {w.H} divisible by ranks x head groups = {P * G}, N divisible by {P}, a forward workload")
    dev = f"cuda:{local}" if cuda else "cpu"
    if cuda:
        torch.cuda.set_device(local)
    n, hg = w.N // P, w.H // (P * G)
    # this rank's token shard of the SAME global tensors every rank would draw (seeded per tensor and rank: no rank ever
    # materialises the 1.2 GB global problem just to slice it)
    gen = torch.Generator().manual_seed(w.seed * 1000 + rank)
    shard = []
    for i in range(6):
        x = torch.randn((w.B, w.H, n, w.d), generator=gen, dtype=torch.float32)
        if i >= 3:
            x.mul_(w.tangent_std)
        shard.append(x.to(w.torch_dtype).to(dev))
    esz = shard[0].element_size()
    bytes_in = 6 * shard[0].numel() * esz * (P - 1) // P          # what leaves this rank per step and direction
    bytes_out = 2 * shard[0].numel() * esz * (P - 1) // P
    K, W = args.steps, max(args.warmup, 1)

    def noop(g, q, k, v, tq, tk, tv):
        return torch.empty_like(q), torch.empty_like(q), None

    plan = None
    if cuda:
        from paper_2606_25473_b200 import binding as aj
        kind = {"teacher_forcing": aj.AJ_MASK_TEACHER_FORCING, "block_causal": aj.AJ_MASK_BLOCK_CAUSAL, "full": aj.AJ_MASK_FULL}[w.mask]
        tz = aj.AJ_TANGENT_CLEAN_ZERO if w.clean_tangent_zero else aj.AJ_TANGENT_DENSE
        plan = aj.attn_jvp_plan_create(aj.make_problem(w.B, hg, w.N, w.N, w.d, aj.AJ_BF16 if w.dtype == "bf16" else aj.AJ_FP32),
                                       aj.make_mask(kind, w.frame_len, w.num_frames, w.chunk_frames, tangent_zero=tz)[0])
        stream = torch.cuda.current_stream()
        local_op = ulysses.local_attn_jvp(plan, stream.cuda_stream)
    else:
        local_op = noop

    def timed(fn):
        for _ in range(W):
            fn()
        if cuda:
            torch.cuda.synchronize()
        dist.barrier()
        if cuda:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(K):
                fn()
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / K
        else:
            t0 = time.perf_counter()
            for _ in range(K):
                fn()
            ms = 1e3 * (time.perf_counter() - t0) / K
        dist.barrier()
        t = torch.tensor([ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    step_ms = timed(lambda: ulysses.ulysses_attn_jvp(local_op, *shard, head_groups=G, mode=args.exchange))
    comm_ms = timed(lambda: ulysses.ulysses_attn_jvp(noop, *shard, head_groups=G, mode=args.exchange))
    kernel_ms = None
    if cuda:
        hs = [torch.empty((w.B, hg, w.N, w.d), dtype=w.torch_dtype, device=dev).normal_() for _ in range(6)]
        kernel_ms = timed(lambda: [local_op(g, *hs) for g in range(G)])
        aj.attn_jvp_plan_destroy(plan)
    dist.barrier()
    if rank == 0:
        flops = flops_per_call(w)
        peaks, peak_src = load_peaks()
        line = {"metric": METRIC, "value": flops / (step_ms * 1e-3) / 1e12 if cuda else None, "unit": UNIT, "n_gpus": world,
                "steps": K, "warmup": W, "ms_per_step": step_ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                "dtype": "bf16" if w.dtype == "bf16" else "f32", "data": "synthetic", "mode": "ulysses", "exchange": args.exchange,
                "config": dict(workload_config(w), parallelism=f"ulysses cp{P}, {G} head group(s) per rank",
                               tokens_per_rank=n, heads_per_rank=w.H // P),
                "comm_ms": comm_ms, "kernel_ms": kernel_ms, "a2a_bytes_in_per_rank": bytes_in, "a2a_bytes_out_per_rank": bytes_out,
                "overlap": None if kernel_ms is None else {"serial_ms": comm_ms + kernel_ms, "hidden_ms": comm_ms + kernel_ms - step_ms},
                "collectives_per_step": 2 * G, "backend": dist.get_backend(), "dry_run": not cuda,
                "gpu_launches": K * G if cuda else 0}
        if cuda:
            peak = float(peaks.get("bf16_tflops", FALLBACK_PEAKS["bf16_tflops"])) * world
            line["roofline"] = {"bound": "tensor", "achieved": line["value"], "peak": peak, "unit": "TFLOP/s",
                                "frac": line["value"] / peak, "traffic": None, "peak_source": f"{peak_src} bf16_tflops x {world} GPUs",
                                "kernel": "attn_jvp_umma_pair_kernel + " + ("batch_isend_irecv (zero-copy chunks)" if args.exchange == "p2p" else "all_to_all_single (packed)")}
        print(json.dumps(line), flush=True)
    dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=list(WORKLOADS) + list(EXTRA_WORKLOADS))
    ap.add_argument("--cpu-budget-s", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-energy", action="store_true", help="skip the 2.5 s power loop")
    ap.add_argument("--bwd-parity-samples", type=int, default=512, help="backward workloads: query rows / keys of head (0,0) held against the oracle")
    ap.add_argument("--ulysses", action="store_true", help="sequence-sharded ranks with the all-to-all on both sides of the kernel")
    ap.add_argument("--head-groups", type=int, default=2, help="--ulysses: head groups per rank (exchange / kernel pipelining)")
    ap.add_argument("--exchange", default="p2p", choices=["p2p", "packed"],
                    help="--ulysses: zero-copy grouped point-to-point transfers (default) or the packed all_to_all_single")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup
    w = {**WORKLOADS, **EXTRA_WORKLOADS}[args.workload]
    if args.impl == "reference":
        run_reference(args, w)
    elif args.ulysses:
        run_ulysses(args, w)
        return
    else:
        run_cuda(args, w)
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
