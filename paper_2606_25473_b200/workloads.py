"""Seeded synthetic workloads (BASELINE.json `configs`) -- shapes and random draws only.

This module holds NONE of the method's arithmetic: it names the five benchmark
configurations, and draws Q, K, V, tQ, tK, tV from a seeded CPU generator.  Both the
CUDA path's callers (tests, bench.py) and the oracle's callers use it, so the two
sides see bit-identical inputs; neither side's arithmetic lives here.

Recipe: one ``torch.Generator`` (CPU) seeded with
``seed`` draws Q, K, V, tQ, tK, tV in that order as fp32 N(0,1) of shape [B,H,N,d];
the tangents are multiplied by ``tangent_std``; everything is then cast to the config
dtype (round-to-nearest-even).  The oracle receives the cast values widened to fp32.
These tensors stand in for Wan2.1-1.3B activations, which are not
available here.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Dict, List

import torch


@dataclass(frozen=True)
class Workload:
    name: str
    B: int
    H: int
    d: int
    mask: str            # "teacher_forcing" | "block_causal" | "full"
    frame_len: int       # L tokens per latent frame
    num_frames: int      # F latent frames (per half for teacher forcing)
    chunk_frames: int    # frames per block: 1 = frame-wise (c1-1), 3 = chunk-wise (c3-3)
    dtype: str           # "bf16" | "fp32"
    tangent_std: float
    seed: int = 0
    clean_tangent_zero: bool = False   # teacher forcing: tQ, tK, tV rows of the clean half are zero
    no_tangents: bool = False          # plain masked attention forward: tQ = tK = tV = 0 (no JVP at inference)
    Nq: int = 0                        # full mask only: query rows when they differ from the keys (current chunk x cached prefix)
    backward: bool = False             # the step is the primal backward (dQ, dK, dV from dO, O, lse), not the forward

    @property
    def block_len(self) -> int:
        return self.frame_len * self.chunk_frames

    @property
    def num_blocks(self) -> int:
        assert self.num_frames % self.chunk_frames == 0
        return self.num_frames // self.chunk_frames

    @property
    def N(self) -> int:
        half = self.frame_len * self.num_frames
        return 2 * half if self.mask == "teacher_forcing" else half

    @property
    def num_queries(self) -> int:
        return self.Nq or self.N

    @property
    def torch_dtype(self):
        return torch.bfloat16 if self.dtype == "bf16" else torch.float32

    @property
    def unmasked_pairs_per_head(self) -> int:
        """Size of the allowed set, from the shape alone (closed form; P6)."""
        n, C = self.num_blocks, self.block_len
        tri = n * (n + 1) // 2
        if self.mask == "teacher_forcing":
            return 2 * tri * C * C
        if self.mask == "block_causal":
            return tri * C * C
        return self.num_queries * self.N


# BASELINE.json configs[0..4] (+ the full-mask control of configs[4]).
WORKLOADS: Dict[str, Workload] = {w.name: w for w in [
    Workload("tiny_tf_fp32", 1, 2, 64, "teacher_forcing", 16, 3, 1, "fp32", 1.0),
    Workload("wan13b_tf_framewise", 1, 12, 128, "teacher_forcing", 1560, 21, 1, "bf16", 0.1),
    Workload("wan13b_tf_chunkwise", 1, 12, 128, "teacher_forcing", 1560, 21, 3, "bf16", 0.1),
    Workload("block_causal_b2", 2, 12, 128, "block_causal", 1560, 21, 1, "bf16", 0.1),
    Workload("dit_large_tf_chunkwise", 1, 24, 128, "teacher_forcing", 3600, 16, 2, "bf16", 0.1),
    Workload("dit_large_full", 1, 24, 128, "full", 3600, 32, 2, "bf16", 0.1),
]}
CONFIG_ORDER: List[str] = list(WORKLOADS)

# SURVEY.md section 8(f) "next" rows, measured separately from the BASELINE.json configs.
# N1: the real TF-sCM call: "The tangent of the clean context is zero" -> configs[1] with zero clean tangents.
EXTRA_WORKLOADS: Dict[str, Workload] = {w.name: w for w in [
    Workload("wan13b_tf_framewise_cleanzero", 1, 12, 128, "teacher_forcing", 1560, 21, 1, "bf16", 0.1, 0, True),
    Workload("wan13b_tf_chunkwise_cleanzero", 1, 12, 128, "teacher_forcing", 1560, 21, 3, "bf16", 0.1, 0, True),
    # N3: attention without tangents.  The teacher-forcing / diffusion-forcing packed forward of the non-JVP stages
    # (PAPER.md:180), and the rollout shape: one chunk of queries against the cached prefix plus itself.
    Workload("wan13b_tf_framewise_fwd", 1, 12, 128, "teacher_forcing", 1560, 21, 1, "bf16", 0.0, 0, False, True),
    Workload("wan13b_chunk_vs_prefix_fwd", 8, 12, 128, "full", 1560, 21, 1, "bf16", 0.0, 0, False, True, 3 * 1560),
    # ... at the batch size the paper's inference uses (PAPER.md:410 "batch size 1"; :326 one block at a time against the cached
    # prefix): a frame (1560 queries) or a 3-frame chunk (4680) against 21 frames of keys, all 12 heads and one rank's 3 heads
    # behind a P = 4 Ulysses split.  7 / 19 query tiles per head: fewer tasks than SM pairs (no split of a task's key stream yet).
    Workload("wan13b_frame_vs_prefix_fwd_b1", 1, 12, 128, "full", 1560, 21, 1, "bf16", 0.0, 0, False, True, 1560),
    Workload("wan13b_chunk_vs_prefix_fwd_b1", 1, 12, 128, "full", 1560, 21, 1, "bf16", 0.0, 0, False, True, 3 * 1560),
    Workload("wan13b_frame_vs_prefix_fwd_b1_h3", 1, 3, 128, "full", 1560, 21, 1, "bf16", 0.0, 0, False, True, 1560),
    Workload("wan13b_chunk_vs_prefix_fwd_b1_h3", 1, 3, 128, "full", 1560, 21, 1, "bf16", 0.0, 0, False, True, 3 * 1560),
    # N2: the primal backward of configs[1]
    Workload("wan13b_tf_framewise_bwd", 1, 12, 128, "teacher_forcing", 1560, 21, 1, "bf16", 0.1, 0, False, False, 0, True),
    # The plain-FMA (SIMT) correctness paths at a size that gives a throughput figure: fp32 inputs (the 1e-4 path of configs[0])
    # and bf16 with d = 64 (single-CTA tcgen05 kernel).  Same teacher-forcing structure, 2 x 4 frames of 512 tokens.
    Workload("mid_tf_fp32_d64", 1, 4, 64, "teacher_forcing", 512, 4, 1, "fp32", 1.0),
    Workload("mid_tf_bf16_d64", 1, 4, 64, "teacher_forcing", 512, 4, 1, "bf16", 0.1),
    # bf16 with d = 64 on the single-CTA tcgen05 kernel at a size that fills the chip: configs[1]'s mask and length, 24 heads
    Workload("wan13b_tf_framewise_d64", 1, 24, 64, "teacher_forcing", 1560, 21, 1, "bf16", 0.1),
    Workload("wan13b_tf_framewise_d64_bwd", 1, 24, 64, "teacher_forcing", 1560, 21, 1, "bf16", 0.1, 0, False, False, 0, True),
]}


def scaled_down(w: Workload, frame_len: int, num_frames: int = 0, H: int = 0, B: int = 0) -> Workload:
    """Same structure, smaller extent (parity cases the oracle finishes in seconds)."""
    return Workload(f"{w.name}@L{frame_len}", B or w.B, H or w.H, w.d, w.mask, frame_len,
                    num_frames or w.num_frames, w.chunk_frames, w.dtype, w.tangent_std, w.seed, w.clean_tangent_zero,
                    w.no_tangents, 0, w.backward)


def make_inputs(w: Workload, device: str = "cpu", pin: bool = False):
    """Returns [q, k, v, tq, tk, tv]: q, tq [B, H, Nq, d], the rest [B, H, N, d], in the config dtype."""
    g = torch.Generator(device="cpu")
    g.manual_seed(w.seed)
    out = []
    for i in range(6):
        shape = (w.B, w.H, w.num_queries if i in (0, 3) else w.N, w.d)
        x = torch.randn(shape, generator=g, dtype=torch.float32)
        if i >= 3:
            x.mul_(0.0 if w.no_tangents else w.tangent_std)
            if w.clean_tangent_zero:
                assert w.mask == "teacher_forcing"
                x[:, :, :w.N // 2] = 0.0          # the packed sequence is [clean | noisy]
        x = x.to(w.torch_dtype)
        if device != "cpu":
            x = x.to(device)
        elif pin:
            x = x.pin_memory()
        out.append(x)
    return out
