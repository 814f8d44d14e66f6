"""Test-side glue: workload -> oracle mask, input widening, comparison metric."""
import numpy as np
import torch

import oracle
from paper_2606_25473_b200.workloads import Workload


def oracle_mask(w: Workload) -> oracle.Mask:
    if w.mask == "teacher_forcing":
        return oracle.teacher_forcing_mask(w.block_len, w.num_blocks)
    if w.mask == "block_causal":
        return oracle.block_causal_mask(w.block_len, w.num_blocks)
    return oracle.full_mask()


def widen(t: torch.Tensor) -> np.ndarray:
    """bf16/fp32 torch tensor -> float32 numpy (exact)."""
    return t.detach().to("cpu", torch.float32).numpy()


def max_norm_err(got, ref) -> float:
    """max|got-ref| / max|ref| (BASELINE.json north_star metric; R11)."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    denom = np.max(np.abs(ref))
    return float(np.max(np.abs(got - ref)) / (denom if denom > 0 else 1.0))
