"""ctypes binding of libattn_jvp.so: same names as include/attn_jvp.h, argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; nothing here computes.
There is no fallback: if the shared library is missing or a call fails, this raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence, Tuple

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libattn_jvp.so")

AJ_OK, AJ_ERR_INVALID_ARG, AJ_ERR_UNSUPPORTED, AJ_ERR_CUDA, AJ_ERR_OOM = 0, -1, -2, -3, -4
AJ_BF16, AJ_FP32 = 0, 1
AJ_MASK_FULL, AJ_MASK_BLOCK_CAUSAL, AJ_MASK_TEACHER_FORCING, AJ_MASK_RANGES = 0, 1, 2, 3
AJ_KERNEL_AUTO, AJ_KERNEL_SIMT, AJ_KERNEL_UMMA, AJ_KERNEL_UMMA_PAIR, AJ_KERNEL_UMMA_PAIR_ONE = 0, 1, 2, 3, 4
AJ_TILING_PER_GROUP, AJ_TILING_PACKED = 0, 1
AJ_TANGENT_DENSE, AJ_TANGENT_CLEAN_ZERO, AJ_TANGENT_NONE = 0, 1, 2
AJ_TASK_PRIMAL_ONLY = 1
AJ_STATIC_SCRATCH_MAX_ROWS = 1048576
AJ_RENDEZVOUS_AUTO, AJ_RENDEZVOUS_OFF, AJ_RENDEZVOUS_PER_SLOT, AJ_RENDEZVOUS_PER_HEAD = 0, 1, 2, 3

_I32P = ctypes.POINTER(ctypes.c_int32)


class aj_mask_desc(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int32), ("frame_len", ctypes.c_int32), ("num_frames", ctypes.c_int32),
                ("chunk_frames", ctypes.c_int32), ("first_chunk_frames", ctypes.c_int32),
                ("num_groups", ctypes.c_int32), ("tangent_zero", ctypes.c_int32), ("q_begin", _I32P), ("q_end", _I32P),
                ("range_offset", _I32P), ("k_begin", _I32P), ("k_end", _I32P),
                ("q_tangent_zero", _I32P), ("k_tangent_zero", _I32P)]


class aj_problem(ctypes.Structure):
    _fields_ = [("B", ctypes.c_int32), ("H", ctypes.c_int32), ("Nq", ctypes.c_int32), ("Nk", ctypes.c_int32),
                ("d", ctypes.c_int32), ("dtype", ctypes.c_int32), ("scale", ctypes.c_float)]


class aj_tensor(ctypes.Structure):
    _fields_ = [("ptr", ctypes.c_void_p), ("stride_b", ctypes.c_int64), ("stride_h", ctypes.c_int64),
                ("stride_n", ctypes.c_int64)]


class aj_task(ctypes.Structure):
    _fields_ = [("b", ctypes.c_int32), ("h", ctypes.c_int32), ("q_begin", ctypes.c_int32), ("q_rows", ctypes.c_int32),
                ("range_begin", ctypes.c_int32), ("range_count", ctypes.c_int32), ("num_kv_tiles", ctypes.c_int32),
                ("group", ctypes.c_int32), ("flags", ctypes.c_int32)]


class AttnJvpError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"attn_jvp status {status}: {message}")
        self.status = status


# Every symbol include/attn_jvp.h declares (tests check that the library exports all of them).
SYMBOLS = [
    "attn_jvp_schedule_create", "attn_jvp_schedule_create_tiled", "attn_jvp_schedule_entries", "attn_jvp_schedule_destroy", "attn_jvp_schedule_info", "attn_jvp_schedule_get", "attn_jvp_schedule_assign",
    "attn_jvp_schedule_create_transposed", "attn_jvp_schedule_entry_flags", "attn_jvp_schedule_pair_classes", "attn_jvp_plan_pair_classes", "attn_fwd", "attn_bwd",
    "attn_jvp_plan_create", "attn_jvp_plan_destroy", "attn_jvp_plan_info", "attn_jvp_plan_set_kernel", "attn_jvp_plan_set_tiling",
    "attn_jvp_plan_kernel", "attn_jvp_plan_device_status", "attn_jvp_fwd", "attn_jvp_fwd_host", "attn_jvp_last_error", "attn_jvp_version",
    "attn_jvp_fwd_tl", "attn_bwd_host", "attn_jvp_plan_tensor_map_stats", "attn_jvp_schedule_create_transposed_tiled",
    "attn_bwd_static", "attn_jvp_plan_set_rendezvous", "attn_jvp_plan_rendezvous",
    "attn_jvp_plan_set_workers", "attn_jvp_plan_workers",
]

_lib = None


def lib():
    """Loads libattn_jvp.so or raises: there is no non-CUDA path."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_25473_b200.build` "
                              "(or __graft_entry__.build()); this package has no fallback path")
        l = ctypes.CDLL(LIB_PATH)
        vp, i32, i64p = ctypes.c_void_p, ctypes.c_int32, ctypes.POINTER(ctypes.c_int64)
        l.attn_jvp_schedule_create.argtypes = [ctypes.POINTER(aj_problem), ctypes.POINTER(aj_mask_desc), i32, i32, ctypes.POINTER(vp)]
        l.attn_jvp_schedule_create_tiled.argtypes = [ctypes.POINTER(aj_problem), ctypes.POINTER(aj_mask_desc), i32, i32, i32, ctypes.POINTER(vp)]
        l.attn_jvp_schedule_create_transposed.argtypes = [ctypes.POINTER(aj_problem), ctypes.POINTER(aj_mask_desc), i32, i32, ctypes.POINTER(vp)]
        l.attn_jvp_schedule_create_transposed_tiled.argtypes = [ctypes.POINTER(aj_problem), ctypes.POINTER(aj_mask_desc), i32, i32, i32, ctypes.POINTER(vp)]
        l.attn_jvp_schedule_entries.argtypes = [vp, _I32P, _I32P, _I32P, _I32P, _I32P]
        l.attn_jvp_schedule_assign.argtypes = [vp, i32, _I32P, _I32P]
        l.attn_jvp_schedule_entry_flags.argtypes = [vp, _I32P]
        l.attn_jvp_schedule_pair_classes.argtypes = [vp, i64p]
        l.attn_jvp_plan_pair_classes.argtypes = [vp, i64p]
        l.attn_fwd.argtypes = [vp] + [ctypes.POINTER(aj_tensor)] * 4 + [vp, vp]
        l.attn_bwd.argtypes = [vp] + [ctypes.POINTER(aj_tensor)] * 4 + [vp] + [ctypes.POINTER(aj_tensor)] * 4 + [vp]
        l.attn_jvp_schedule_destroy.argtypes = [vp]
        l.attn_jvp_schedule_info.argtypes = [vp, _I32P, _I32P, _I32P, i64p]
        l.attn_jvp_schedule_get.argtypes = [vp, _I32P, _I32P, _I32P, _I32P, _I32P, ctypes.POINTER(aj_task)]
        l.attn_jvp_plan_create.argtypes = [ctypes.POINTER(aj_problem), ctypes.POINTER(aj_mask_desc), ctypes.POINTER(vp)]
        l.attn_jvp_plan_destroy.argtypes = [vp]
        l.attn_jvp_plan_info.argtypes = [vp, i64p, _I32P]
        l.attn_jvp_plan_set_kernel.argtypes = [vp, i32]
        l.attn_jvp_plan_set_tiling.argtypes = [vp, i32]
        l.attn_jvp_plan_kernel.argtypes = [vp, _I32P, _I32P]
        l.attn_jvp_plan_set_rendezvous.argtypes = [vp, i32]
        l.attn_jvp_plan_rendezvous.argtypes = [vp, _I32P]
        l.attn_jvp_plan_set_workers.argtypes = [vp, i32]
        l.attn_jvp_plan_workers.argtypes = [vp, _I32P, _I32P]
        l.attn_jvp_plan_device_status.argtypes = [vp, _I32P]
        l.attn_jvp_fwd.argtypes = [vp] + [ctypes.POINTER(aj_tensor)] * 8 + [vp, vp]
        l.attn_jvp_fwd_host.argtypes = [vp] * 11
        l.attn_jvp_fwd_tl.argtypes = [vp] + [ctypes.POINTER(aj_tensor)] * 8 + [vp, vp, vp]
        l.attn_bwd_host.argtypes = [vp] * 11
        l.attn_jvp_plan_tensor_map_stats.argtypes = [vp, i64p, i64p]
        l.attn_bwd_static.argtypes = ([ctypes.POINTER(aj_problem), ctypes.POINTER(aj_mask_desc)] + [ctypes.POINTER(aj_tensor)] * 4 + [vp] +
                                      [ctypes.POINTER(aj_tensor)] * 4 + [vp])
        for name in SYMBOLS:
            getattr(l, name).restype = ctypes.c_int
        l.attn_jvp_last_error.restype = ctypes.c_char_p
        l.attn_jvp_last_error.argtypes = []
        l.attn_jvp_version.restype = ctypes.c_char_p
        l.attn_jvp_version.argtypes = []
        _lib = l
    return _lib


def _check(status: int):
    if status != AJ_OK:
        raise AttnJvpError(status, lib().attn_jvp_last_error().decode())


def attn_jvp_last_error() -> str:
    return lib().attn_jvp_last_error().decode()


def attn_jvp_version() -> str:
    return lib().attn_jvp_version().decode()


def make_problem(B: int, H: int, Nq: int, Nk: int, d: int, dtype: int, scale: float = 0.0) -> aj_problem:
    return aj_problem(B, H, Nq, Nk, d, dtype, scale)


def make_mask(kind: int, frame_len: int = 0, num_frames: int = 0, chunk_frames: int = 1, first_chunk_frames: int = 0,
              groups: Optional[Sequence[Tuple[int, int, Sequence[Tuple[int, int]]]]] = None,
              tangent_zero: int = AJ_TANGENT_DENSE, q_tangent_zero: Optional[Sequence[int]] = None,
              k_tangent_zero: Optional[Sequence[int]] = None):
    """Returns (aj_mask_desc, keepalive).  `groups` = [(q_begin, q_end, [(k_begin, k_end), ...]), ...] for AJ_MASK_RANGES;
    q_tangent_zero [len(groups)] / k_tangent_zero [total ranges] are its AJ_TANGENT_CLEAN_ZERO flags."""
    m = aj_mask_desc(kind, frame_len, num_frames, chunk_frames, first_chunk_frames, 0, tangent_zero,
                     None, None, None, None, None, None, None)
    keep = []
    if groups is not None:
        ng = len(groups)
        qb = (ctypes.c_int32 * max(ng, 1))(*[g[0] for g in groups])
        qe = (ctypes.c_int32 * max(ng, 1))(*[g[1] for g in groups])
        off, kb, ke = [0], [], []
        for g in groups:
            for (a, b) in g[2]:
                kb.append(a)
                ke.append(b)
            off.append(len(kb))
        offa = (ctypes.c_int32 * len(off))(*off)
        kba = (ctypes.c_int32 * max(len(kb), 1))(*kb)
        kea = (ctypes.c_int32 * max(len(ke), 1))(*ke)
        m.num_groups = ng
        m.q_begin, m.q_end, m.range_offset = qb, qe, offa
        m.k_begin, m.k_end = kba, kea
        keep = [qb, qe, offa, kba, kea]
        if q_tangent_zero is not None:
            qz = (ctypes.c_int32 * max(ng, 1))(*q_tangent_zero)
            m.q_tangent_zero = qz
            keep.append(qz)
        if k_tangent_zero is not None:
            kz = (ctypes.c_int32 * max(len(kb), 1))(*k_tangent_zero)
            m.k_tangent_zero = kz
            keep.append(kz)
    return m, keep


# ---- host-side scheduler -------------------------------------------------------------------------------------------
def attn_jvp_schedule_create(problem: aj_problem, mask: aj_mask_desc, tile_q: int, tile_k: int) -> ctypes.c_void_p:
    out = ctypes.c_void_p()
    _check(lib().attn_jvp_schedule_create(ctypes.byref(problem), ctypes.byref(mask), tile_q, tile_k, ctypes.byref(out)))
    return out


def attn_jvp_schedule_create_tiled(problem: aj_problem, mask: aj_mask_desc, tile_q: int, tile_k: int, tiling: int) -> ctypes.c_void_p:
    out = ctypes.c_void_p()
    _check(lib().attn_jvp_schedule_create_tiled(ctypes.byref(problem), ctypes.byref(mask), tile_q, tile_k, tiling, ctypes.byref(out)))
    return out


def attn_jvp_schedule_create_transposed(problem: aj_problem, mask: aj_mask_desc, tile_keys: int, tile_rows: int) -> ctypes.c_void_p:
    out = ctypes.c_void_p()
    _check(lib().attn_jvp_schedule_create_transposed(ctypes.byref(problem), ctypes.byref(mask), tile_keys, tile_rows, ctypes.byref(out)))
    return out


def attn_jvp_schedule_create_transposed_tiled(problem: aj_problem, mask: aj_mask_desc, tile_keys: int, tile_rows: int, tiling: int) -> ctypes.c_void_p:
    out = ctypes.c_void_p()
    _check(lib().attn_jvp_schedule_create_transposed_tiled(ctypes.byref(problem), ctypes.byref(mask), tile_keys, tile_rows, tiling, ctypes.byref(out)))
    return out


def attn_jvp_schedule_entries(sched):
    """-> dict(k_begin, k_end, row_begin, row_end: lists), the entries aj_task.range_begin / range_count index"""
    n = ctypes.c_int32()
    _check(lib().attn_jvp_schedule_entries(sched, ctypes.byref(n), None, None, None, None))
    arrs = [(ctypes.c_int32 * max(n.value, 1))() for _ in range(4)]
    _check(lib().attn_jvp_schedule_entries(sched, ctypes.byref(n), *arrs))
    return dict(zip(("k_begin", "k_end", "row_begin", "row_end"), (list(a)[:n.value] for a in arrs)))


def attn_jvp_schedule_entry_flags(sched):
    """-> key_tangent_zero per entry (list of 0/1)"""
    n = ctypes.c_int32()
    _check(lib().attn_jvp_schedule_entries(sched, ctypes.byref(n), None, None, None, None))
    arr = (ctypes.c_int32 * max(n.value, 1))()
    _check(lib().attn_jvp_schedule_entry_flags(sched, arr))
    return list(arr)[:n.value]


def attn_jvp_schedule_pair_classes(sched):
    """-> [pairs needing 2, 4, 6 contractions] per head"""
    arr = (ctypes.c_int64 * 3)()
    _check(lib().attn_jvp_schedule_pair_classes(sched, arr))
    return list(arr)


def attn_jvp_schedule_assign(sched, num_workers: int):
    """-> (worker_offset [num_workers + 1], task_ids [num_tasks]) as lists"""
    nt = attn_jvp_schedule_info(sched)[2]
    off = (ctypes.c_int32 * (max(num_workers, 0) + 1))()
    ids = (ctypes.c_int32 * max(nt, 1))()
    _check(lib().attn_jvp_schedule_assign(sched, num_workers, off, ids))
    return list(off), list(ids)[:nt]


def attn_jvp_schedule_destroy(sched) -> None:
    _check(lib().attn_jvp_schedule_destroy(sched))


def attn_jvp_schedule_info(sched):
    """-> (num_groups, num_ranges, num_tasks, unmasked_pairs_per_head)"""
    a, b, c, d = ctypes.c_int32(), ctypes.c_int32(), ctypes.c_int32(), ctypes.c_int64()
    _check(lib().attn_jvp_schedule_info(sched, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c), ctypes.byref(d)))
    return a.value, b.value, c.value, d.value


def attn_jvp_schedule_get(sched):
    """-> dict(q_begin, q_end, range_offset, k_begin, k_end: lists; tasks: list of aj_task)"""
    ng, nr, nt, _ = attn_jvp_schedule_info(sched)
    qb, qe = (ctypes.c_int32 * max(ng, 1))(), (ctypes.c_int32 * max(ng, 1))()
    off = (ctypes.c_int32 * (ng + 1))()
    kb, ke = (ctypes.c_int32 * max(nr, 1))(), (ctypes.c_int32 * max(nr, 1))()
    tasks = (aj_task * max(nt, 1))()
    _check(lib().attn_jvp_schedule_get(sched, qb, qe, off, kb, ke, tasks))
    return dict(q_begin=list(qb)[:ng], q_end=list(qe)[:ng], range_offset=list(off), k_begin=list(kb)[:nr],
                k_end=list(ke)[:nr], tasks=[tasks[i] for i in range(nt)])


# ---- plans and the forward call ------------------------------------------------------------------------------------
_PLANS = {}   # plan handle -> (B, H, Nq, Nk, d, dtype): what the tensors of a call must look like


def attn_jvp_plan_create(problem: aj_problem, mask: aj_mask_desc) -> ctypes.c_void_p:
    out = ctypes.c_void_p()
    _check(lib().attn_jvp_plan_create(ctypes.byref(problem), ctypes.byref(mask), ctypes.byref(out)))
    _PLANS[out.value] = (problem.B, problem.H, problem.Nq, problem.Nk, problem.d, problem.dtype)
    return out


def attn_jvp_plan_destroy(plan) -> None:
    _PLANS.pop(getattr(plan, "value", plan), None)
    _check(lib().attn_jvp_plan_destroy(plan))


def attn_jvp_plan_tensor_map_stats(plan):
    """-> (TMA tensor maps encoded so far, cache hits so far)"""
    a, b = ctypes.c_int64(), ctypes.c_int64()
    _check(lib().attn_jvp_plan_tensor_map_stats(plan, ctypes.byref(a), ctypes.byref(b)))
    return a.value, b.value


def attn_jvp_plan_info(plan):
    """-> (unmasked_pairs_per_head, num_tasks)"""
    a, b = ctypes.c_int64(), ctypes.c_int32()
    _check(lib().attn_jvp_plan_info(plan, ctypes.byref(a), ctypes.byref(b)))
    return a.value, b.value


def attn_jvp_plan_pair_classes(plan):
    """-> [pairs needing 2, 4, 6 contractions] per head"""
    arr = (ctypes.c_int64 * 3)()
    _check(lib().attn_jvp_plan_pair_classes(plan, arr))
    return list(arr)


def attn_jvp_plan_set_kernel(plan, kernel: int) -> None:
    _check(lib().attn_jvp_plan_set_kernel(plan, kernel))


def attn_jvp_plan_set_tiling(plan, tiling: int) -> None:
    _check(lib().attn_jvp_plan_set_tiling(plan, tiling))


def attn_jvp_plan_set_rendezvous(plan, mode: int) -> None:
    _check(lib().attn_jvp_plan_set_rendezvous(plan, mode))


def attn_jvp_plan_rendezvous(plan) -> int:
    """-> the rendezvous mode in effect (AJ_RENDEZVOUS_OFF, PER_SLOT or PER_HEAD)"""
    a = ctypes.c_int32()
    _check(lib().attn_jvp_plan_rendezvous(plan, ctypes.byref(a)))
    return a.value


def attn_jvp_plan_set_workers(plan, num_pairs: int) -> None:
    """Budget of SM pairs for the CTA-pair kernels (0 = all)."""
    _check(lib().attn_jvp_plan_set_workers(plan, num_pairs))


def attn_jvp_plan_workers(plan):
    """-> (CTA pairs of the general kernel, CTA pairs of the forward-only kernel)"""
    a, b = ctypes.c_int32(), ctypes.c_int32()
    _check(lib().attn_jvp_plan_workers(plan, ctypes.byref(a), ctypes.byref(b)))
    return a.value, b.value


def attn_jvp_plan_kernel(plan):
    """-> (kernel, launches_per_call)"""
    a, b = ctypes.c_int32(), ctypes.c_int32()
    _check(lib().attn_jvp_plan_kernel(plan, ctypes.byref(a), ctypes.byref(b)))
    return a.value, b.value


def attn_jvp_plan_device_status(plan) -> int:
    """Synchronises the device; 0 if every launch of the plan completed, else the kernel's abort code."""
    a = ctypes.c_int32()
    _check(lib().attn_jvp_plan_device_status(plan, ctypes.byref(a)))
    return a.value


def _torch_dtype(dtype: int):
    import torch
    return torch.bfloat16 if dtype == AJ_BF16 else torch.float32


def _tensor(t, plan=None, name: str = "tensor", keys: bool = False, cuda: bool = True) -> aj_tensor:
    """torch [B,H,N,d] tensor (d contiguous) -> aj_tensor view, checked against the plan's problem: the kernels index by
    the plan's (B, H, N, d), so a wrong shape, dtype or device must fail here, not fault on the device."""
    if t.dim() != 4 or t.stride(3) != 1:
        raise ValueError(f"{name}: expected a [B, H, N, d] tensor with contiguous d")
    info = _PLANS.get(getattr(plan, "value", plan))
    if info is not None:
        B, H, Nq, Nk, d, dtype = info
        want = (B, H, Nk if keys else Nq, d)
        if tuple(t.shape) != want:
            raise ValueError(f"{name}: shape {tuple(t.shape)} does not match the plan's {want}")
        if t.dtype != _torch_dtype(dtype):
            raise ValueError(f"{name}: dtype {t.dtype} does not match the plan's {_torch_dtype(dtype)}")
        if t.is_cuda != cuda:
            raise ValueError(f"{name}: expected a {'CUDA' if cuda else 'host'} tensor")
    return aj_tensor(t.data_ptr(), t.stride(0), t.stride(1), t.stride(2))


def _rowvec(x, plan, name: str, cuda: bool = True):
    """lse-like argument: contiguous fp32 [B, H, Nq] (or None) -> pointer"""
    if x is None:
        return None
    import torch
    info = _PLANS.get(getattr(plan, "value", plan))
    if x.dtype != torch.float32 or not x.is_contiguous() or x.is_cuda != cuda:
        raise ValueError(f"{name}: expected a contiguous fp32 {'CUDA' if cuda else 'host'} tensor")
    if info is not None and tuple(x.shape) != (info[0], info[1], info[2]):
        raise ValueError(f"{name}: shape {tuple(x.shape)} does not match the plan's {(info[0], info[1], info[2])}")
    return x.data_ptr()


_FWD_NAMES = ("q", "k", "v", "tq", "tk", "tv", "o", "to")
_FWD_KEYS = (False, True, True, False, True, True, False, False)


def attn_jvp_fwd(plan, q, k, v, tq, tk, tv, o, to, lse=None, stream: int = 0, tlse=None) -> None:
    """Device tensors (torch.cuda); enqueues on `stream` (a cudaStream_t handle, 0 = default) and returns.
    tq, tk, tv, to may be None on AJ_TANGENT_NONE plans.  tlse: optional fp32 [B,H,Nq] for the tangent of lse."""
    ts = [None if x is None else _tensor(x, plan, n, kk) for x, n, kk in zip((q, k, v, tq, tk, tv, o, to), _FWD_NAMES, _FWD_KEYS)]
    args = [None if x is None else ctypes.byref(x) for x in ts]
    if tlse is None:
        _check(lib().attn_jvp_fwd(plan, *args, _rowvec(lse, plan, "lse"), stream))
    else:
        _check(lib().attn_jvp_fwd_tl(plan, *args, _rowvec(lse, plan, "lse"), _rowvec(tlse, plan, "tlse"), stream))


def attn_fwd(plan, q, k, v, o, lse=None, stream: int = 0) -> None:
    """Masked attention forward without tangents (AJ_TANGENT_NONE plans): O and lse only."""
    ts = [_tensor(x, plan, n, kk) for x, n, kk in zip((q, k, v, o), ("q", "k", "v", "o"), (False, True, True, False))]
    _check(lib().attn_fwd(plan, *[ctypes.byref(x) for x in ts], _rowvec(lse, plan, "lse"), stream))


_BWD_NAMES = ("q", "k", "v", "o", "dout", "dq", "dk", "dv")
_BWD_KEYS = (False, True, True, False, False, False, True, True)


def attn_bwd(plan, q, k, v, o, lse, dout, dq, dk, dv, stream: int = 0) -> None:
    """Primal backward: device tensors; lse is the forward's fp32 [B,H,Nq]; writes dq, dk, dv."""
    ts = [_tensor(x, plan, n, kk) for x, n, kk in zip((q, k, v, o, dout, dq, dk, dv), _BWD_NAMES, _BWD_KEYS)]
    if lse is None:
        raise ValueError("attn_bwd needs the forward's lse")
    _check(lib().attn_bwd(plan, *[ctypes.byref(x) for x in ts[:4]], _rowvec(lse, plan, "lse"),
                          *[ctypes.byref(x) for x in ts[4:]], stream))


def _host(t, plan, name, keys):
    _tensor(t, plan, name, keys, cuda=False)
    if not t.is_contiguous():
        raise ValueError(f"{name}: the host-buffer calls expect contiguous tensors")
    return t.data_ptr()


def attn_jvp_fwd_host(plan, q, k, v, tq, tk, tv, o, to, lse=None, stream: int = 0) -> None:
    """Host tensors (contiguous [B,H,N,d], ideally pinned); copies + kernel are enqueued on `stream`.
    tq, tk, tv, to may be None on AJ_TANGENT_NONE plans."""
    ptrs = [None if x is None else _host(x, plan, n, kk) for x, n, kk in zip((q, k, v, tq, tk, tv, o, to), _FWD_NAMES, _FWD_KEYS)]
    _check(lib().attn_jvp_fwd_host(plan, *ptrs, _rowvec(lse, plan, "lse", cuda=False), stream))


def attn_bwd_host(plan, q, k, v, o, lse, dout, dq, dk, dv, stream: int = 0) -> None:
    """attn_bwd on host tensors (contiguous, ideally pinned): copies + the three kernels are enqueued on `stream`."""
    ptrs = [_host(x, plan, n, kk) for x, n, kk in zip((q, k, v, o, dout, dq, dk, dv), _BWD_NAMES, _BWD_KEYS)]
    if lse is None:
        raise ValueError("attn_bwd_host needs the forward's lse")
    _check(lib().attn_bwd_host(plan, *ptrs[:4], _rowvec(lse, plan, "lse", cuda=False), *ptrs[4:], stream))


def attn_bwd_static(problem: aj_problem, mask: aj_mask_desc, q, k, v, o, lse, dout, dq, dk, dv, stream: int = 0) -> None:
    """attn_bwd without a plan and without any device allocation, for processes that cannot call cudaMalloc (their own pool
    owns the GPU's memory) or must not (an allocation can stall every stream of the device).  Device tensors as for attn_bwd;
    the mask descriptor is evaluated inside the kernels (FULL, BLOCK_CAUSAL, TEACHER_FORCING).  The per-row scratch is a
    fixed array in the library: B * H * Nq <= AJ_STATIC_SCRATCH_MAX_ROWS, and calls that overlap on the GPU race on it."""
    import torch
    want_q, want_k = (problem.B, problem.H, problem.Nq, problem.d), (problem.B, problem.H, problem.Nk, problem.d)
    ts = []
    for x, n, kk in zip((q, k, v, o, dout, dq, dk, dv), _BWD_NAMES, _BWD_KEYS):
        if tuple(x.shape) != (want_k if kk else want_q) or x.dtype != _torch_dtype(problem.dtype) or not x.is_cuda:
            raise ValueError(f"{n}: expected a CUDA {_torch_dtype(problem.dtype)} tensor of shape {want_k if kk else want_q}")
        ts.append(_tensor(x, None, n, kk))
    if lse is None or lse.dtype != torch.float32 or not lse.is_contiguous() or not lse.is_cuda or tuple(lse.shape) != want_q[:3]:
        raise ValueError("lse: expected the forward's contiguous fp32 CUDA tensor [B, H, Nq]")
    _check(lib().attn_bwd_static(ctypes.byref(problem), ctypes.byref(mask), *[ctypes.byref(x) for x in ts[:4]], lse.data_ptr(),
                                 *[ctypes.byref(x) for x in ts[4:]], stream))
