"""fp64 CPU oracle for masked attention + JVP -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes loader around ``attn_jvp_oracle.c`` (plain C, fp64, OpenMP over query
rows; App. B Eq. 42-44 by definition).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It imports nothing from ``paper_2606_25473_b200`` and
the CUDA path never imports it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "attn_jvp_oracle.c")
_LIB = os.path.join(_HERE, "libattn_jvp_oracle.so")

MASK_FULL, MASK_BLOCK_CAUSAL, MASK_TEACHER_FORCING, MASK_RANGES = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no fast-math: summation order is as written)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _CMask(ctypes.Structure):
    _fields_ = [
        ("kind", ctypes.c_int32),
        ("block_len", ctypes.c_int32),
        ("num_blocks", ctypes.c_int32),
        ("first_block_len", ctypes.c_int32),
        ("num_groups", ctypes.c_int32),
        ("q_begin", ctypes.POINTER(ctypes.c_int32)),
        ("q_end", ctypes.POINTER(ctypes.c_int32)),
        ("range_offset", ctypes.POINTER(ctypes.c_int32)),
        ("k_begin", ctypes.POINTER(ctypes.c_int32)),
        ("k_end", ctypes.POINTER(ctypes.c_int32)),
    ]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.attn_jvp_oracle_allowed.restype = ctypes.c_int
        lib.attn_jvp_oracle_allowed.argtypes = [ctypes.POINTER(_CMask), ctypes.c_int64, ctypes.c_int64]
        lib.attn_jvp_oracle_count_pairs.restype = ctypes.c_int64
        lib.attn_jvp_oracle_count_pairs.argtypes = [ctypes.POINTER(_CMask), ctypes.c_int64, ctypes.c_int64]
        lib.attn_jvp_oracle_rows.restype = ctypes.c_int
        lib.attn_jvp_oracle_rows.argtypes = [
            ctypes.POINTER(_CMask), ctypes.c_int64, ctypes.c_int64, ctypes.c_int32, ctypes.c_double,
            ctypes.c_int32] + [ctypes.c_void_p] * 6 + [
            ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.attn_jvp_oracle_rows_tl.restype = ctypes.c_int
        lib.attn_jvp_oracle_rows_tl.argtypes = lib.attn_jvp_oracle_rows.argtypes + [ctypes.c_void_p]
        lib.attn_jvp_oracle_bwd.restype = ctypes.c_int
        lib.attn_jvp_oracle_bwd.argtypes = [
            ctypes.POINTER(_CMask), ctypes.c_int64, ctypes.c_int64, ctypes.c_int32, ctypes.c_double, ctypes.c_int32] + \
            [ctypes.c_void_p] * 4 + [ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int64] + [ctypes.c_void_p] * 3
        lib.attn_jvp_oracle_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


@dataclass
class Mask:
    """The oracle's own mask description (independent of the CUDA path's descriptor)."""
    kind: int
    block_len: int = 0
    num_blocks: int = 0
    first_block_len: int = 0
    # MASK_RANGES: list of (q_begin, q_end, [(k_begin, k_end), ...])
    groups: Sequence = field(default_factory=list)

    def _c(self):
        keep = []
        m = _CMask(self.kind, self.block_len, self.num_blocks, self.first_block_len, 0,
                   None, None, None, None, None)
        if self.kind == MASK_RANGES:
            qb = np.array([g[0] for g in self.groups], dtype=np.int32)
            qe = np.array([g[1] for g in self.groups], dtype=np.int32)
            off = np.zeros(len(self.groups) + 1, dtype=np.int32)
            kb, ke = [], []
            for i, g in enumerate(self.groups):
                for (a, b) in g[2]:
                    kb.append(a)
                    ke.append(b)
                off[i + 1] = len(kb)
            kb = np.array(kb, dtype=np.int32)
            ke = np.array(ke, dtype=np.int32)
            keep = [qb, qe, off, kb, ke]
            p = lambda a: a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))
            m.num_groups = len(self.groups)
            m.q_begin, m.q_end, m.range_offset, m.k_begin, m.k_end = p(qb), p(qe), p(off), p(kb), p(ke)
        return m, keep


def full_mask() -> Mask:
    return Mask(MASK_FULL)


def block_causal_mask(block_len: int, num_blocks: int, first_block_len: int = 0) -> Mask:
    return Mask(MASK_BLOCK_CAUSAL, block_len, num_blocks, first_block_len)


def teacher_forcing_mask(block_len: int, num_blocks: int, first_block_len: int = 0) -> Mask:
    return Mask(MASK_TEACHER_FORCING, block_len, num_blocks, first_block_len)


def ranges_mask(groups) -> Mask:
    return Mask(MASK_RANGES, groups=list(groups))


def allowed(mask: Mask, a: int, b: int) -> bool:
    cm, keep = mask._c()
    return bool(_load().attn_jvp_oracle_allowed(ctypes.byref(cm), a, b))


def dense_mask(mask: Mask, nq: int, nk: int) -> np.ndarray:
    """Boolean [nq, nk] rasterisation of the predicate (small sizes only)."""
    cm, keep = mask._c()
    lib = _load()
    out = np.zeros((nq, nk), dtype=bool)
    for a in range(nq):
        for b in range(nk):
            out[a, b] = bool(lib.attn_jvp_oracle_allowed(ctypes.byref(cm), a, b))
    return out


def count_pairs(mask: Mask, nq: int, nk: int) -> int:
    cm, keep = mask._c()
    return int(_load().attn_jvp_oracle_count_pairs(ctypes.byref(cm), nq, nk))


def num_threads() -> int:
    return int(_load().attn_jvp_oracle_num_threads())


def attn_jvp_head(mask: Mask, q, k, v, tq, tk, tv, scale: float,
                  rows: Optional[np.ndarray] = None, with_tlse: bool = False):
    """One (batch, head) slice: q, tq [Nq, d]; k, v, tk, tv [Nk, d] (float32 or float64 numpy).

    Returns (o [R, d], to [R, d], lse [R]) in float64 for the R requested rows
    (all rows if ``rows`` is None); with ``with_tlse`` also tlse [R], the tangent of lse
    (sum_b p_ab tS_ab = r / l).
    """
    lib = _load()
    dt = np.float64 if q.dtype == np.float64 else np.float32
    arrs = [np.ascontiguousarray(x, dtype=dt) for x in (q, k, v, tq, tk, tv)]
    nq, d = arrs[0].shape
    nk = arrs[1].shape[0]
    assert arrs[3].shape == (nq, d)
    for x in (arrs[1], arrs[2], arrs[4], arrs[5]):
        assert x.shape == (nk, d)
    if rows is None:
        rows_arr = None
        nrows = nq
    else:
        rows_arr = np.ascontiguousarray(rows, dtype=np.int64)
        nrows = rows_arr.shape[0]
    o = np.empty((nrows, d), dtype=np.float64)
    to = np.empty((nrows, d), dtype=np.float64)
    lse = np.empty((nrows,), dtype=np.float64)
    tlse = np.empty((nrows,), dtype=np.float64) if with_tlse else None
    cm, keep = mask._c()
    rc = lib.attn_jvp_oracle_rows_tl(
        ctypes.byref(cm), nq, nk, d, float(scale), 1 if dt == np.float64 else 0,
        *[x.ctypes.data for x in arrs],
        None if rows_arr is None else rows_arr.ctypes.data, nrows,
        o.ctypes.data, to.ctypes.data, lse.ctypes.data, None if tlse is None else tlse.ctypes.data)
    if rc != 0:
        raise RuntimeError("attn_jvp_oracle_rows failed")
    return (o, to, lse, tlse) if with_tlse else (o, to, lse)


def attn_jvp(mask: Mask, q, k, v, tq, tk, tv, scale: float, rows: Optional[np.ndarray] = None):
    """[B, H, N, d] numpy inputs -> (o [B,H,R,d], to [B,H,R,d], lse [B,H,R]) in float64."""
    B, H = q.shape[:2]
    outs = [[attn_jvp_head(mask, q[b, h], k[b, h], v[b, h], tq[b, h], tk[b, h], tv[b, h], scale, rows)
             for h in range(H)] for b in range(B)]
    o = np.stack([np.stack([outs[b][h][0] for h in range(H)]) for b in range(B)])
    to = np.stack([np.stack([outs[b][h][1] for h in range(H)]) for b in range(B)])
    lse = np.stack([np.stack([outs[b][h][2] for h in range(H)]) for b in range(B)])
    return o, to, lse


def attn_bwd_head(mask: Mask, q, k, v, dout, scale: float, rows: Optional[np.ndarray] = None,
                  keys: Optional[np.ndarray] = None):
    """Primal backward of one (batch, head) slice: q, dout [Nq, d]; k, v [Nk, d] (float32 or float64 numpy).

    Returns (dq [R, d], dk [Kn, d], dv [Kn, d]) in float64 for the requested query rows / keys (all if None).
    """
    lib = _load()
    dt = np.float64 if q.dtype == np.float64 else np.float32
    arrs = [np.ascontiguousarray(x, dtype=dt) for x in (q, k, v, dout)]
    nq, d = arrs[0].shape
    nk = arrs[1].shape[0]
    assert arrs[3].shape == (nq, d) and arrs[2].shape == (nk, d)
    rows_arr = None if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
    keys_arr = None if keys is None else np.ascontiguousarray(keys, dtype=np.int64)
    nrows = nq if rows_arr is None else rows_arr.shape[0]
    nkeys = nk if keys_arr is None else keys_arr.shape[0]
    dq = np.empty((nrows, d), dtype=np.float64)
    dk = np.empty((nkeys, d), dtype=np.float64)
    dv = np.empty((nkeys, d), dtype=np.float64)
    cm, keep = mask._c()
    rc = lib.attn_jvp_oracle_bwd(
        ctypes.byref(cm), nq, nk, d, float(scale), 1 if dt == np.float64 else 0, *[x.ctypes.data for x in arrs],
        None if rows_arr is None else rows_arr.ctypes.data, nrows,
        None if keys_arr is None else keys_arr.ctypes.data, nkeys,
        dq.ctypes.data, dk.ctypes.data, dv.ctypes.data)
    if rc != 0:
        raise RuntimeError("attn_jvp_oracle_bwd failed")
    return dq, dk, dv
