"""Host-side logic of the CUDA library, no GPU: library exports, mask lowering, tile tasks, error codes.

The lowered mask (query groups + key ranges) and the task rectangles are rasterised and
compared bit for bit with the oracle's token-by-token predicate (the two share no code).
"""
import ctypes
import os
import re

import numpy as np
import pytest

from helpers import oracle_mask
from paper_2606_25473_b200 import binding as aj
from paper_2606_25473_b200 import build as aj_build
from paper_2606_25473_b200.workloads import WORKLOADS, Workload

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    aj_build.build_library()


def _kind(w: Workload) -> int:
    return {"teacher_forcing": aj.AJ_MASK_TEACHER_FORCING, "block_causal": aj.AJ_MASK_BLOCK_CAUSAL,
            "full": aj.AJ_MASK_FULL}[w.mask]


def _schedule(w: Workload, tile_q: int, tile_k: int):
    prob = aj.make_problem(w.B, w.H, w.N, w.N, w.d, aj.AJ_BF16 if w.dtype == "bf16" else aj.AJ_FP32)
    mask, keep = aj.make_mask(_kind(w), w.frame_len, w.num_frames, w.chunk_frames)
    s = aj.attn_jvp_schedule_create(prob, mask, tile_q, tile_k)
    info = aj.attn_jvp_schedule_info(s)
    got = aj.attn_jvp_schedule_get(s)
    aj.attn_jvp_schedule_destroy(s)
    return info, got


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "attn_jvp.h")).read()
    declared = set(re.findall(r"\b(attn_(?:jvp_)?[a-z_]+)\s*\(", header))
    assert declared == set(aj.SYMBOLS)
    lib = ctypes.CDLL(aj.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), name
    assert "sm_100a" in aj.attn_jvp_version()


def test_struct_layouts_match_header():
    assert ctypes.sizeof(aj.aj_task) == 36
    assert ctypes.sizeof(aj.aj_problem) == 28
    assert ctypes.sizeof(aj.aj_tensor) == 32
    assert ctypes.sizeof(aj.aj_mask_desc) == 32 + 7 * ctypes.sizeof(ctypes.c_void_p)


@pytest.mark.parametrize("mask,L,F,cf", [
    ("teacher_forcing", 16, 3, 1), ("teacher_forcing", 10, 6, 3), ("teacher_forcing", 7, 4, 2),
    ("block_causal", 16, 3, 1), ("block_causal", 9, 6, 2), ("full", 13, 5, 1)])
@pytest.mark.parametrize("tile_q,tile_k", [(16, 32), (8, 4), (128, 64)])
def test_task_rectangles_cover_the_mask_exactly_once(oracle, mask, L, F, cf, tile_q, tile_k):
    w = Workload("t", 1, 1, 64, mask, L, F, cf, "fp32", 1.0)
    (ng, nr, nt, pairs), got = _schedule(w, tile_q, tile_k)
    want = oracle.dense_mask(oracle_mask(w), w.N, w.N)
    cover = np.zeros((w.N, w.N), dtype=np.int32)
    rows_seen = np.zeros(w.N, dtype=np.int32)
    for t in got["tasks"]:
        assert 0 < t.q_rows <= tile_q
        g = t.group
        assert got["q_begin"][g] <= t.q_begin and t.q_begin + t.q_rows <= got["q_end"][g]
        assert (t.q_begin - got["q_begin"][g]) % tile_q == 0          # tiles start at the group start (R8)
        assert (t.range_begin, t.range_begin + t.range_count) == (got["range_offset"][g], got["range_offset"][g + 1])
        tiles = 0
        for r in range(t.range_begin, t.range_begin + t.range_count):
            k0, k1 = got["k_begin"][r], got["k_end"][r]
            cover[t.q_begin:t.q_begin + t.q_rows, k0:k1] += 1
            tiles += -(-(k1 - k0) // tile_k)
        assert tiles == t.num_kv_tiles
        rows_seen[t.q_begin:t.q_begin + t.q_rows] += 1
    assert np.array_equal(cover, want.astype(np.int32))              # every unmasked pair once, no masked pair
    assert np.all(rows_seen == 1)                                    # every output row is written by one task
    assert pairs == int(want.sum()) == w.unmasked_pairs_per_head
    kv = [t.num_kv_tiles for t in got["tasks"]]
    assert kv == sorted(kv, reverse=True)                            # longest first


def test_ranges_are_sorted_disjoint_and_merged():
    w = Workload("t", 1, 1, 64, "teacher_forcing", 8, 4, 1, "fp32", 1.0)
    _, got = _schedule(w, 16, 32)
    off = got["range_offset"]
    for g in range(len(got["q_begin"])):
        rs = [(got["k_begin"][r], got["k_end"][r]) for r in range(off[g], off[g + 1])]
        for (a0, a1), (b0, b1) in zip(rs, rs[1:]):
            assert a1 < b0                                           # touching ranges were merged
    # noisy block 0 sees no clean keys: one range only; clean groups always have exactly one
    n = 4
    assert off[n + 1] - off[n] == 1
    assert all(off[g + 1] - off[g] == 1 for g in range(n))


@pytest.mark.parametrize("name", list(WORKLOADS))
def test_full_size_configs_counts(name):
    w = WORKLOADS[name]
    (ng, nr, nt, pairs), _ = _schedule(w, 128, 64)
    assert pairs == w.unmasked_pairs_per_head
    tiles_per_block = -(-w.block_len // 128)
    groups = {"teacher_forcing": 2 * w.num_blocks, "block_causal": w.num_blocks, "full": 1}[w.mask]
    assert ng == groups
    if w.mask == "full":
        assert nt == w.B * w.H * -(-w.N // 128)
    else:
        assert nt == w.B * w.H * groups * tiles_per_block


def test_generic_ranges_and_uncovered_rows(oracle):
    groups = [(4, 20, [(0, 5), (5, 9), (30, 40)]), (24, 31, [(2, 3)]), (33, 40, [])]
    prob = aj.make_problem(1, 1, 40, 48, 64, aj.AJ_FP32)
    mask, keep = aj.make_mask(aj.AJ_MASK_RANGES, groups=groups)
    s = aj.attn_jvp_schedule_create(prob, mask, 8, 4)
    ng, nr, nt, pairs = aj.attn_jvp_schedule_info(s)
    got = aj.attn_jvp_schedule_get(s)
    aj.attn_jvp_schedule_destroy(s)
    want = oracle.dense_mask(oracle.ranges_mask(groups), 40, 48)
    cover = np.zeros((40, 48), dtype=np.int32)
    rows_seen = np.zeros(40, dtype=np.int32)
    for t in got["tasks"]:
        for r in range(t.range_begin, t.range_begin + t.range_count):
            cover[t.q_begin:t.q_begin + t.q_rows, got["k_begin"][r]:got["k_end"][r]] += 1
        rows_seen[t.q_begin:t.q_begin + t.q_rows] += 1
    assert np.array_equal(cover, want.astype(np.int32))
    assert np.all(rows_seen == 1)          # rows in no group become key-less tasks (O = 0, tO = 0, lse = -inf)
    assert pairs == int(want.sum())
    assert (0, 9) in list(zip(got["k_begin"], got["k_end"]))   # (0,5)+(5,9) merged


def test_first_chunk_frames(oracle):
    prob = aj.make_problem(1, 1, 2 * 7 * 5, 2 * 7 * 5, 64, aj.AJ_FP32)
    mask, keep = aj.make_mask(aj.AJ_MASK_TEACHER_FORCING, 5, 7, 3, first_chunk_frames=1)
    s = aj.attn_jvp_schedule_create(prob, mask, 4, 4)
    got = aj.attn_jvp_schedule_get(s)
    _, _, _, pairs = aj.attn_jvp_schedule_info(s)
    aj.attn_jvp_schedule_destroy(s)
    om = oracle.teacher_forcing_mask(15, 3, first_block_len=5)
    want = oracle.dense_mask(om, 70, 70)
    cover = np.zeros((70, 70), dtype=np.int32)
    for t in got["tasks"]:
        for r in range(t.range_begin, t.range_begin + t.range_count):
            cover[t.q_begin:t.q_begin + t.q_rows, got["k_begin"][r]:got["k_end"][r]] += 1
    assert np.array_equal(cover, want.astype(np.int32))
    assert pairs == int(want.sum())


def _expect(status, fn, *args):
    with pytest.raises(aj.AttnJvpError) as e:
        fn(*args)
    assert e.value.status == status
    assert aj.attn_jvp_last_error() != ""


def test_schedule_error_codes():
    ok_prob = aj.make_problem(1, 1, 96, 96, 64, aj.AJ_FP32)
    tf, _ = aj.make_mask(aj.AJ_MASK_TEACHER_FORCING, 16, 3, 1)
    bad = aj.AJ_ERR_INVALID_ARG
    _expect(bad, aj.attn_jvp_schedule_create, aj.make_problem(1, 1, 95, 96, 64, aj.AJ_FP32), tf, 16, 32)   # Nq mismatch
    _expect(bad, aj.attn_jvp_schedule_create, aj.make_problem(0, 1, 96, 96, 64, aj.AJ_FP32), tf, 16, 32)
    _expect(bad, aj.attn_jvp_schedule_create, aj.make_problem(1, 1, 96, 96, 64, 7), tf, 16, 32)            # dtype
    _expect(bad, aj.attn_jvp_schedule_create, ok_prob, tf, 0, 32)
    m, _ = aj.make_mask(aj.AJ_MASK_TEACHER_FORCING, 16, 3, 2)                                              # 3 % 2
    _expect(bad, aj.attn_jvp_schedule_create, ok_prob, m, 16, 32)
    m, _ = aj.make_mask(9, 16, 3, 1)
    _expect(bad, aj.attn_jvp_schedule_create, ok_prob, m, 16, 32)
    for groups in ([(0, 10, [(0, 4)]), (5, 12, [(0, 4)])],          # overlapping query groups
                   [(0, 10, [(4, 8), (0, 2)])],                     # unsorted ranges
                   [(0, 10, [(0, 5), (4, 8)])],                     # overlapping ranges
                   [(0, 10, [(0, 97)])],                            # outside Nk
                   [(0, 97, [(0, 4)])],                             # outside Nq
                   [(5, 5, [(0, 4)])]):                             # empty group
        m, keep = aj.make_mask(aj.AJ_MASK_RANGES, groups=groups)
        _expect(bad, aj.attn_jvp_schedule_create, ok_prob, m, 16, 32)
    # NULL out pointer / NULL problem go through the raw ABI
    lib = aj.lib()
    assert lib.attn_jvp_schedule_create(None, ctypes.byref(tf), 16, 32, ctypes.byref(ctypes.c_void_p())) == bad
    assert lib.attn_jvp_schedule_create(ctypes.byref(ok_prob), ctypes.byref(tf), 16, 32, None) == bad
    assert lib.attn_jvp_schedule_info(None, None, None, None, None) == bad
    assert lib.attn_jvp_schedule_destroy(None) == aj.AJ_OK


def test_plan_create_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    tf, _ = aj.make_mask(aj.AJ_MASK_TEACHER_FORCING, 16, 3, 1)
    _expect(aj.AJ_ERR_CUDA, aj.attn_jvp_plan_create, aj.make_problem(1, 1, 96, 96, 64, aj.AJ_FP32), tf)
    _expect(aj.AJ_ERR_UNSUPPORTED, aj.attn_jvp_plan_create, aj.make_problem(1, 1, 96, 96, 32, aj.AJ_FP32), tf)


# ---------------------------------------------------------------------------------------------- packed tiling
def _packed(prob, mask, tile_q, tile_k):
    s = aj.attn_jvp_schedule_create_tiled(prob, mask, tile_q, tile_k, aj.AJ_TILING_PACKED)
    info = aj.attn_jvp_schedule_info(s)
    got = aj.attn_jvp_schedule_get(s)
    ent = aj.attn_jvp_schedule_entries(s)
    aj.attn_jvp_schedule_destroy(s)
    return info, got, ent


def _check_packed(want, Nq, info, got, ent, tile_q, tile_k, heads=1):
    """Every unmasked pair is covered by exactly one (entry, row interval) of exactly one task; no masked pair."""
    cover = np.zeros(want.shape, dtype=np.int32)
    rows_seen = np.zeros(Nq, dtype=np.int32)
    for t in got["tasks"]:
        if (t.b, t.h) != (0, 0):
            continue
        assert t.group == -1 and t.q_begin % tile_q == 0 and t.q_rows == min(tile_q, Nq - t.q_begin)
        tiles = 0
        for e in range(t.range_begin, t.range_begin + t.range_count):
            k0, k1, r0, r1 = ent["k_begin"][e], ent["k_end"][e], ent["row_begin"][e], ent["row_end"][e]
            assert 0 <= r0 < r1 <= t.q_rows and k0 < k1
            cover[t.q_begin + r0:t.q_begin + r1, k0:k1] += 1
            tiles += -(-(k1 - k0) // tile_k)
        assert tiles == t.num_kv_tiles
        rows_seen[t.q_begin:t.q_begin + t.q_rows] += 1
    assert np.array_equal(cover, want.astype(np.int32))
    assert np.all(rows_seen == 1)
    assert info[3] == int(want.sum())
    assert len(got["tasks"]) == heads * -(-Nq // tile_q)
    kv = [t.num_kv_tiles for t in got["tasks"]]
    assert kv == sorted(kv, reverse=True)


@pytest.mark.parametrize("mask,L,F,cf", [
    ("teacher_forcing", 16, 3, 1), ("teacher_forcing", 10, 6, 3), ("teacher_forcing", 7, 4, 2),
    ("block_causal", 16, 3, 1), ("block_causal", 9, 6, 2), ("full", 13, 5, 1), ("teacher_forcing", 3, 5, 1)])
@pytest.mark.parametrize("tile_q,tile_k", [(16, 32), (8, 4), (128, 64), (5, 3), (256, 64)])
def test_packed_tiles_cover_the_mask_exactly_once(oracle, mask, L, F, cf, tile_q, tile_k):
    w = Workload("t", 1, 2, 64, mask, L, F, cf, "fp32", 1.0)
    prob = aj.make_problem(w.B, w.H, w.N, w.N, w.d, aj.AJ_FP32)
    kind = {"teacher_forcing": aj.AJ_MASK_TEACHER_FORCING, "block_causal": aj.AJ_MASK_BLOCK_CAUSAL, "full": aj.AJ_MASK_FULL}[mask]
    m, keep = aj.make_mask(kind, L, F, cf)
    info, got, ent = _packed(prob, m, tile_q, tile_k)
    want = oracle.dense_mask(oracle_mask(w), w.N, w.N)
    _check_packed(want, w.N, info, got, ent, tile_q, tile_k, heads=2)


def test_packed_generic_ranges_with_gaps_and_split_row_runs(oracle):
    # groups 0 and 2 share keys (30,40) but group 1 between them does not: rows that see them are not one interval
    groups = [(4, 9, [(0, 5), (5, 9), (30, 40)]), (9, 13, [(2, 3)]), (13, 20, [(30, 40), (44, 48)]), (33, 40, [])]
    prob = aj.make_problem(1, 1, 40, 48, 64, aj.AJ_FP32)
    mask, keep = aj.make_mask(aj.AJ_MASK_RANGES, groups=groups)
    want = oracle.dense_mask(oracle.ranges_mask(groups), 40, 48)
    for tile_q, tile_k in [(8, 4), (16, 8), (64, 64), (3, 5)]:
        info, got, ent = _packed(prob, mask, tile_q, tile_k)
        _check_packed(want, 40, info, got, ent, tile_q, tile_k)


def test_packed_tiling_wastes_fewer_tile_rows_on_config_2():
    w = WORKLOADS["wan13b_tf_framewise"]
    prob = aj.make_problem(1, 1, w.N, w.N, w.d, aj.AJ_BF16)
    m, keep = aj.make_mask(aj.AJ_MASK_TEACHER_FORCING, w.frame_len, w.num_frames, w.chunk_frames)
    per_group = aj.attn_jvp_schedule_create(prob, m, 128, 64)
    pg = aj.attn_jvp_schedule_get(per_group)
    aj.attn_jvp_schedule_destroy(per_group)
    info, got, ent = _packed(prob, m, 128, 64)
    area = lambda tasks: sum(t.num_kv_tiles for t in tasks) * 128 * 64
    eff_pg, eff_pk = w.unmasked_pairs_per_head / area(pg["tasks"]), w.unmasked_pairs_per_head / area(got["tasks"])
    assert 0.93 < eff_pg < 0.94 and eff_pk > 0.975, (eff_pg, eff_pk)
    assert len(got["tasks"]) == 512            # 65520 rows / 128


# ---------------------------------------------------------------------------------------------- CTA-pair kernel schedule
def test_pair_tiling_256_rows_on_config_2_and_worker_assignment():
    """The cta_group::2 kernel's schedule: packed 256-row tiles, tasks assigned head by head to 74 SM pairs."""
    w = WORKLOADS["wan13b_tf_framewise"]
    prob = aj.make_problem(w.B, w.H, w.N, w.N, w.d, aj.AJ_BF16)
    m, keep = aj.make_mask(aj.AJ_MASK_TEACHER_FORCING, w.frame_len, w.num_frames, w.chunk_frames)
    s = aj.attn_jvp_schedule_create_tiled(prob, m, 256, 64, aj.AJ_TILING_PACKED)
    tasks = aj.attn_jvp_schedule_get(s)["tasks"]
    nt = len(tasks)
    assert nt == w.H * 256                       # 65520 rows / 256
    # executed tile area (pair-steps cover two 64-key tiles; an odd tail pays for a masked tile) vs counted pairs
    area = sum(((t.num_kv_tiles + 1) // 2) * 2 for t in tasks) * 256 * 64
    assert w.H * w.unmasked_pairs_per_head / area > 0.965
    workers = 74
    off, ids = aj.attn_jvp_schedule_assign(s, workers)
    aj.attn_jvp_schedule_destroy(s)
    assert off[0] == 0 and off[-1] == nt and sorted(ids) == list(range(nt))      # every task exactly once
    cost = lambda t: (t.num_kv_tiles + 1) // 2 + 1
    loads = [sum(cost(tasks[i]) for i in ids[off[k]:off[k + 1]]) for k in range(workers)]
    assert max(loads) - min(loads) <= max(cost(t) for t in tasks)
    assert max(loads) <= 1.01 * sum(loads) / workers                            # tail under 1 %
    # head-major: the heads a worker visits never go backwards, so all workers stream the same head's K/V together
    for k in range(workers):
        heads = [tasks[i].h for i in ids[off[k]:off[k + 1]]]
        assert heads == sorted(heads)


@pytest.mark.parametrize("workers", [1, 3, 7])
def test_worker_assignment_small_and_errors(workers):
    prob = aj.make_problem(2, 2, 96, 96, 64, aj.AJ_FP32)
    m, keep = aj.make_mask(aj.AJ_MASK_TEACHER_FORCING, 16, 3, 1)
    s = aj.attn_jvp_schedule_create_tiled(prob, m, 16, 8, aj.AJ_TILING_PACKED)
    nt = aj.attn_jvp_schedule_info(s)[2]
    off, ids = aj.attn_jvp_schedule_assign(s, workers)
    assert len(off) == workers + 1 and off[-1] == nt and sorted(ids) == list(range(nt))
    assert aj.lib().attn_jvp_schedule_assign(s, 0, None, None) == aj.AJ_ERR_INVALID_ARG
    assert aj.lib().attn_jvp_schedule_assign(None, 2, None, None) == aj.AJ_ERR_INVALID_ARG
    aj.attn_jvp_schedule_destroy(s)


# ---------------------------------------------------------------------------------------------- structural-zero tangents
def _classes_by_brute_force(want, q_zero, k_zero):
    """Pairs needing 2 / 4 / 6 contractions from the rasterised mask and per-token zero-tangent flags."""
    qz, kz = np.asarray(q_zero, bool)[:, None], np.asarray(k_zero, bool)[None, :]
    return [int((want & qz & kz).sum()), int((want & ~qz & kz).sum()), int((want & ~kz).sum())]


@pytest.mark.parametrize("L,F,cf", [(16, 3, 1), (10, 6, 3), (7, 4, 2), (3, 5, 1)])
@pytest.mark.parametrize("tile_q,tile_k", [(16, 32), (8, 4), (256, 64), (5, 3)])
def test_clean_zero_flags_follow_the_clean_half(oracle, L, F, cf, tile_q, tile_k):
    """AJ_TANGENT_CLEAN_ZERO on a teacher-forcing mask: an entry is flagged iff all its keys are clean, a
    task is primal-only iff all its rows are clean; the mask itself does not change."""
    w = Workload("t", 1, 1, 64, "teacher_forcing", L, F, cf, "fp32", 1.0)
    half = w.N // 2
    prob = aj.make_problem(1, 1, w.N, w.N, w.d, aj.AJ_FP32)
    m, keep = aj.make_mask(aj.AJ_MASK_TEACHER_FORCING, L, F, cf, tangent_zero=aj.AJ_TANGENT_CLEAN_ZERO)
    want = oracle.dense_mask(oracle_mask(w), w.N, w.N)
    clean = np.arange(w.N) < half
    for tiling in (aj.AJ_TILING_PACKED, aj.AJ_TILING_PER_GROUP):
        s = aj.attn_jvp_schedule_create_tiled(prob, m, tile_q, tile_k, tiling)
        info, got, ent = aj.attn_jvp_schedule_info(s), aj.attn_jvp_schedule_get(s), aj.attn_jvp_schedule_entries(s)
        flags, classes = aj.attn_jvp_schedule_entry_flags(s), aj.attn_jvp_schedule_pair_classes(s)
        aj.attn_jvp_schedule_destroy(s)
        if tiling == aj.AJ_TILING_PACKED:
            _check_packed(want, w.N, info, got, ent, tile_q, tile_k)
        assert classes == _classes_by_brute_force(want, clean, clean) and sum(classes) == info[3]
        for t in got["tasks"]:
            all_clean = t.q_begin + t.q_rows <= half
            assert bool(t.flags & aj.AJ_TASK_PRIMAL_ONLY) == all_clean
            for e in range(t.range_begin, t.range_begin + t.range_count):
                assert bool(flags[e]) == (ent["k_end"][e] <= half)     # no entry mixes clean and noisy keys
                assert ent["k_end"][e] <= half or ent["k_begin"][e] >= half


def test_tangent_none_marks_everything_and_dense_marks_nothing():
    for kind, args in [(aj.AJ_MASK_TEACHER_FORCING, (16, 3, 1)), (aj.AJ_MASK_BLOCK_CAUSAL, (16, 6, 2)), (aj.AJ_MASK_FULL, ())]:
        prob = aj.make_problem(1, 2, 96, 96, 64, aj.AJ_FP32)
        for tz, want_flag in [(aj.AJ_TANGENT_NONE, 1), (aj.AJ_TANGENT_DENSE, 0)]:
            m, keep = aj.make_mask(kind, *args, tangent_zero=tz)
            s = aj.attn_jvp_schedule_create_tiled(prob, m, 32, 16, aj.AJ_TILING_PACKED)
            pairs = aj.attn_jvp_schedule_info(s)[3]
            assert all(f == want_flag for f in aj.attn_jvp_schedule_entry_flags(s))
            assert all((t.flags & aj.AJ_TASK_PRIMAL_ONLY) == want_flag for t in aj.attn_jvp_schedule_get(s)["tasks"])
            assert aj.attn_jvp_schedule_pair_classes(s) == ([pairs, 0, 0] if want_flag else [0, 0, pairs])
            aj.attn_jvp_schedule_destroy(s)
    bc, _ = aj.make_mask(aj.AJ_MASK_BLOCK_CAUSAL, 16, 6, 2, tangent_zero=aj.AJ_TANGENT_CLEAN_ZERO)   # no clean half
    _expect(aj.AJ_ERR_INVALID_ARG, aj.attn_jvp_schedule_create, aj.make_problem(1, 1, 96, 96, 64, aj.AJ_FP32), bc, 16, 32)
    bad, _ = aj.make_mask(aj.AJ_MASK_FULL, tangent_zero=5)
    _expect(aj.AJ_ERR_INVALID_ARG, aj.attn_jvp_schedule_create, aj.make_problem(1, 1, 96, 96, 64, aj.AJ_FP32), bad, 16, 32)


def test_ranges_mask_with_per_group_and_per_range_zero_flags(oracle):
    # keys [0, 20) have zero tangents; groups 0 and 1 have zero tQ.  Adjacent ranges with different flags must not merge.
    groups = [(0, 12, [(0, 10), (10, 20)]), (12, 20, [(0, 20), (20, 30)]), (20, 40, [(5, 20), (20, 25), (30, 48)])]
    qz, kz = [1, 1, 0], [1, 1, 1, 0, 1, 0, 0]
    prob = aj.make_problem(1, 1, 40, 48, 64, aj.AJ_FP32)
    m, keep = aj.make_mask(aj.AJ_MASK_RANGES, groups=groups, tangent_zero=aj.AJ_TANGENT_CLEAN_ZERO, q_tangent_zero=qz, k_tangent_zero=kz)
    want = oracle.dense_mask(oracle.ranges_mask(groups), 40, 48)
    q_zero, k_zero = np.arange(40) < 20, np.arange(48) < 20
    for tile_q, tile_k in [(8, 4), (16, 8), (64, 64), (3, 5)]:
        s = aj.attn_jvp_schedule_create_tiled(prob, m, tile_q, tile_k, aj.AJ_TILING_PACKED)
        info, got, ent = aj.attn_jvp_schedule_info(s), aj.attn_jvp_schedule_get(s), aj.attn_jvp_schedule_entries(s)
        flags, classes = aj.attn_jvp_schedule_entry_flags(s), aj.attn_jvp_schedule_pair_classes(s)
        aj.attn_jvp_schedule_destroy(s)
        _check_packed(want, 40, info, got, ent, tile_q, tile_k)
        assert classes == _classes_by_brute_force(want, q_zero, k_zero)
        for t in got["tasks"]:
            es = range(t.range_begin, t.range_begin + t.range_count)
            for e in es:
                assert bool(flags[e]) == (ent["k_end"][e] <= 20)
            assert bool(t.flags & aj.AJ_TASK_PRIMAL_ONLY) == (t.q_begin + t.q_rows <= 20 and all(flags[e] for e in es))
    # the flags are ignored unless the descriptor says CLEAN_ZERO
    m2, keep2 = aj.make_mask(aj.AJ_MASK_RANGES, groups=groups, q_tangent_zero=qz, k_tangent_zero=kz)
    s = aj.attn_jvp_schedule_create_tiled(prob, m2, 8, 4, aj.AJ_TILING_PACKED)
    assert not any(aj.attn_jvp_schedule_entry_flags(s))
    aj.attn_jvp_schedule_destroy(s)


def test_worker_assignment_weights_cheaper_pair_steps_on_config_2_clean_zero():
    w = WORKLOADS["wan13b_tf_framewise"]
    prob = aj.make_problem(w.B, w.H, w.N, w.N, w.d, aj.AJ_BF16)
    m, keep = aj.make_mask(aj.AJ_MASK_TEACHER_FORCING, w.frame_len, w.num_frames, w.chunk_frames, tangent_zero=aj.AJ_TANGENT_CLEAN_ZERO)
    s = aj.attn_jvp_schedule_create_tiled(prob, m, 256, 64, aj.AJ_TILING_PACKED)
    tasks = aj.attn_jvp_schedule_get(s)["tasks"]
    n, C = w.num_blocks, w.block_len
    assert aj.attn_jvp_schedule_pair_classes(s) == [n * (n + 1) // 2 * C * C, n * (n - 1) // 2 * C * C, n * C * C]
    assert sum(1 for t in tasks if t.flags & aj.AJ_TASK_PRIMAL_ONLY) == w.H * (w.N // 2 // 256)    # 127 all-clean tiles per head
    off, ids = aj.attn_jvp_schedule_assign(s, 74)
    aj.attn_jvp_schedule_destroy(s)
    assert sorted(ids) == list(range(len(tasks)))
    # primal-only tasks cost about half a full task per pair-step, so a worker's share of key tiles is no longer equal:
    # workers holding more primal-only tasks stream more tiles
    tiles = [sum(tasks[i].num_kv_tiles for i in ids[off[k]:off[k + 1]]) for k in range(74)]
    primal = [sum(tasks[i].num_kv_tiles for i in ids[off[k]:off[k + 1]] if tasks[i].flags & 1) for k in range(74)]
    assert np.corrcoef(tiles, primal)[0, 1] > 0.5


# ---------------------------------------------------------------------------------------------- transposed (backward) schedule
def _check_transposed(want, prob, mask, tile_keys, tile_rows):
    """Key-tile tasks with row ranges cover the TRANSPOSE of the mask exactly once; every key belongs to one task."""
    s = aj.attn_jvp_schedule_create_transposed(prob, mask, tile_keys, tile_rows)
    ng, nr, nt, pairs = aj.attn_jvp_schedule_info(s)
    got = aj.attn_jvp_schedule_get(s)
    aj.attn_jvp_schedule_destroy(s)
    Nq, Nk = want.shape
    cover = np.zeros((Nk, Nq), dtype=np.int32)
    keys_seen = np.zeros(Nk, dtype=np.int32)
    for t in got["tasks"]:
        if (t.b, t.h) != (0, 0):
            continue
        assert 0 < t.q_rows <= tile_keys
        tiles = 0
        for r in range(t.range_begin, t.range_begin + t.range_count):
            r0, r1 = got["k_begin"][r], got["k_end"][r]
            cover[t.q_begin:t.q_begin + t.q_rows, r0:r1] += 1
            tiles += -(-(r1 - r0) // tile_rows)
        assert tiles == t.num_kv_tiles
        keys_seen[t.q_begin:t.q_begin + t.q_rows] += 1
    assert np.array_equal(cover, want.T.astype(np.int32))
    assert np.all(keys_seen == 1)
    assert pairs == int(want.sum())
    off = got["range_offset"]
    for g in range(ng):                                      # row ranges of a key group: sorted, disjoint, merged
        rs = [(got["k_begin"][r], got["k_end"][r]) for r in range(off[g], off[g + 1])]
        for (a0, a1), (b0, b1) in zip(rs, rs[1:]):
            assert a1 < b0
    return ng


@pytest.mark.parametrize("mask,L,F,cf", [
    ("teacher_forcing", 16, 3, 1), ("teacher_forcing", 10, 6, 3), ("teacher_forcing", 7, 4, 2),
    ("block_causal", 16, 3, 1), ("block_causal", 9, 6, 2), ("full", 13, 5, 1)])
@pytest.mark.parametrize("tile_keys,tile_rows", [(16, 32), (8, 4), (5, 3)])
def test_transposed_schedule_covers_the_transposed_mask_exactly_once(oracle, mask, L, F, cf, tile_keys, tile_rows):
    w = Workload("t", 1, 2, 64, mask, L, F, cf, "fp32", 1.0)
    prob = aj.make_problem(w.B, w.H, w.N, w.N, w.d, aj.AJ_FP32)
    m, keep = aj.make_mask(_kind(w), L, F, cf)
    want = oracle.dense_mask(oracle_mask(w), w.N, w.N)
    ng = _check_transposed(want, prob, m, tile_keys, tile_rows)
    n = w.num_blocks
    # teacher forcing: clean key block j is seen by clean blocks >= j and noisy blocks > j; noisy key block j by itself
    assert ng == {"teacher_forcing": 2 * n, "block_causal": n, "full": 1}[mask]


def test_transposed_schedule_of_generic_ranges_with_unseen_keys(oracle):
    groups = [(4, 9, [(0, 5), (5, 9), (30, 40)]), (9, 13, [(2, 3)]), (13, 20, [(30, 40), (44, 48)]), (33, 40, [])]
    prob = aj.make_problem(1, 1, 40, 48, 64, aj.AJ_FP32)
    mask, keep = aj.make_mask(aj.AJ_MASK_RANGES, groups=groups)
    want = oracle.dense_mask(oracle.ranges_mask(groups), 40, 48)
    for tk, tr in [(8, 4), (16, 8), (3, 5)]:
        _check_transposed(want, prob, mask, tk, tr)


# ---------------------------------------------------------------------------------------------- transposed + packed (CTA-pair backward)
def _transposed_packed(prob, mask, tile_keys, tile_rows):
    s = aj.attn_jvp_schedule_create_transposed_tiled(prob, mask, tile_keys, tile_rows, aj.AJ_TILING_PACKED)
    info = aj.attn_jvp_schedule_info(s)
    got = aj.attn_jvp_schedule_get(s)
    ent = aj.attn_jvp_schedule_entries(s)
    aj.attn_jvp_schedule_destroy(s)
    return info, got, ent


@pytest.mark.parametrize("mask,L,F,cf", [
    ("teacher_forcing", 16, 3, 1), ("teacher_forcing", 10, 6, 3), ("teacher_forcing", 7, 4, 2),
    ("block_causal", 16, 3, 1), ("block_causal", 9, 6, 2), ("full", 13, 5, 1), ("teacher_forcing", 3, 5, 1)])
@pytest.mark.parametrize("tile_keys,tile_rows", [(16, 32), (8, 4), (256, 64), (5, 3)])
def test_transposed_packed_tiles_cover_the_transposed_mask_exactly_once(oracle, mask, L, F, cf, tile_keys, tile_rows):
    # key tiles on a global grid; an entry = query rows [k_begin, k_end) seen by the tile's keys [row_begin, row_end)
    w = Workload("t", 1, 2, 64, mask, L, F, cf, "fp32", 1.0)
    prob = aj.make_problem(w.B, w.H, w.N, w.N, w.d, aj.AJ_FP32)
    m, keep = aj.make_mask(_kind(w), L, F, cf)
    info, got, ent = _transposed_packed(prob, m, tile_keys, tile_rows)
    want = oracle.dense_mask(oracle_mask(w), w.N, w.N)
    _check_packed(want.T, w.N, info, got, ent, tile_keys, tile_rows, heads=2)


def test_transposed_packed_generic_ranges_with_unseen_keys_and_nq_ne_nk(oracle):
    groups = [(4, 9, [(0, 5), (5, 9), (30, 40)]), (9, 13, [(2, 3)]), (13, 20, [(30, 40), (44, 48)]), (33, 40, [])]
    prob = aj.make_problem(1, 1, 40, 48, 64, aj.AJ_FP32)
    mask, keep = aj.make_mask(aj.AJ_MASK_RANGES, groups=groups)
    want = oracle.dense_mask(oracle.ranges_mask(groups), 40, 48)
    for tk, tr in [(8, 4), (16, 8), (64, 64), (3, 5)]:
        info, got, ent = _transposed_packed(prob, mask, tk, tr)
        _check_packed(want.T, 48, info, got, ent, tk, tr)


def test_transposed_packed_ignores_tangent_promises():
    # the backward has no tangents: a CLEAN_ZERO descriptor lowered with the promise stripped flags no task
    w = Workload("t", 1, 1, 128, "teacher_forcing", 300, 3, 1, "bf16", 0.1)
    prob = aj.make_problem(1, 1, w.N, w.N, w.d, aj.AJ_BF16)
    m, keep = aj.make_mask(aj.AJ_MASK_TEACHER_FORCING, w.frame_len, w.num_frames, 1, tangent_zero=aj.AJ_TANGENT_DENSE)
    info, got, ent = _transposed_packed(prob, m, 256, 64)
    assert all(t.flags == 0 for t in got["tasks"])
