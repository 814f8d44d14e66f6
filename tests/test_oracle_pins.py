"""Pins for the fp64 oracle (`oracle/`), none of which re-type its formula.

P1 central finite differences of O along the tangent   (BASELINE.json north_star: <= 1e-6 at h = 1e-4)
P2 brute-force dense masked attention, numpy matrices, mask built independently from block structure
P3 library autodiff: torch.func.jvp through a 3-line dense attention; SDPA; torch.logsumexp
P4 invariants (zero tangents, full mask, masked keys have no effect)
P5 closed forms
P6 pair counts against closed forms and tests/golden/pair_counts.txt
TL the lse tangent (tlse = r / l): finite differences of lse, torch.func.jvp(logsumexp), closed forms
"""
import os

import numpy as np
import pytest
import torch

from helpers import oracle_mask, widen, max_norm_err
from paper_2606_25473_b200.workloads import WORKLOADS, make_inputs, scaled_down

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rand(shape, seed, std=1.0):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(shape) * std


def _tf_dense_mask(n, C):
    """TF mask from its block picture (BASELINE.json config 1), via Kronecker
    products -- deliberately not the oracle's token-by-token predicate."""
    tril = np.tril(np.ones((n, n), dtype=bool))            # clean i -> clean <= i
    strict = np.tril(np.ones((n, n), dtype=bool), k=-1)    # noisy i -> clean < i
    eye = np.eye(n, dtype=bool)                            # noisy i -> noisy i
    zero = np.zeros((n, n), dtype=bool)
    blocks = np.block([[tril, zero], [strict, eye]])
    return np.kron(blocks, np.ones((C, C), dtype=bool))


def _bc_dense_mask(n, C):
    return np.kron(np.tril(np.ones((n, n), dtype=bool)), np.ones((C, C), dtype=bool))


def _dense_attention_jvp(mask, q, k, v, tq, tk, tv, scale):
    """Brute force with full matrices (one head): additive -inf mask, dense softmax, dense Eq. 44."""
    S = scale * (q @ k.T)
    tS = scale * (tq @ k.T + q @ tk.T)
    S = np.where(mask, S, -np.inf)
    tS = np.where(mask, tS, 0.0)
    m = S.max(axis=1, keepdims=True)
    E = np.exp(S - m)
    Z = E.sum(axis=1, keepdims=True)
    P = E / Z
    O = P @ v
    mu = (P * tS).sum(axis=1, keepdims=True)
    tO = P @ tv + (P * (tS - mu)) @ v
    lse = (m + np.log(Z))[:, 0]
    return O, tO, lse


# ----------------------------------------------------------------------------- P1
@pytest.mark.parametrize("kind", ["teacher_forcing", "block_causal", "full"])
def test_p1_finite_differences(oracle, kind):
    # config-1 shape: H=2, d=64, 3 frames x 16 tokens (96 packed tokens for TF)
    n, C, d = 3, 16, 64
    N = 2 * n * C if kind == "teacher_forcing" else n * C
    mask = {"teacher_forcing": oracle.teacher_forcing_mask(C, n),
            "block_causal": oracle.block_causal_mask(C, n), "full": oracle.full_mask()}[kind]
    x = [_rand((1, 2, N, d), s) for s in range(6)]
    q, k, v, tq, tk, tv = x
    scale = 1.0 / np.sqrt(d)
    _, to, _ = oracle.attn_jvp(mask, q, k, v, tq, tk, tv, scale)
    h = 1e-4
    zero = np.zeros_like(q)
    op, _, lp = oracle.attn_jvp(mask, q + h * tq, k + h * tk, v + h * tv, zero, zero, zero, scale)
    om, _, lm = oracle.attn_jvp(mask, q - h * tq, k - h * tk, v - h * tv, zero, zero, zero, scale)
    fd = (op - om) / (2 * h)
    assert max_norm_err(fd, to) <= 1e-6


# ----------------------------------------------------------------------------- P2
@pytest.mark.parametrize("n,C,d", [(3, 16, 64), (4, 5, 8), (2, 7, 16)])
def test_p2_brute_force_dense_tf(oracle, n, C, d):
    N = 2 * n * C
    q, k, v, tq, tk, tv = [_rand((N, d), 10 + s) for s in range(6)]
    scale = 1.0 / np.sqrt(d)
    dense = _tf_dense_mask(n, C)
    assert np.array_equal(dense, oracle.dense_mask(oracle.teacher_forcing_mask(C, n), N, N))
    O, tO, lse = _dense_attention_jvp(dense, q, k, v, tq, tk, tv, scale)
    o, to, l = oracle.attn_jvp_head(oracle.teacher_forcing_mask(C, n), q, k, v, tq, tk, tv, scale)
    assert np.max(np.abs(o - O)) < 1e-13
    assert np.max(np.abs(to - tO)) < 1e-13
    assert np.max(np.abs(l - lse)) < 1e-13


@pytest.mark.parametrize("n,C,d", [(5, 6, 16)])
def test_p2_brute_force_dense_block_causal_and_ranges(oracle, n, C, d):
    N = n * C
    q, k, v, tq, tk, tv = [_rand((N, d), 20 + s) for s in range(6)]
    scale = 0.37  # scale is a parameter, not only 1/sqrt(d)
    dense = _bc_dense_mask(n, C)
    assert np.array_equal(dense, oracle.dense_mask(oracle.block_causal_mask(C, n), N, N))
    O, tO, lse = _dense_attention_jvp(dense, q, k, v, tq, tk, tv, scale)
    o, to, l = oracle.attn_jvp_head(oracle.block_causal_mask(C, n), q, k, v, tq, tk, tv, scale)
    assert np.max(np.abs(o - O)) < 1e-13 and np.max(np.abs(to - tO)) < 1e-13
    assert np.max(np.abs(l - lse)) < 1e-13
    # the same mask written as the paper's generic range list
    groups = [(i * C, (i + 1) * C, [(0, (i + 1) * C)]) for i in range(n)]
    o2, to2, l2 = oracle.attn_jvp_head(oracle.ranges_mask(groups), q, k, v, tq, tk, tv, scale)
    assert np.array_equal(o, o2) and np.array_equal(to, to2) and np.array_equal(l, l2)


def test_p2_first_block_len(oracle):
    # blocks of length 3, 5, 5 (first_block_len != block_len), TF: dense mask from explicit block ids
    C1, C, n, d = 3, 5, 3, 8
    half = C1 + (n - 1) * C
    blk = np.array([0] * C1 + sum([[i] * C for i in range(1, n)], []))
    N = 2 * half
    dense = np.zeros((N, N), dtype=bool)
    for a in range(N):
        for b in range(N):
            if a < half:
                dense[a, b] = b < half and blk[b] <= blk[a]
            else:
                i = blk[a - half]
                dense[a, b] = (blk[b] < i) if b < half else (blk[b - half] == i)
    m = oracle.teacher_forcing_mask(C, n, first_block_len=C1)
    assert np.array_equal(dense, oracle.dense_mask(m, N, N))
    q, k, v, tq, tk, tv = [_rand((N, d), 30 + s) for s in range(6)]
    O, tO, lse = _dense_attention_jvp(dense, q, k, v, tq, tk, tv, 0.5)
    o, to, l = oracle.attn_jvp_head(m, q, k, v, tq, tk, tv, 0.5)
    assert np.max(np.abs(o - O)) < 1e-13 and np.max(np.abs(to - tO)) < 1e-13


# ----------------------------------------------------------------------------- P3
def test_p3_autodiff_sdpa_logsumexp(oracle):
    w = WORKLOADS["tiny_tf_fp32"]
    q, k, v, tq, tk, tv = [t.double() for t in make_inputs(w)]
    scale = 1.0 / np.sqrt(w.d)
    mask_t = torch.from_numpy(_tf_dense_mask(w.num_blocks, w.block_len))

    def attn(q_, k_, v_):
        s = torch.where(mask_t, (q_ @ k_.transpose(-1, -2)) * scale, torch.tensor(-float("inf"), dtype=q_.dtype))
        return torch.softmax(s, dim=-1) @ v_

    O_ad, tO_ad = torch.func.jvp(attn, (q, k, v), (tq, tk, tv))
    O_sdpa = torch.nn.functional.scaled_dot_product_attention(q, k, v, attn_mask=mask_t, scale=scale)
    s = torch.where(mask_t, (q @ k.transpose(-1, -2)) * scale, torch.tensor(-float("inf"), dtype=q.dtype))
    lse_t = torch.logsumexp(s, dim=-1)
    o, to, lse = oracle.attn_jvp(oracle_mask(w), *[x.numpy() for x in (q, k, v, tq, tk, tv)], scale)
    assert np.max(np.abs(o - O_ad.numpy())) < 1e-13
    assert np.max(np.abs(o - O_sdpa.numpy())) < 1e-13
    assert np.max(np.abs(to - tO_ad.numpy())) < 1e-12
    assert np.max(np.abs(lse - lse_t.numpy())) < 1e-13


# ----------------------------------------------------------------------------- P4
def test_p4_zero_tangents_give_zero(oracle):
    n, C, d = 3, 8, 16
    N = 2 * n * C
    q, k, v = [_rand((N, d), 40 + s) for s in range(3)]
    z = np.zeros((N, d))
    _, to, _ = oracle.attn_jvp_head(oracle.teacher_forcing_mask(C, n), q, k, v, z, z, z, 0.25)
    assert np.all(to == 0.0)


def test_p4_full_mask_is_standard_attention_jvp(oracle):
    N, d = 40, 16
    x = [torch.from_numpy(_rand((N, d), 50 + s)) for s in range(6)]
    f = lambda q_, k_, v_: torch.softmax((q_ @ k_.T) * 0.25, dim=-1) @ v_
    O, tO = torch.func.jvp(f, tuple(x[:3]), tuple(x[3:]))
    o, to, _ = oracle.attn_jvp_head(oracle.full_mask(), *[t.numpy() for t in x], 0.25)
    assert np.max(np.abs(o - O.numpy())) < 1e-13 and np.max(np.abs(to - tO.numpy())) < 1e-13


def test_p4_masked_keys_have_no_effect(oracle):
    n, C, d = 4, 6, 8
    N = 2 * n * C
    m = oracle.teacher_forcing_mask(C, n)
    dense = _tf_dense_mask(n, C)
    q, k, v, tq, tk, tv = [_rand((N, d), 60 + s) for s in range(6)]
    base = oracle.attn_jvp_head(m, q, k, v, tq, tk, tv, 0.3)
    for a in [0, C, n * C - 1, n * C, n * C + C + 1, N - 1]:
        k2, v2, tk2, tv2 = k.copy(), v.copy(), tk.copy(), tv.copy()
        bad = ~dense[a]
        for arr in (k2, v2, tk2, tv2):
            arr[bad] += 1e3 * _rand((int(bad.sum()), d), 99)
        o, to, l = oracle.attn_jvp_head(m, q, k2, v2, tq, tk2, tv2, 0.3, rows=np.array([a]))
        assert np.array_equal(o[0], base[0][a]) and np.array_equal(to[0], base[1][a]) and l[0] == base[2][a]


def test_p4_rows_subset_matches_full(oracle):
    n, C, d = 3, 5, 8
    N = 2 * n * C
    m = oracle.teacher_forcing_mask(C, n)
    x = [_rand((N, d), 70 + s) for s in range(6)]
    full = oracle.attn_jvp_head(m, *x, 0.3)
    rows = np.array([N - 1, 0, 7, 16, 7])
    sub = oracle.attn_jvp_head(m, *x, 0.3, rows=rows)
    for f, s in zip(full, sub):
        assert np.array_equal(f[rows], s)


# ----------------------------------------------------------------------------- P5
def test_p5_single_allowed_key(oracle):
    # TF: clean block 0 with C = 1 sees only key 0; noisy block 0 sees only itself
    n, d = 3, 8
    N = 2 * n
    q, k, v, tq, tk, tv = [_rand((N, d), 80 + s) for s in range(6)]
    o, to, lse = oracle.attn_jvp_head(oracle.teacher_forcing_mask(1, n), q, k, v, tq, tk, tv, 0.7)
    for a, b in [(0, 0), (n, n)]:
        assert np.allclose(o[a], v[b], rtol=0, atol=1e-15)
        assert np.allclose(to[a], tv[b], rtol=0, atol=1e-15)
        assert abs(lse[a] - 0.7 * q[a] @ k[b]) < 1e-14


def test_p5_zero_query_gives_means_and_counts(oracle):
    # Q = tQ = 0 -> P uniform on the allowed set: O = mean V, tO = mean tV, lse = ln(count)
    n, C, d = 4, 3, 8
    N = 2 * n * C
    _, k, v, _, tk, tv = [_rand((N, d), 90 + s) for s in range(6)]
    z = np.zeros((N, d))
    o, to, lse = oracle.attn_jvp_head(oracle.teacher_forcing_mask(C, n), z, k, v, z, tk, tv, 0.3)
    for a in range(N):
        i = (a % (n * C)) // C
        assert abs(lse[a] - np.log((i + 1) * C)) < 1e-13  # allowed-set size (i+1)*C in both halves
        if a < n * C:
            keys = np.arange(0, (i + 1) * C)
        else:
            keys = np.concatenate([np.arange(0, i * C), np.arange(n * C + i * C, n * C + (i + 1) * C)])
        assert np.allclose(o[a], v[keys].mean(0), atol=1e-14)
        assert np.allclose(to[a], tv[keys].mean(0), atol=1e-14)


def test_p5_only_tv_tangent_is_attention_of_tv(oracle):
    n, C, d = 3, 4, 8
    N = 2 * n * C
    m = oracle.teacher_forcing_mask(C, n)
    q, k, v, _, _, tv = [_rand((N, d), 100 + s) for s in range(6)]
    z = np.zeros((N, d))
    _, to, _ = oracle.attn_jvp_head(m, q, k, v, z, z, tv, 0.3)
    o_tv, _, _ = oracle.attn_jvp_head(m, q, k, tv, z, z, z, 0.3)
    assert np.max(np.abs(to - o_tv)) < 1e-14


def test_p5_constant_v_rows_kill_score_tangent_term(oracle):
    n, C, d = 3, 4, 8
    N = 2 * n * C
    q, k, _, tq, tk, _ = [_rand((N, d), 110 + s) for s in range(6)]
    v = np.tile(_rand((1, d), 5), (N, 1))
    _, to, _ = oracle.attn_jvp_head(oracle.teacher_forcing_mask(C, n), q, k, v, tq, tk, np.zeros((N, d)), 0.3)
    assert np.max(np.abs(to)) < 1e-13


def test_p5_common_shift_invariances(oracle):
    # adding one vector u to every tK row shifts tS_ab by s<q_a,u> for all b: the -mu term cancels it
    n, C, d = 3, 4, 8
    N = 2 * n * C
    m = oracle.teacher_forcing_mask(C, n)
    q, k, v, tq, tk, tv = [_rand((N, d), 120 + s) for s in range(6)]
    u = _rand((1, d), 7)
    o0, to0, l0 = oracle.attn_jvp_head(m, q, k, v, tq, tk, tv, 0.3)
    o1, to1, l1 = oracle.attn_jvp_head(m, q, k, v, tq, tk + u, tv, 0.3)
    assert np.max(np.abs(to1 - to0)) < 1e-12 and np.array_equal(o0, o1)
    # adding u to every K row: P, O unchanged; lse moves by s<q_a,u>; tS moves by s<tq_a,u> (cancels)
    o2, to2, l2 = oracle.attn_jvp_head(m, q, k + u, v, tq, tk, tv, 0.3)
    assert np.max(np.abs(o2 - o0)) < 1e-12 and np.max(np.abs(to2 - to0)) < 1e-12
    assert np.max(np.abs((l2 - l0) - 0.3 * (q @ u[0]))) < 1e-12


def test_p5_linearity_in_tangents(oracle):
    n, C, d = 3, 4, 8
    N = 2 * n * C
    m = oracle.teacher_forcing_mask(C, n)
    q, k, v = [_rand((N, d), 130 + s) for s in range(3)]
    t1 = [_rand((N, d), 140 + s) for s in range(3)]
    t2 = [_rand((N, d), 150 + s) for s in range(3)]
    a, b = 0.7, -1.9
    o1, to1, _ = oracle.attn_jvp_head(m, q, k, v, *t1, 0.3)
    o2, to2, _ = oracle.attn_jvp_head(m, q, k, v, *t2, 0.3)
    o3, to3, _ = oracle.attn_jvp_head(m, q, k, v, *[a * x + b * y for x, y in zip(t1, t2)], 0.3)
    assert np.array_equal(o1, o2) and np.array_equal(o1, o3)
    assert np.max(np.abs(to3 - (a * to1 + b * to2))) < 1e-13


def test_p5_scale_enters_both_s_and_ts(oracle):
    # DESIGN.md R1: doubling `scale` equals doubling Q and tQ (both S and tS carry the scale)
    N, d = 24, 8
    q, k, v, tq, tk, tv = [_rand((N, d), 160 + s) for s in range(6)]
    m = oracle.block_causal_mask(6, 4)
    a = oracle.attn_jvp_head(m, q, k, v, tq, tk, tv, 0.6)
    b = oracle.attn_jvp_head(m, 2 * q, k, v, 2 * tq, tk, tv, 0.3)
    for x, y in zip(a, b):
        assert np.max(np.abs(x - y)) < 1e-13


def test_r9_row_without_keys(oracle):
    N, d = 8, 4
    x = [_rand((N, d), 170 + s) for s in range(6)]
    m = oracle.ranges_mask([(0, 4, [(0, 8)])])  # rows 4..7 are in no group
    o, to, lse = oracle.attn_jvp_head(m, *x, 0.5)
    assert np.all(o[4:] == 0) and np.all(to[4:] == 0) and np.all(np.isneginf(lse[4:]))
    assert np.all(np.isfinite(lse[:4]))


def test_float32_inputs_are_widened_exactly(oracle):
    w = scaled_down(WORKLOADS["wan13b_tf_framewise"], 8, 3, H=1)
    x32 = [widen(t)[0, 0] for t in make_inputs(w)]          # bf16 values held in float32
    x64 = [a.astype(np.float64) for a in x32]
    m = oracle_mask(w)
    a = oracle.attn_jvp_head(m, *x32, 0.1)
    b = oracle.attn_jvp_head(m, *x64, 0.1)
    for p, r in zip(a, b):
        assert np.array_equal(p, r)


# ----------------------------------------------------------------------------- TL: the lse tangent
@pytest.mark.parametrize("kind", ["teacher_forcing", "block_causal", "full"])
def test_tl_finite_differences_of_lse(oracle, kind):
    n, C, d = 3, 16, 64
    N = 2 * n * C if kind == "teacher_forcing" else n * C
    mask = {"teacher_forcing": oracle.teacher_forcing_mask(C, n),
            "block_causal": oracle.block_causal_mask(C, n), "full": oracle.full_mask()}[kind]
    q, k, v, tq, tk, tv = [_rand((N, d), 200 + s) for s in range(6)]
    scale = 1.0 / np.sqrt(d)
    o, to, lse, tlse = oracle.attn_jvp_head(mask, q, k, v, tq, tk, tv, scale, with_tlse=True)
    o3, to3, lse3 = oracle.attn_jvp_head(mask, q, k, v, tq, tk, tv, scale)
    assert np.array_equal(o, o3) and np.array_equal(to, to3) and np.array_equal(lse, lse3)
    h = 1e-4
    z = np.zeros_like(q)
    _, _, lp = oracle.attn_jvp_head(mask, q + h * tq, k + h * tk, v, z, z, z, scale)
    _, _, lm = oracle.attn_jvp_head(mask, q - h * tq, k - h * tk, v, z, z, z, scale)
    assert max_norm_err((lp - lm) / (2 * h), tlse) <= 1e-6


def test_tl_autodiff_logsumexp(oracle):
    w = WORKLOADS["tiny_tf_fp32"]
    q, k, v, tq, tk, tv = [t.double() for t in make_inputs(w)]
    scale = 1.0 / np.sqrt(w.d)
    mask_t = torch.from_numpy(_tf_dense_mask(w.num_blocks, w.block_len))

    def lse_fn(q_, k_):
        s = torch.where(mask_t, (q_ @ k_.transpose(-1, -2)) * scale, torch.tensor(-float("inf"), dtype=q_.dtype))
        return torch.logsumexp(s, dim=-1)

    _, tl_ad = torch.func.jvp(lse_fn, (q, k), (tq, tk))
    om = oracle_mask(w)
    for h in range(w.H):
        tl = oracle.attn_jvp_head(om, *[x[0, h].numpy() for x in (q, k, v, tq, tk, tv)], scale, with_tlse=True)[3]
        assert np.max(np.abs(tl - tl_ad[0, h].numpy())) < 1e-13


def test_tl_closed_forms(oracle):
    n, C, d = 3, 4, 8
    N = 2 * n * C
    m = oracle.teacher_forcing_mask(C, n)
    q, k, v, tq, tk, tv = [_rand((N, d), 210 + s) for s in range(6)]
    z = np.zeros((N, d))
    # one allowed key (C = 1): tlse = s (<tq, k> + <q, tk>)
    q1, k1, v1, tq1, tk1, tv1 = [x[:2 * n] for x in (q, k, v, tq, tk, tv)]
    tl = oracle.attn_jvp_head(oracle.teacher_forcing_mask(1, n), q1, k1, v1, tq1, tk1, tv1, 0.7, with_tlse=True)[3]
    for a, b in [(0, 0), (n, n)]:
        assert abs(tl[a] - 0.7 * (tq1[a] @ k1[b] + q1[a] @ tk1[b])) < 1e-14
    # Q = tQ = 0: every tS is zero
    assert np.all(oracle.attn_jvp_head(m, z, k, v, z, tk, tv, 0.3, with_tlse=True)[3] == 0.0)
    # zero tangents: tlse = 0; tV never enters
    assert np.all(oracle.attn_jvp_head(m, q, k, v, z, z, tv, 0.3, with_tlse=True)[3] == 0.0)
    # a common vector u added to every tK row moves every tS_ab of row a by s <q_a, u>, hence tlse by the same
    u = _rand((1, d), 8)
    t0 = oracle.attn_jvp_head(m, q, k, v, tq, tk, tv, 0.3, with_tlse=True)[3]
    t1 = oracle.attn_jvp_head(m, q, k, v, tq, tk + u, tv, 0.3, with_tlse=True)[3]
    assert np.max(np.abs((t1 - t0) - 0.3 * (q @ u[0]))) < 1e-12
    # rows without keys: 0 (R9)
    x = [_rand((8, 4), 220 + s) for s in range(6)]
    tl = oracle.attn_jvp_head(oracle.ranges_mask([(0, 4, [(0, 8)])]), *x, 0.5, with_tlse=True)[3]
    assert np.all(tl[4:] == 0.0) and np.all(tl[:4] != 0.0)
    # Eq. 44 can be written with it: tO = P tV + (P o tS) V - tlse * O
    o, to, lse, tl = oracle.attn_jvp_head(oracle.full_mask(), q, k, v, tq, tk, tv, 0.3, with_tlse=True)
    P = np.exp(0.3 * q @ k.T - lse[:, None])
    tS = 0.3 * (tq @ k.T + q @ tk.T)
    assert np.max(np.abs(to - (P @ tv + (P * tS) @ v - tl[:, None] * o))) < 1e-13


# ----------------------------------------------------------------------------- P6
def test_p6_pair_counts_closed_forms(oracle):
    for n, C in [(3, 16), (4, 5), (7, 3)]:
        tri = n * (n + 1) // 2
        assert oracle.count_pairs(oracle.teacher_forcing_mask(C, n), 2 * n * C, 2 * n * C) == 2 * tri * C * C
        assert oracle.count_pairs(oracle.block_causal_mask(C, n), n * C, n * C) == tri * C * C
        assert oracle.count_pairs(oracle.full_mask(), n * C, n * C) == (n * C) ** 2
        assert int(_tf_dense_mask(n, C).sum()) == 2 * tri * C * C


def test_p6_golden_pair_counts():
    # tests/golden/pair_counts.txt: BASELINE.md section 4 (closed forms of the five configs)
    rows = {}
    with open(os.path.join(GOLDEN, "pair_counts.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, pairs = line.split()
            rows[name] = int(pairs)
    assert set(rows) == set(WORKLOADS)
    for name, w in WORKLOADS.items():
        assert w.unmasked_pairs_per_head == rows[name], name


def test_p6_oracle_counts_match_workload_closed_form_mid_size(oracle):
    w = scaled_down(WORKLOADS["wan13b_tf_chunkwise"], 20, 6)
    assert oracle.count_pairs(oracle_mask(w), w.N, w.N) == w.unmasked_pairs_per_head
