"""Pins for the oracle's primal backward (`oracle.attn_bwd_head`), none of which re-type its formula.

B1 library autodiff: torch.autograd through a 3-line fp64 dense masked attention (mask rasterised independently)
B2 central finite differences of the scalar <O, dO> along random directions of Q, K and V (O from the forward oracle)
B3 invariants: keys no row may see get dK = dV = 0; masked keys' values do not matter; rows with no key get dQ = 0;
   linearity in dO; the row/key subsets select rows of the full result
B4 closed forms: one allowed key (P = 1: dV = sum of dO, dQ = dK = 0); Q = 0 (uniform P: dV_b = mean-weighted dO)
"""
import numpy as np
import pytest
import torch

import oracle
from test_oracle_pins import _bc_dense_mask, _rand, _tf_dense_mask


def _case(kind, seed=0):
    if kind == "teacher_forcing":
        n, C = 3, 5
        return oracle.teacher_forcing_mask(C, n), _tf_dense_mask(n, C), 2 * n * C, 2 * n * C
    if kind == "block_causal":
        n, C = 4, 6
        return oracle.block_causal_mask(C, n), _bc_dense_mask(n, C), n * C, n * C
    if kind == "full":
        return oracle.full_mask(), np.ones((17, 29), dtype=bool), 17, 29
    groups = [(0, 7, [(2, 9), (15, 20)]), (9, 20, [(0, 3), (3, 11), (25, 26)]), (20, 23, [])]
    dense = np.zeros((23, 26), dtype=bool)
    for q0, q1, rs in groups:
        for k0, k1 in rs:
            dense[q0:q1, k0:k1] = True
    return oracle.ranges_mask(groups), dense, 23, 26


KINDS = ["teacher_forcing", "block_causal", "full", "ranges"]


def _inputs(nq, nk, d, seed):
    return _rand((nq, d), seed), _rand((nk, d), seed + 1), _rand((nk, d), seed + 2), _rand((nq, d), seed + 3)


# ----------------------------------------------------------------------------- B1
@pytest.mark.parametrize("kind", KINDS)
def test_backward_matches_torch_autograd(kind):
    om, dense, nq, nk = _case(kind)
    d, scale = 8, 0.37
    q, k, v, dout = _inputs(nq, nk, d, 10)
    tq, tk, tv = [torch.tensor(x, dtype=torch.float64, requires_grad=True) for x in (q, k, v)]
    m = torch.tensor(dense)
    s = torch.where(m, scale * tq @ tk.T, torch.tensor(-float("inf"), dtype=torch.float64))
    p = torch.softmax(s, dim=1)
    p = torch.where(m.any(dim=1, keepdim=True), p, torch.zeros_like(p))      # rows with no key: O = 0 (R9)
    (p @ tv).backward(torch.tensor(dout))
    dq, dk, dv = oracle.attn_bwd_head(om, q, k, v, dout, scale)
    assert np.abs(dq - tq.grad.numpy()).max() < 1e-12
    assert np.abs(dk - tk.grad.numpy()).max() < 1e-12
    assert np.abs(dv - tv.grad.numpy()).max() < 1e-12
    assert np.abs(dk).max() > 1e-3 and np.abs(dq).max() > 1e-3               # not a comparison of zeros


# ----------------------------------------------------------------------------- B2
@pytest.mark.parametrize("kind", KINDS)
def test_backward_matches_finite_differences_of_the_forward_oracle(kind):
    om, dense, nq, nk = _case(kind)
    d, scale, h = 6, 1.0 / np.sqrt(6), 1e-5
    q, k, v, dout = _inputs(nq, nk, d, 20)
    dq, dk, dv = oracle.attn_bwd_head(om, q, k, v, dout, scale)
    z = np.zeros_like

    def loss(q_, k_, v_):
        o, _, _ = oracle.attn_jvp_head(om, q_, k_, v_, z(q_), z(k_), z(v_), scale)
        return float((o * dout).sum())

    for seed in range(3):
        uq, uk, uv = _rand(q.shape, 30 + seed), _rand(k.shape, 40 + seed), _rand(v.shape, 50 + seed)
        fd = (loss(q + h * uq, k + h * uk, v + h * uv) - loss(q - h * uq, k - h * uk, v - h * uv)) / (2 * h)
        an = float((dq * uq).sum() + (dk * uk).sum() + (dv * uv).sum())
        assert abs(fd - an) <= 1e-7 * max(1.0, abs(an)), (fd, an)
    # each input separately, so that a term swapped between dK and dV cannot cancel
    for which, grad in enumerate((dq, dk, dv)):
        u = [z(q), z(k), z(v)]
        u[which] = _rand(grad.shape, 60 + which)
        fd = (loss(q + h * u[0], k + h * u[1], v + h * u[2]) - loss(q - h * u[0], k - h * u[1], v - h * u[2])) / (2 * h)
        an = float((grad * u[which]).sum())
        assert abs(fd - an) <= 1e-7 * max(1.0, abs(an)), (which, fd, an)


# ----------------------------------------------------------------------------- B3
def test_backward_invariants():
    om, dense, nq, nk = _case("ranges")
    d, scale = 8, 0.3
    q, k, v, dout = _inputs(nq, nk, d, 70)
    dq, dk, dv = oracle.attn_bwd_head(om, q, k, v, dout, scale)
    unseen = ~dense.any(axis=0)
    assert unseen.any() and np.all(dk[unseen] == 0) and np.all(dv[unseen] == 0)
    keyless = ~dense.any(axis=1)
    assert keyless.any() and np.all(dq[keyless] == 0)
    # K, V of keys nobody sees do not matter
    k2, v2 = k.copy(), v.copy()
    k2[unseen] = 99.0
    v2[unseen] = -7.0
    dq2, dk2, dv2 = oracle.attn_bwd_head(om, q, k2, v2, dout, scale)
    assert np.array_equal(dq, dq2) and np.array_equal(dk, dk2) and np.array_equal(dv, dv2)
    # dO of rows with no key does not matter
    dout2 = dout.copy()
    dout2[keyless] = 5.0
    for a, b in zip((dq, dk, dv), oracle.attn_bwd_head(om, q, k, v, dout2, scale)):
        assert np.array_equal(a, b)
    # linear in dO
    dout_b = _rand(dout.shape, 71)
    gb = oracle.attn_bwd_head(om, q, k, v, dout_b, scale)
    gc = oracle.attn_bwd_head(om, q, k, v, 2.0 * dout - 3.0 * dout_b, scale)
    for a, b, c in zip((dq, dk, dv), gb, gc):
        assert np.abs(2.0 * a - 3.0 * b - c).max() < 1e-12
    # subsets select rows of the full result
    rows, keys = np.array([19, 0, 5, 21]), np.array([25, 2, 2, 12])
    sq, sk, sv = oracle.attn_bwd_head(om, q, k, v, dout, scale, rows, keys)
    assert np.array_equal(sq, dq[rows]) and np.array_equal(sk, dk[keys]) and np.array_equal(sv, dv[keys])
    # float32 inputs are widened exactly
    f = [x.astype(np.float32) for x in (q, k, v, dout)]
    a32 = oracle.attn_bwd_head(om, *f, scale)
    a64 = oracle.attn_bwd_head(om, *[x.astype(np.float64) for x in f], scale)
    for a, b in zip(a32, a64):
        assert np.array_equal(a, b)


# ----------------------------------------------------------------------------- B4
def test_backward_closed_forms():
    d, scale = 4, 0.5
    # every row sees exactly one key (key 3): P = 1, so dS = 0, dQ = dK = 0 and dV_3 = sum_a dO_a
    groups = [(0, 6, [(3, 4)])]
    q, k, v, dout = _inputs(6, 5, d, 80)
    dq, dk, dv = oracle.attn_bwd_head(oracle.ranges_mask(groups), q, k, v, dout, scale)
    assert np.abs(dq).max() < 1e-15 and np.abs(dk).max() < 1e-15
    assert np.abs(dv[3] - dout.sum(axis=0)).max() < 1e-14 and np.all(dv[[0, 1, 2, 4]] == 0)
    # Q = 0: P uniform over the allowed set; block-causal n = 3, C = 2: row a sees 2 (blk(a) + 1) keys
    om = oracle.block_causal_mask(2, 3)
    q0 = np.zeros((6, d))
    _, k, v, dout = _inputs(6, 6, d, 81)
    dq, dk, dv = oracle.attn_bwd_head(om, q0, k, v, dout, scale)
    cnt = np.array([2, 2, 4, 4, 6, 6], dtype=float)
    want_dv = np.stack([sum(dout[a] / cnt[a] for a in range(6) if a // 2 >= b // 2) for b in range(6)])
    assert np.abs(dv - want_dv).max() < 1e-14
    assert np.abs(dk).max() < 1e-15                       # dK_b = scale sum_a dS_ab q_a with q = 0
    # dQ_a = scale * sum_b p (dP_b - mean dP) k_b = scale * Cov_b(dP_b, k_b) over the allowed set
    for a in range(6):
        nb = int(cnt[a])
        dp = v[:nb] @ dout[a]
        want = scale * ((dp - dp.mean())[:, None] * k[:nb]).mean(axis=0)
        assert np.abs(dq[a] - want).max() < 1e-14
