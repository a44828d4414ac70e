"""Pins of oracle/training.py (f4: teacher / student distributions, DenseKL, SparseKL) against what the
paper and the mathematics fix: closed forms worked by hand, library routines (torch softmax, scipy entropy), special cases
that reduce Eq. 4 to Eq. 3, and brute force for the selected token set."""
import math

import numpy as np
import pytest
import scipy.stats
import torch

from oracle import training as OT


def _rand(seed, L=40, H_q=4, H_kv=2, D=8, H_idx=2, d_idx=8):
    rng = np.random.default_rng(seed)
    Q = rng.standard_normal((L, H_q, D))
    K = rng.standard_normal((L, H_kv, D))
    sq = rng.standard_normal((L, H_idx, d_idx))
    sk = rng.standard_normal((L, H_idx, d_idx))
    w = rng.standard_normal((L, H_idx))          # any sign (R13)
    return Q, K, sq, w, sk


def test_teacher_is_softmax_then_mean_not_mean_then_softmax():
    """Eq. 1 by hand: two heads, two keys, query 1.  Head A logits (0, ln 3) -> (1/4, 3/4); head B (0, 0) -> (1/2, 1/2);
    the teacher is their mean (3/8, 5/8) -- the softmax of the mean logits would be (0.366, 0.634)."""
    D = 2
    K = np.zeros((2, 1, D)); K[1, 0, 0] = 1.0
    Q = np.zeros((2, 2, D)); Q[1, 0, 0] = math.log(3.0)          # head A sees ln 3 on key 1; head B sees zeros
    p = OT.teacher_distribution(Q, K, 1.0)
    assert np.allclose(p[1], [3 / 8, 5 / 8], atol=1e-15)
    assert np.allclose(p[0], [1.0, 0.0])                        # causal: query 0 sees key 0 only
    wrong = np.exp([0.0, math.log(3.0) / 2]); wrong /= wrong.sum()
    assert abs(p[1, 0] - wrong[0]) > 5e-3


def test_teacher_closed_forms_and_library():
    Q, K, *_ = _rand(1)
    p = OT.teacher_distribution(Q, K, 0.35)
    assert np.allclose(p.sum(axis=1), 1.0, atol=1e-14) and np.all(np.triu(p, 1) == 0)
    # identical keys -> uniform over the visible prefix, whatever the queries
    Ku = np.repeat(K[:1], K.shape[0], axis=0)
    pu = OT.teacher_distribution(Q, Ku, 0.35)
    for q in (0, 5, 39):
        assert np.allclose(pu[q, :q + 1], 1.0 / (q + 1), atol=1e-15)
    # library: torch softmax over masked logits, GQA by repeat_interleave, then the head mean
    Qt, Kt = torch.from_numpy(Q), torch.from_numpy(K).repeat_interleave(2, dim=1)
    s = 0.35 * torch.einsum("qhd,thd->hqt", Qt, Kt)
    s = s.masked_fill(torch.triu(torch.ones(40, 40, dtype=torch.bool), 1), float("-inf"))
    assert np.allclose(p, torch.softmax(s, dim=-1).mean(dim=0).numpy(), atol=1e-15)
    # one dominant key per head -> (nearly) one-hot on it
    Kh = np.zeros_like(K); Kh[7] = 50.0 * np.sign(Q[30, ::2, :])
    ph = OT.teacher_distribution(np.abs(Q), np.abs(Kh), 1.0)
    assert ph[30, 7] > 1 - 1e-9
    # teacher_lse of training_reductions = torch.logsumexp
    out = OT.training_reductions(Q, K, 0.35, *_rand(1)[2:], blk=4, k_blocks=3)
    assert np.allclose(out["teacher_lse"], torch.logsumexp(s, dim=-1).numpy().T, atol=1e-13)


def test_student_is_one_softmax_of_the_selector_scores():
    _, _, sq, w, sk = _rand(2)
    s = OT.student_scores(sq, w, sk)
    for q, t in ((0, 0), (9, 3), (39, 39), (17, 0)):
        want = sum(w[q, h] * max(0.0, float(np.dot(sq[q, h], sk[t, h]))) for h in range(sq.shape[1]))
        assert abs(s[q, t] - want) < 1e-13
    assert np.all(np.isneginf(s[np.triu_indices(40, 1)]))
    p = OT.student_distribution(s)
    for q in (0, 11, 39):
        assert np.allclose(p[q, :q + 1], scipy.special.softmax(s[q, :q + 1]), atol=1e-15)


def test_dense_kl_library_and_properties():
    Q, K, sq, w, sk = _rand(3)
    out = OT.training_reductions(Q, K, 0.3, sq, w, sk, blk=4, k_blocks=100)
    for q in (0, 1, 13, 39):
        assert abs(out["dense_kl"][q] - scipy.stats.entropy(out["p_tau"][q, :q + 1], out["p_sigma"][q, :q + 1])) < 1e-13
    assert np.all(out["dense_kl"] >= -1e-15) and out["dense_kl"][0] == 0.0      # one visible key: both are (1)
    assert np.allclose(OT.kl_rows(out["p_tau"], out["p_tau"]), 0.0, atol=1e-15)
    # K >= every block: S_q is everything and Eq. 4 is Eq. 3
    assert np.allclose(out["sparse_kl"], out["dense_kl"], atol=1e-14)


def test_sparse_kl_by_hand():
    """p^tau = (.5, .3, .2), p^sigma = (.6, .3, .1), S = {0, 1}: renormalised (.625, .375) vs (2/3, 1/3), ratios .9375 and
    1.125 -> KL = .625 ln .9375 + .375 ln 1.125."""
    want = 0.625 * math.log(0.9375) + 0.375 * math.log(1.125)
    pt, ps = np.array([[0.5, 0.3, 0.2]]), np.array([[0.6, 0.3, 0.1]])
    m = np.array([True, True, False])
    got = OT.kl_rows((pt[:, m] / pt[:, m].sum()), (ps[:, m] / ps[:, m].sum()))[0]
    assert abs(got - want) < 1e-15 and abs(want - 0.0038319) < 1e-6
    # through sparse_kl: three one-token blocks, student scores ranking token 2 last, K = 2 blocks
    s_s = np.array([[0.0, -np.inf, -np.inf], [0.0, 0.0, -np.inf], [math.log(6.0), math.log(3.0), 0.0]])
    p_sigma = OT.student_distribution(s_s)
    assert np.allclose(p_sigma[2], [0.6, 0.3, 0.1])
    p_tau = np.array([[1.0, 0, 0], [0.5, 0.5, 0], [0.5, 0.3, 0.2]])
    out = OT.sparse_kl(p_tau, p_sigma, s_s, blk=1, k_blocks=2)
    assert abs(out[2] - want) < 1e-15 and out[0] == 0.0


def test_selected_token_set_is_the_top_blocks_by_block_max():
    rng = np.random.default_rng(5)
    for q, blk, k in ((37, 4, 3), (15, 4, 2), (5, 4, 1), (63, 16, 2), (40, 8, 9)):
        s = rng.standard_normal(q + 1)
        n_b = -(-(q + 1) // blk)
        bmax = [s[b * blk:min((b + 1) * blk, q + 1)].max() for b in range(n_b)]
        top = sorted(range(n_b), key=lambda b: (-bmax[b], b))[:k]
        want = np.zeros(q + 1, dtype=bool)
        for b in top:
            want[b * blk:(b + 1) * blk] = True
        assert np.array_equal(OT.selected_tokens(s, q, blk, k), want)
    # reserved blocks count inside K (R10): sink 1 + recency 1 of K = 3 leaves one content block
    s = np.array([0.0, 0, 9, 9, 5, 5, 1, 1, 0, 0])
    assert OT.selected_tokens(s, 9, 2, 3, sink_blocks=1, recency_blocks=1).tolist() == [True, True, True, True, False, False, False, False, True, True]


def test_sparse_kl_is_nonnegative_and_differs_from_dense():
    Q, K, sq, w, sk = _rand(7, L=64)
    out = OT.training_reductions(Q, K, 0.3, sq, w, sk, blk=4, k_blocks=4)
    assert np.all(out["sparse_kl"] >= -1e-15)
    assert np.abs(out["sparse_kl"][32:] - out["dense_kl"][32:]).max() > 1e-3
    assert np.allclose(out["sparse_kl"][:16], out["dense_kl"][:16], atol=1e-14)      # <= 4 blocks visible: all selected


def test_training_row_equals_the_rows_of_the_full_reductions():
    """training_row (the prefix form used for sampled rows of long sequences) against training_reductions, which the tests
    above pin: every row of a short sequence, reserved blocks and ragged last blocks included."""
    Q, K, sq, w, sk = _rand(11, L=53)
    for blk, kb, sink, rec in ((4, 3, 0, 0), (8, 4, 1, 1), (16, 2, 0, 1)):
        full = OT.training_reductions(Q, K, 0.3, sq, w, sk, blk, kb, sink, rec)
        for q in range(53):
            row = OT.training_row(q, Q[q], K[:q + 1], 0.3, sq[q], w[q], sk[:q + 1], blk, kb, sink, rec)
            assert abs(row["dense_kl"] - full["dense_kl"][q]) <= 1e-12
            assert abs(row["sparse_kl"] - full["sparse_kl"][q]) <= 1e-12
            assert np.allclose(row["teacher_lse"], full["teacher_lse"][q], atol=1e-12)
            assert np.allclose(row["s_s"], full["s_s"][q, :q + 1], atol=0, rtol=0)
