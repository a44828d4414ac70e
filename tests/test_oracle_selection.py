"""Pins for oracle/selection.py (steps a1/a2).  None re-types the oracle's formula:
golden vector (tests/golden), invariants the paper states, exhaustive enumeration on tiny
inputs, special cases that reduce to library routines, scalar Python-loop restatements of
PAPER.md:39 / :71 with asymmetric shapes (catch transposed operands / wrong index)."""
import math

import numpy as np
import pytest
from scipy.special import softmax as scipy_softmax

from oracle import selection as S
from oracle import brute


def test_golden_10_blocks(golden):
    g = golden("selection_10blocks.txt")
    scores = np.array([float(x) for x in g["scores"][0]])
    want_probs = {int(t.split(":")[0]): float(t.split(":")[1]) for t in g["probs"][0]}
    want_order = [int(x) for x in g["order"][0]]
    want_cum = [float(x) for x in g["cum"][0]]
    sel = S.select_dual_topp(scores, 0.9, 1, 2, 0)
    for b, pm in want_probs.items():
        assert sel.probs[b] == pytest.approx(pm, abs=1e-6)
    assert sel.probs[[0, 8, 9]].tolist() == [0, 0, 0]
    assert sel.order.tolist() == want_order
    assert np.allclose(sel.cum, want_cum, atol=1.5e-6)
    for case in g["case"]:
        p, kmin = float(case[0]), int(case[1])
        want = [int(x) for x in case[3:]]
        got = S.select_dual_topp(scores, p, 1, 2, kmin)
        assert got.indices.tolist() == want, (p, kmin)
        assert got.budget == len(want)


def _token_scores_loops(q, w, k):
    """PAPER.md:39 written out with scalar loops."""
    L, H, d = len(k), len(q), len(q[0])
    out = []
    for t in range(L):
        s = 0.0
        for h in range(H):
            dot = 0.0
            for i in range(d):
                dot += float(q[h][i]) * float(k[t][h][i])
            s += float(w[h]) * max(0.0, dot)
        out.append(s)
    return np.array(out)


def test_token_scores_and_block_max_against_scalar_loops():
    rng = np.random.default_rng(1)
    L, H, d, blk = 37, 3, 5, 8                       # asymmetric on purpose
    q = rng.standard_normal((H, d))
    w = np.array([0.7, -0.4, 1.3])                   # negative weight (R13)
    k = rng.standard_normal((L, H, d))
    s = S.token_scores(q, w, k)
    assert np.allclose(s, _token_scores_loops(q, w, k), rtol=0, atol=1e-13)
    sb = S.block_max(s, blk)
    assert len(sb) == 5
    for b in range(5):
        assert sb[b] == max(s[b * blk:min((b + 1) * blk, L)])
    # ReLU matters and sits inside the head sum: a key anti-aligned with q scores 0 for that head
    q1 = np.array([[1.0, 0.0]]); k1 = np.array([[[-3.0, 0.0]], [[2.0, 5.0]]])
    assert S.token_scores(q1, np.array([2.0]), k1).tolist() == [0.0, 4.0]


def test_single_head_reduces_to_softmax_of_maxpooled_dots():
    rng = np.random.default_rng(2)
    L, d, blk = 96, 16, 16
    q = np.abs(rng.standard_normal((1, d)))
    k = np.abs(rng.standard_normal((L, 1, d)))       # non-negative dots: ReLU is the identity
    s_bar = S.block_max(S.token_scores(q, np.ones(1), k), blk)
    dots = (k[:, 0, :] @ q[0]).reshape(L // blk, blk).max(axis=1)
    assert np.allclose(s_bar, dots, atol=1e-13)
    p = S.residual_distribution(s_bar, 0, 0)
    assert np.allclose(p, scipy_softmax(dots), atol=1e-14)
    assert abs(p.sum() - 1) < 1e-12
    # temperature
    assert np.allclose(S.residual_distribution(s_bar, 0, 0, 2.0), scipy_softmax(dots / 2.0), atol=1e-14)


def _check_invariants(z, p, sink, rec, kmin):
    n_b = len(z)
    sel = S.select_dual_topp(z, p, sink, rec, kmin)
    idx = sel.indices
    res = np.ones(n_b, bool); res[:min(sink, n_b)] = False; res[max(0, n_b - rec):] = False
    reserved = set(np.nonzero(~res)[0].tolist())
    chosen = set(idx.tolist())
    assert reserved <= chosen                                          # S_sink U S_rec in S_q
    assert np.all(np.diff(idx) > 0) and (len(idx) == 0 or (idx[0] >= 0 and idx[-1] < n_b))
    assert sel.budget == len(idx) >= min(kmin, n_b)                    # Eq. 8 floor
    if res.any():
        assert abs(sel.probs[res].sum() - 1.0) < 1e-12                 # Eq. 7 sums to 1 on B_res
        assert np.all(sel.probs[~res] == 0)
        nuc = sel.order[:sel.n_star]
        mass = sel.probs[nuc].sum()
        if p < 1:
            assert mass >= p - 1e-12                                   # reaches p
            if sel.n_star > 0:
                assert sel.probs[nuc[:-1]].sum() < p                   # minimal
        else:
            assert sel.n_star == res.sum()
        # nucleus members all score >= non-members
        rest = [b for b in np.nonzero(res)[0] if b not in set(nuc.tolist())]
        if len(nuc) and rest:
            assert z[nuc].min() >= z[rest].max()
    else:
        assert chosen == set(range(n_b))
    return sel


def test_invariants_random_and_monotone_in_p():
    rng = np.random.default_rng(3)
    for trial in range(300):
        n_b = int(rng.integers(1, 40))
        z = rng.standard_normal(n_b) * rng.uniform(0.1, 6)
        if trial % 5 == 0:
            z = np.round(z)                                            # exact ties
        sink, rec, kmin = int(rng.integers(0, 4)), int(rng.integers(0, 4)), int(rng.integers(0, 12))
        prev = -1
        for p in (0.05, 0.5, 0.7, 0.8, 0.9, 0.95, 0.999, 1.0):
            sel = _check_invariants(z, p, sink, rec, kmin)
            assert sel.budget >= prev                                  # budget monotone in p
            prev = sel.budget


def test_nucleus_against_exhaustive_enumeration():
    rng = np.random.default_rng(4)
    for trial in range(60):
        n_b = int(rng.integers(3, 13))
        z = rng.standard_normal(n_b) * 2
        sink, rec = int(rng.integers(0, 2)), int(rng.integers(0, 3))
        p = float(rng.choice([0.3, 0.5, 0.7, 0.9, 0.97]))
        sel = S.select_dual_topp(z, p, sink, rec, 0)
        res = [b for b in range(n_b) if sel.probs[b] > 0 or (b >= sink and b < n_b - rec)]
        probs = {b: float(sel.probs[b]) for b in res}
        if not probs:
            continue
        k, best, arg = brute.min_cardinality_max_mass(probs, p)
        nuc = set(sel.order[:sel.n_star].tolist())
        assert len(nuc) == k                                           # minimum cardinality
        assert abs(sum(probs[b] for b in nuc) - best) < 1e-12          # maximum mass at that size
        assert nuc in arg or len(arg) > 1


def test_topk_is_eq6_and_matches_library_sort_and_enumeration():
    rng = np.random.default_rng(5)
    for trial in range(50):
        n_b = int(rng.integers(2, 14))
        z = np.round(rng.standard_normal(n_b) * 2, 1)                  # ties likely
        K = int(rng.integers(0, n_b + 1))
        sel = S.select_topk(z, K)                                      # no reserved blocks: Eq. 6
        want = set(np.argsort(-z, kind="stable")[:K].tolist())         # library sort, stable = low index first
        assert set(sel.indices.tolist()) == want
        assert set(sel.indices.tolist()) == brute.topk_by_enumeration(z.tolist(), K)
    # K counts reserved blocks (R10): config 1's K=16 with 1 sink + 2 recency
    z = rng.standard_normal(64)
    sel = S.select_topk(z, 16, 1, 2)
    assert sel.budget == 16 and {0, 62, 63} <= set(sel.indices.tolist())
    inner = np.argsort(-z[1:62], kind="stable")[:13] + 1
    assert set(sel.indices.tolist()) == {0, 62, 63} | set(inner.tolist())


def test_special_cases():
    z = np.array([0.3, 2.0, -1.0, 7.5, 0.1, 0.0, 1.0, 0.2])
    # p -> 0+, K_min = 0: reserved U {argmax of residual}  (StreamingLLM window + 1 block)
    sel = S.select_dual_topp(z, 1e-9, 1, 2, 0)
    assert sel.indices.tolist() == [0, 3, 6, 7]
    # peaky distribution: nucleus saturates immediately, the K_min floor governs
    zp = np.zeros(64); zp[17] = 50.0
    for p in (0.7, 0.9, 0.99):
        sel = S.select_dual_topp(zp, p, 1, 2, 8)
        assert sel.n_star == 1 and sel.budget == 8
        assert sel.indices.tolist() == [0, 1, 2, 3, 4, 17, 62, 63]     # extension along descending score, low index first
    # small contexts (R21): everything reserved -> all blocks; overlapping sink/recency -> union
    assert S.select_dual_topp(np.array([1.0, 2.0]), 0.9, 1, 2, 8).indices.tolist() == [0, 1]
    assert S.select_dual_topp(np.array([1.0, 2.0, 3.0]), 0.5, 2, 2, 0).indices.tolist() == [0, 1, 2]
    assert S.select_dual_topp(np.array([5.0]), 0.9, 0, 0, 8).indices.tolist() == [0]
    # p = 1 selects all of B_res by definition (R20)
    assert S.select_dual_topp(np.arange(20.0) * 5, 1.0, 1, 2, 0).budget == 20
    # -0.0 and +0.0 tie; lower index wins
    zz = np.array([0.0, -0.0, 0.0, -0.0])
    assert S.select_topk(zz, 2).indices.tolist() == [0, 1]
    # uniform scores: p~ = 1/n each; p = 0.5 of 8 residual blocks -> 4 lowest indices
    sel = S.select_dual_topp(np.ones(8), 0.5, 0, 0, 0)
    assert sel.indices.tolist() == [0, 1, 2, 3]


def test_decode_form_ragged_tail_and_appended_token():
    rng = np.random.default_rng(6)
    L, blk = 150, 64                                  # 3 blocks, last has 22 tokens
    q = rng.standard_normal((4, 8)); w = np.full(4, 0.25); k = rng.standard_normal((200, 4, 8))
    k[170] = 100 * q                                  # beyond L: must be ignored
    s_bar, sel = S.select_decode(q, w, k, L, blk, "dual_topp", p=0.9, sink_blocks=1,
                                 recency_blocks=1, kmin_blocks=0)
    assert len(s_bar) == 3 and s_bar.max() < 50
    assert s_bar[2] == S.token_scores(q, w, k[128:150]).max()
    assert 2 in sel.indices                           # the block holding the query is reserved (R15)


def test_prefill_reduces_to_decode_at_q_block_1_and_bounds_members():
    rng = np.random.default_rng(8)
    L, blk, H, d = 96, 16, 2, 4
    sq = rng.standard_normal((L, H, d)); w = rng.standard_normal((L, H)); sk = rng.standard_normal((L, H, d))
    # q_block = 1: identical to the decode oracle at every position
    tiles = S.tile_scores_prefill(sq[40:48], w[40:48], sk, 40, 1, blk)
    for i, tile in enumerate(tiles):
        pos = 40 + i
        s_bar, _ = S.select_decode(sq[pos], w[pos], sk, pos + 1, blk, "topk", top_k=1)
        assert np.array_equal(tile, s_bar)
    # q_block = 16: tile score >= every member query's block score, and equals the max of them
    tiles = S.tile_scores_prefill(sq[32:64], w[32:64], sk, 32, 16, blk)
    assert [len(t) for t in tiles] == [3, 4]
    for i, tile in enumerate(tiles):
        members = []
        for qq in range(16):
            pos = 32 + 16 * i + qq
            s_bar = S.block_max(S.token_scores(sq[pos], w[pos], sk[:pos + 1]), blk)
            assert np.all(tile[:len(s_bar)] >= s_bar)
            members.append(np.pad(s_bar, (0, len(tile) - len(s_bar)), constant_values=-np.inf))
        assert np.array_equal(tile, np.max(members, axis=0))
    # selection per query block: recency = diagonal block + the ones before it
    res = S.select_prefill(sq[32:64], w[32:64], sk, 32, 16, blk, "dual_topp", p=0.5, sink_blocks=1,
                           recency_blocks=2, kmin_blocks=0)
    assert {0, 1, 2} <= set(res[0][1].indices.tolist()) and {0, 2, 3} <= set(res[1][1].indices.tolist())
