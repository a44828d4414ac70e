"""Pins for oracle/attention.py (steps a3/a3'): the all-blocks case against textbook dense
attention (scalar loops, and torch's fp64 CPU SDPA as an independent library routine),
gather form against mask form, closed-form special cases."""
import numpy as np
import pytest
import torch

from oracle import attention as A


def _rand(rng, L, H_q, H_kv, D):
    return (rng.standard_normal((H_q, D)), rng.standard_normal((L, H_kv, D)),
            rng.standard_normal((L, H_kv, D)))


def test_all_blocks_equals_textbook_dense_loops():
    rng = np.random.default_rng(1)
    L, H_q, H_kv, D, blk = 23, 4, 2, 6, 8             # ragged last block, GQA 2
    q, K, V = _rand(rng, L, H_q, H_kv, D)
    sc = 1 / np.sqrt(D)
    out, lse = A.sparse_attn_decode(q, K, V, range(3), L, blk, sc)
    ref = A.dense_attn_decode_loops(q.tolist(), K.tolist(), V.tolist(), L, sc)
    assert np.allclose(out, ref, atol=1e-13)


def test_all_blocks_equals_torch_sdpa_fp64_with_gqa():
    rng = np.random.default_rng(2)
    L, H_q, H_kv, D, blk = 300, 8, 2, 32, 64
    q, K, V = _rand(rng, L, H_q, H_kv, D)
    sc = 1 / np.sqrt(D)
    out, lse = A.sparse_attn_decode(q, K, V, range(5), L, blk, sc)
    G = H_q // H_kv
    tq = torch.from_numpy(q)[None, :, None, :]                                    # [1,Hq,1,D]
    tK = torch.from_numpy(K).permute(1, 0, 2).repeat_interleave(G, 0)[None]       # head h -> kv head h // G
    tV = torch.from_numpy(V).permute(1, 0, 2).repeat_interleave(G, 0)[None]
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tK, tV, scale=sc)[0, :, 0, :].numpy()
    assert np.allclose(out, ref, atol=1e-12)
    ref_lse = torch.logsumexp(sc * torch.einsum("hd,htd->ht", torch.from_numpy(q), tK[0]), dim=1).numpy()
    assert np.allclose(lse, ref_lse, atol=1e-12)


def test_gather_form_equals_mask_form_and_torch_masked_sdpa():
    rng = np.random.default_rng(3)
    L, H_q, H_kv, D, blk = 500, 8, 4, 16, 64
    q, K, V = _rand(rng, L, H_q, H_kv, D)
    sc = 0.3
    for blocks in ([0, 7], [1, 2, 5], [7], list(range(8))):
        out, _ = A.sparse_attn_decode(q, K, V, blocks, L, blk, sc)
        out2 = A.sparse_attn_decode_masked(q, K, V, blocks, L, blk, sc)
        assert np.allclose(out, out2, atol=1e-12)
        keep = torch.zeros(L, dtype=torch.bool)
        for b in blocks:
            keep[b * blk:(b + 1) * blk] = True
        G = H_q // H_kv
        tq = torch.from_numpy(q)[None, :, None, :]
        tK = torch.from_numpy(K).permute(1, 0, 2).repeat_interleave(G, 0)[None]
        tV = torch.from_numpy(V).permute(1, 0, 2).repeat_interleave(G, 0)[None]
        ref = torch.nn.functional.scaled_dot_product_attention(tq, tK, tV, attn_mask=keep[None, None, None, :],
                                                               scale=sc)[0, :, 0, :].numpy()
        assert np.allclose(out, ref, atol=1e-12)
    # order of the block list is irrelevant (it is a set)
    a, _ = A.sparse_attn_decode(q, K, V, [5, 1, 2], L, blk, sc)
    b, _ = A.sparse_attn_decode(q, K, V, [1, 2, 5], L, blk, sc)
    assert np.allclose(a, b, atol=1e-14)


def test_closed_forms():
    rng = np.random.default_rng(4)
    L, H_q, H_kv, D, blk = 128, 4, 2, 8, 64
    q, K, V = _rand(rng, L, H_q, H_kv, D)
    # identical V rows inside the selected block -> output is that row, whatever the logits
    V[64:128] = V[64]
    out, _ = A.sparse_attn_decode(q, K, V, [1], L, blk, 1.0)
    for h in range(H_q):
        assert np.allclose(out[h], V[64, h // 2], atol=1e-13)
    # zero query -> uniform average over the selected tokens; GQA map: head h reads KV head h // G
    V = rng.standard_normal((L, H_kv, D))
    out, lse = A.sparse_attn_decode(np.zeros((H_q, D)), K, V, [0], L, blk, 1.0)
    for h in range(H_q):
        assert np.allclose(out[h], V[:64, h // 2].mean(0), atol=1e-13)
    assert np.allclose(lse, np.log(64.0))
    # one dominant key -> output ~ its value row
    K2 = K.copy(); K2[70, :, :] = 0; K2[70, 0, :] = 100 * q[0]
    out, _ = A.sparse_attn_decode(q, K2, V, [0, 1], L, blk, 1.0)
    assert np.allclose(out[0], V[70, 0], atol=1e-9)
    # shift invariance of softmax: adding c*q-independent constant to all logits (scale K along q) unchanged
    # unselected tokens never matter
    V3 = V.copy(); V3[:64] = 1e9; K3 = K.copy(); K3[:64] = 1e3
    a, _ = A.sparse_attn_decode(q, K, V, [1], L, blk, 1.0)
    b, _ = A.sparse_attn_decode(q, K3, V3, [1], L, blk, 1.0)
    assert np.array_equal(a, b)


def test_prefill_form_against_torch_block_sparse_causal_mask_and_decode_form():
    rng = np.random.default_rng(5)
    L, H_q, H_kv, D, blk = 256, 4, 2, 8, 64
    Q = rng.standard_normal((128, H_q, D)); K = rng.standard_normal((L, H_kv, D)); V = rng.standard_normal((L, H_kv, D))
    q_start, sc = 128, 0.35
    lists = [[0, 2], [1, 2, 3]]                       # diagonal blocks 2 and 3 included
    out = A.sparse_attn_prefill(Q, K, V, lists, q_start, 64, blk, sc)
    G = H_q // H_kv
    mask = torch.zeros(128, L, dtype=torch.bool)
    for i, bl in enumerate(lists):
        for qq in range(64 * i, 64 * i + 64):
            for b in bl:
                for t in range(b * blk, (b + 1) * blk):
                    mask[qq, t] = t <= q_start + qq
    tq = torch.from_numpy(Q).permute(1, 0, 2)[None]
    tK = torch.from_numpy(K).permute(1, 0, 2).repeat_interleave(G, 0)[None]
    tV = torch.from_numpy(V).permute(1, 0, 2).repeat_interleave(G, 0)[None]
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tK, tV, attn_mask=mask[None, None], scale=sc)
    assert np.allclose(out, ref[0].permute(1, 0, 2).numpy(), atol=1e-12)
    # each query row equals the decode form with L = pos + 1
    for qq in (0, 63, 64, 127):
        pos = q_start + qq
        o, _ = A.sparse_attn_decode(Q[qq], K, V, lists[qq // 64], pos + 1, blk, sc)
        assert np.allclose(out[qq], o, atol=1e-13)


def test_paged_gather_round_trip_and_identity():
    """f3 / R32: scattering a logical cache into randomly placed pages and gathering it back is the identity (also with
    a ragged last page and pages shared with another sequence's allocation); the identity table is a plain reshape."""
    rng = np.random.default_rng(12)
    L, pt, H_kv, D = 1000, 64, 2, 8
    logical = rng.standard_normal((L, H_kv, D))
    n_log = -(-L // pt)
    n_pages = 40
    table = rng.permutation(n_pages)[:n_log]
    pool = rng.standard_normal((n_pages, pt, H_kv, D))                 # other sequences' pages: garbage to us
    for lp in range(n_log):
        t0, t1 = lp * pt, min((lp + 1) * pt, L)
        pool[table[lp], :t1 - t0] = logical[t0:t1]
    got = A.gather_paged_kv(pool, table, L, pt)
    assert np.array_equal(got, logical)
    ident = A.gather_paged_kv(logical[:960].reshape(15, pt, H_kv, D), np.arange(15), 960, pt)
    assert np.array_equal(ident, logical[:960])
    # a wrong table entry is visible: swapping two pages moves exactly those 128 tokens
    t2 = table.copy()
    t2[[3, 7]] = t2[[7, 3]]
    bad = A.gather_paged_kv(pool, t2, L, pt)
    diff = np.flatnonzero(np.any(bad != logical, axis=(1, 2)))
    assert set(diff // pt) == {3, 7}
