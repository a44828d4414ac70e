"""Steps a3/a3' -- attention over the tokens of the selected blocks (oracle).

TEST INFRASTRUCTURE (see oracle/__init__.py).  fp64, max-subtracted softmax.

PAPER.md:47 (Fig. 2): "attention runs only over the gathered K_I, V_I";
PAPER.md:71: "the layer attends only to keys in a selected subset S_q of
blocks".  Standard details the paper does not restate (R19): sm_scale =
1/sqrt(D) is passed in, query head h reads KV head floor(h / G) with
G = H_q / H_kv, one index set is shared by all heads (R14).
"""
import numpy as np


def _tokens_of_blocks(blocks, L, blk):
    toks = []
    for b in blocks:
        toks.extend(range(int(b) * blk, min((int(b) + 1) * blk, L)))
    return np.asarray(toks, dtype=np.int64)


def sparse_attn_decode(q, K, V, blocks, L, blk, sm_scale):
    """Gather form.  q [H_q, D], K/V [>=L, H_kv, D], blocks = selected block ids.

    o_h = sum_{t in T_q} softmax_t(sm_scale * q_h . k_{g,t}) * v_{g,t},
    T_q = {t < L : floor(t/blk) in S_q}, g = floor(h / G).
    Returns (out [H_q, D], lse [H_q]) with lse the natural-log sum-exp of the
    scaled logits.
    """
    q = np.asarray(q, dtype=np.float64)
    K = np.asarray(K, dtype=np.float64)
    V = np.asarray(V, dtype=np.float64)
    H_q, D = q.shape
    H_kv = K.shape[1]
    G = H_q // H_kv
    toks = _tokens_of_blocks(blocks, L, blk)
    out = np.zeros((H_q, D))
    lse = np.full(H_q, -np.inf)
    if len(toks) == 0:
        return out, lse
    for h in range(H_q):
        g = h // G
        logits = sm_scale * (K[toks, g, :] @ q[h])
        m = logits.max()
        e = np.exp(logits - m)
        out[h] = (e[:, None] * V[toks, g, :]).sum(axis=0) / e.sum()
        lse[h] = m + np.log(e.sum())
    return out, lse


def sparse_attn_decode_masked(q, K, V, blocks, L, blk, sm_scale):
    """Mask form -- a second, independent coding of the same definition: dense
    attention over all L tokens with the logits of unselected tokens set to
    -inf.  Used only to pin ``sparse_attn_decode``."""
    q = np.asarray(q, dtype=np.float64)
    K = np.asarray(K, dtype=np.float64)[:L]
    V = np.asarray(V, dtype=np.float64)[:L]
    H_q, D = q.shape
    G = H_q // K.shape[1]
    keep = np.zeros(L, dtype=bool)
    for b in blocks:
        keep[int(b) * blk:(int(b) + 1) * blk] = True
    out = np.zeros((H_q, D))
    for h in range(H_q):
        logits = sm_scale * np.einsum("td,d->t", K[:, h // G, :], q[h])
        logits = np.where(keep, logits, -np.inf)
        pr = np.exp(logits - logits.max())
        pr = pr / pr.sum()
        out[h] = pr @ V[:, h // G, :]
    return out


def dense_attn_decode_loops(q, K, V, L, sm_scale):
    """Plain textbook softmax attention with Python loops (tiny inputs only):
    the definition a p = 1 / all-blocks selection must reproduce."""
    import math
    H_q, D = len(q), len(q[0])
    H_kv = len(K[0])
    G = H_q // H_kv
    out = [[0.0] * D for _ in range(H_q)]
    for h in range(H_q):
        g = h // G
        logits = [sm_scale * sum(float(q[h][d]) * float(K[t][g][d]) for d in range(D))
                  for t in range(L)]
        m = max(logits)
        ws = [math.exp(x - m) for x in logits]
        Z = sum(ws)
        for d in range(D):
            out[h][d] = sum(ws[t] * float(V[t][g][d]) for t in range(L)) / Z
    return np.asarray(out)


def sparse_attn_prefill(Q, K, V, block_lists, q_start, q_block, blk, sm_scale):
    """Chunked-prefill form ("the selector and block-sparse
    kernels run ... under a full causal mask").

    Q [Tq, H_q, D] at absolute positions q_start..q_start+Tq-1; block_lists[i]
    = selected key blocks of query block i.  Each query token attends to the
    tokens of its block's selected key blocks with t <= its own position (only
    the diagonal block actually needs the mask).  Returns out [Tq, H_q, D].
    """
    Q = np.asarray(Q, dtype=np.float64)
    K = np.asarray(K, dtype=np.float64)
    V = np.asarray(V, dtype=np.float64)
    Tq, H_q, D = Q.shape
    G = H_q // K.shape[1]
    out = np.zeros((Tq, H_q, D))
    for i, blocks in enumerate(block_lists):
        for qq in range(i * q_block, (i + 1) * q_block):
            pos = q_start + qq
            toks = _tokens_of_blocks(blocks, pos + 1, blk)          # t <= pos
            for h in range(H_q):
                g = h // G
                logits = sm_scale * (K[toks, g, :] @ Q[qq, h])
                e = np.exp(logits - logits.max())
                out[qq, h] = (e[:, None] * V[toks, g, :]).sum(axis=0) / e.sum()
    return out


def gather_paged_kv(pool, page_table, L, page_tokens):
    """f3 (R32) -- a paged K or V cache read back as the logical tensor.

    pool [n_pages][page_tokens][H_kv][D], page_table [ceil(L / page_tokens)] physical page of every logical
    page of ONE sequence -> [L][H_kv][D]: logical token t is row t % page_tokens of page
    page_table[t // page_tokens].  Paging is a storage layout, not arithmetic: attention over a paged cache
    is, by definition, attention over this tensor ("attention runs only over the gathered
    K_I, V_I", says nothing about where the rows live).  Written as the loop it is.
    """
    pool = np.asarray(pool)
    out = np.empty((L,) + pool.shape[2:], dtype=pool.dtype)
    for t in range(L):
        out[t] = pool[int(page_table[t // page_tokens]), t % page_tokens]
    return out
