"""Steps a1/a2 -- selector scoring, block pooling and the two selection rules (oracle).

TEST INFRASTRUCTURE (see oracle/__init__.py).  fp64 throughout, on the exact
values of the BF16 (or dequantised) inputs.  The algorithm is followed step by
step in the paper's order; the readings R* are listed in DESIGN.md section 3.
"""
from dataclasses import dataclass, field

import numpy as np


# --------------------------------------------------------------------------
# a1: score + block max
# --------------------------------------------------------------------------

def token_scores(q_sel, w, k_sel):
    """PAPER.md:39 (section 2.1): s_s[q,t] = sum_h w_h * ReLU(q^I_h . k^I_{h,t}).

    q_sel [H_idx, d_idx], w [H_idx], k_sel [L, H_idx, d_idx]  ->  s [L].
    No 1/sqrt(d) factor (the formula has none, R13); w_h may be negative.
    """
    q_sel = np.asarray(q_sel, dtype=np.float64)
    w = np.asarray(w, dtype=np.float64)
    k_sel = np.asarray(k_sel, dtype=np.float64)
    dots = np.einsum("thd,hd->th", k_sel, q_sel)
    return (w[None, :] * np.maximum(dots, 0.0)).sum(axis=1)


def block_max(s, blk):
    """PAPER.md:71 (section 2.3): s_bar[q,b] = max_{t in b} s_s[q,t].

    s [L] -> s_bar [ceil(L/blk)]; the ragged last block takes the max over its
    valid tokens only.
    """
    s = np.asarray(s, dtype=np.float64)
    L = s.shape[0]
    n_b = -(-L // blk)
    out = np.empty(n_b, dtype=np.float64)
    for b in range(n_b):
        out[b] = s[b * blk:min((b + 1) * blk, L)].max()
    return out


# --------------------------------------------------------------------------
# a2: reserved tier, static top-K (Eq. 6), dual top-p (Eq. 7-8)
# --------------------------------------------------------------------------

@dataclass
class Selection:
    indices: np.ndarray                 # ascending block ids, int64
    budget: int                         # |S_q|, reserved blocks included
    probs: np.ndarray                   # p~ on B_res, 0 on reserved blocks   [n_b]
    order: np.ndarray                   # B_res sorted by (z desc, index asc)
    cum: np.ndarray = field(default=None)    # cumulative mass along `order`
    n_star: int = 0                     # nucleus size before the K_min floor
    n_taken: int = 0                    # residual blocks taken (after the floor)


def reserved_mask(n_b, sink_blocks, recency_blocks):
    """"a fixed prefix of sink blocks S_sink and a fixed suffix of
    recency blocks S_rec ... are reserved".  Block units (R9); the block that
    holds the query is the last recency block (R15); overlapping prefixes and
    suffixes simply union (R21)."""
    m = np.zeros(n_b, dtype=bool)
    m[:min(sink_blocks, n_b)] = True
    m[max(0, n_b - recency_blocks):] = True
    return m


def _sorted_residual(z, res_idx):
    """B_res sorted by score descending, ties -> lower block index first (R7).
    -0.0 and +0.0 compare equal."""
    zz = z[res_idx] + 0.0
    return res_idx[np.lexsort((res_idx, -zz))]


def select_topk(s_bar, top_k, sink_blocks=0, recency_blocks=0):
    """PAPER.md:79 Eq. 6: S_q = argTop-K_b s_bar[q,b].

    With reserved blocks (R10) K counts them: S_q = reserved U the
    max(0, K - |reserved|) best residual blocks.  sink = recency = 0 is Eq. 6
    exactly.
    """
    z = np.asarray(s_bar, dtype=np.float64)
    n_b = z.shape[0]
    res = reserved_mask(n_b, sink_blocks, recency_blocks)
    res_idx = np.nonzero(~res)[0]
    order = _sorted_residual(z, res_idx)
    n_take = min(max(0, top_k - int(res.sum())), len(order))
    sel = res.copy()
    sel[order[:n_take]] = True
    idx = np.nonzero(sel)[0].astype(np.int64)
    return Selection(indices=idx, budget=len(idx), probs=np.zeros(n_b), order=order,
                     n_star=n_take, n_taken=n_take)


def residual_distribution(s_bar, sink_blocks, recency_blocks, temperature=1.0):
    """PAPER.md:85 Eq. 7: p~[q,b] = softmax_{b in B_res} s_bar[q,b] (temperature
    PAPER.md:403, default 1.0).  Returns p~ over all n_b blocks with zeros on
    the reserved ones (R11: the distribution lives on B_res only)."""
    z = np.asarray(s_bar, dtype=np.float64) / float(temperature)
    n_b = z.shape[0]
    res = reserved_mask(n_b, sink_blocks, recency_blocks)
    p = np.zeros(n_b, dtype=np.float64)
    if (~res).any():
        zr = z[~res]
        e = np.exp(zr - zr.max())
        p[~res] = e / e.sum()
    return p


def select_dual_topp(s_bar, p, sink_blocks, recency_blocks, kmin_blocks, temperature=1.0):
    """PAPER.md:83-92 Eq. 7-8.

    Tier 1: reserve S_sink and S_rec.  Tier 2: nucleus on the residual
    distribution p~ (Eq. 7): "the smallest prefix of B_res, sorted by p~
    descending, whose cumulative mass reaches p" (>= p, R6; p >= 1 selects all
    of B_res by definition, R20).  Floor: "extending S_nuc along descending
    scores" until |S_q| >= min(K_min, n_b), reserved blocks counted (R8).
    Sorting by z is the same order as sorting by p~ (softmax is monotone, R25).
    """
    z = np.asarray(s_bar, dtype=np.float64) / float(temperature)
    n_b = z.shape[0]
    res = reserved_mask(n_b, sink_blocks, recency_blocks)
    res_idx = np.nonzero(~res)[0]
    probs = residual_distribution(s_bar, sink_blocks, recency_blocks, temperature)
    order = _sorted_residual(z, res_idx)
    n_res = len(order)
    cum = np.cumsum(probs[order])                    # sequential fp64 prefix mass
    if n_res == 0:
        n_star = 0
    elif p >= 1.0:
        n_star = n_res
    else:
        hit = np.nonzero(cum >= p)[0]
        n_star = int(hit[0]) + 1 if len(hit) else n_res
    n_reserved = int(res.sum())
    n_take = n_star
    target = min(kmin_blocks, n_b)
    if n_reserved + n_take < target:
        n_take = min(n_res, target - n_reserved)
    sel = res.copy()
    sel[order[:n_take]] = True
    idx = np.nonzero(sel)[0].astype(np.int64)
    return Selection(indices=idx, budget=len(idx), probs=probs, order=order, cum=cum,
                     n_star=n_star, n_taken=n_take)


# --------------------------------------------------------------------------
# decode form: one query per sequence
# --------------------------------------------------------------------------

def select_decode(q_sel, w, k_sel, L, blk, mode, *, top_k=0, p=0.9, sink_blocks=0,
                  recency_blocks=0, kmin_blocks=0, temperature=1.0):
    """One decode query at position L-1 against keys 0..L-1 (already appended, R15).

    Returns (s_bar [n_b], Selection)."""
    s = token_scores(q_sel, w, np.asarray(k_sel)[:L])
    s_bar = block_max(s, blk)
    if mode == "topk":
        sel = select_topk(s_bar, top_k, sink_blocks, recency_blocks)
    elif mode == "dual_topp":
        sel = select_dual_topp(s_bar, p, sink_blocks, recency_blocks, kmin_blocks, temperature)
    else:
        raise ValueError(mode)
    return s_bar, sel


# --------------------------------------------------------------------------
# prefill form: one selection per query block (PARITY UNPINNED, see __init__)
# --------------------------------------------------------------------------

def n_blocks_visible(q_start, i, q_block, blk):
    """Number of key blocks the i-th query block can see: index of the block
    holding its last token, plus one."""
    last = q_start + (i + 1) * q_block - 1
    return last // blk + 1


def tile_scores_prefill(q_sel, w, k_sel, q_start, q_block, blk):
    """"Scoring is block-wise: one score per query-block x
    key-block tile".  Reading R2: s_bar[i,j] = max_{q in i} max_{t in j, t<=q}
    s_s[q,t] with per-query weights w_h[q].

    q_sel [Tq, H, d], w [Tq, H], k_sel [>=q_start+Tq, H, d] -> list over query
    blocks i of s_bar_i [n_b(i)].  q_block = 1 reproduces the decode form.
    """
    q_sel = np.asarray(q_sel, dtype=np.float64)
    w = np.asarray(w, dtype=np.float64)
    k_sel = np.asarray(k_sel, dtype=np.float64)
    Tq = q_sel.shape[0]
    assert Tq % q_block == 0
    out = []
    for i in range(Tq // q_block):
        n_b = n_blocks_visible(q_start, i, q_block, blk)
        tile = np.full(n_b, -np.inf)
        for qq in range(i * q_block, (i + 1) * q_block):
            pos = q_start + qq
            s = token_scores(q_sel[qq], w[qq], k_sel[:pos + 1])     # causal: t <= pos
            sb = block_max(s, blk)
            tile[:len(sb)] = np.maximum(tile[:len(sb)], sb)
        out.append(tile)
    return out


def select_prefill(q_sel, w, k_sel, q_start, q_block, blk, mode, **kw):
    """Per query block: tile scores (R2) then steps 3-7 exactly as in decode.
    Recency = the diagonal block and the recency_blocks-1 before it (the last
    recency_blocks visible blocks).  Returns list of (s_bar_i, Selection_i)."""
    tiles = tile_scores_prefill(q_sel, w, k_sel, q_start, q_block, blk)
    res = []
    for s_bar in tiles:
        if mode == "topk":
            sel = select_topk(s_bar, kw.get("top_k", 0), kw.get("sink_blocks", 0),
                              kw.get("recency_blocks", 0))
        else:
            sel = select_dual_topp(s_bar, kw.get("p", 0.9), kw.get("sink_blocks", 0),
                                   kw.get("recency_blocks", 0), kw.get("kmin_blocks", 0),
                                   kw.get("temperature", 1.0))
        res.append((s_bar, sel))
    return res
