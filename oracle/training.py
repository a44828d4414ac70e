"""f4 -- the training-side reductions: teacher and student distributions and the two KL objectives (oracle).

TEST INFRASTRUCTURE (see oracle/__init__.py).  fp64 throughout, one sequence, causal.

PAPER.md:49-53 (Eq. 1, 2): the teacher p^tau[q, t] = (1 / H_q) sum_h softmax_t(s_t[h, q, .]) "averages the H_q per-head
softmaxes (softmax then mean)"; the student p^sigma[q, t] = softmax_t(s_s[q, .]) is "a single softmax over s_s".
PAPER.md:55-58 (Eq. 3): DenseKL = sum_t p^tau log(p^tau / p^sigma) per query, averaged over the B L queries.
PAPER.md:60-64 (Eq. 4): SparseKL, the same "only over the selector's own top-K selected set S_q, with both distributions
renormalized to that set".

Readings: R34 the backbone scores are the usual scaled dot products, s_t[h, q, t] =
sm_scale * q_h . k_{g(h), t} (GQA as in R19), and both softmaxes run over the causally visible keys t <= q.  R35 S_q is
the token set of the inference rule of section 2.3 applied to that query: the K_train / blk best blocks by block-max
score (Eq. 6; ties to the lower index, R7; reserved sink / recency blocks counted inside K, R10), restricted to t <= q --
PAPER.md:96 counts K_train in tokens ("K_train = 8K selected tokens") and PAPER.md:365 fixes 16-token blocks, so
K_train = 8192 is 512 blocks.  R36 0 log 0 = 0; a query whose S_q carries zero teacher mass contributes 0.
"""
import numpy as np

from . import selection as OS


def backbone_logits(Q, K, sm_scale):
    """Q [L, H_q, D], K [L, H_kv, D] -> s_t [H_q, L, L] = sm_scale * q_h . k_{g(h), t}; -inf above the diagonal."""
    Q = np.asarray(Q, dtype=np.float64)
    K = np.asarray(K, dtype=np.float64)
    L, H_q, _ = Q.shape
    G = H_q // K.shape[1]
    out = np.empty((H_q, L, L))
    future = np.triu(np.ones((L, L), dtype=bool), 1)
    for h in range(H_q):
        s = sm_scale * (Q[:, h, :] @ K[:, h // G, :].T)
        s[future] = -np.inf
        out[h] = s
    return out


def _row_softmax(s):
    m = s.max(axis=-1, keepdims=True)
    e = np.exp(s - m)
    return e / e.sum(axis=-1, keepdims=True)


def teacher_distribution(Q, K, sm_scale):
    """Eq. 1: p^tau[q, t] = mean over heads of softmax_t(s_t[h, q, .]) (softmax, THEN mean).  -> [L, L], zero for t > q."""
    s = backbone_logits(Q, K, sm_scale)
    p = np.zeros(s.shape[1:])
    for h in range(s.shape[0]):
        p += _row_softmax(s[h])
    return p / s.shape[0]


def student_scores(sel_q, w, sel_k):
    """s_s[q, t] = sum_h w_h[q] ReLU(q^I_h[q] . k^I_{h,t}) for t <= q, -inf above the diagonal.
    sel_q [L, H, d], w [L, H], sel_k [L, H, d] -> [L, L]."""
    L = np.asarray(sel_q).shape[0]
    s = np.full((L, L), -np.inf)
    for q in range(L):
        s[q, :q + 1] = OS.token_scores(sel_q[q], w[q], np.asarray(sel_k)[:q + 1])
    return s


def student_distribution(s_s):
    """Eq. 2: p^sigma[q, .] = softmax_t(s_s[q, .]) over t <= q."""
    return _row_softmax(np.asarray(s_s, dtype=np.float64))


def kl_rows(p, q_):
    """sum_t p log(p / q) per row with 0 log 0 = 0 (R36)."""
    p = np.asarray(p, dtype=np.float64)
    q_ = np.asarray(q_, dtype=np.float64)
    out = np.zeros(p.shape[0])
    for r in range(p.shape[0]):
        nz = p[r] > 0
        out[r] = np.sum(p[r, nz] * (np.log(p[r, nz]) - np.log(q_[r, nz])))
    return out


def selected_tokens(s_row, q, blk, k_blocks, sink_blocks=0, recency_blocks=0):
    """R35: the tokens t <= q of the blocks Eq. 6 selects for query q (block-max scores over the visible tokens)."""
    s_bar = OS.block_max(np.asarray(s_row, dtype=np.float64)[:q + 1], blk)
    sel = OS.select_topk(s_bar, k_blocks, sink_blocks, recency_blocks)
    mask = np.zeros(q + 1, dtype=bool)
    for b in sel.indices:
        mask[int(b) * blk:min((int(b) + 1) * blk, q + 1)] = True
    return mask


def dense_kl(p_tau, p_sigma):
    """Eq. 3, per query (the loss is the mean over queries)."""
    return kl_rows(p_tau, p_sigma)


def sparse_kl(p_tau, p_sigma, s_s, blk, k_blocks, sink_blocks=0, recency_blocks=0):
    """Eq. 4, per query: both distributions restricted to S_q and renormalised there."""
    L = p_tau.shape[0]
    out = np.zeros(L)
    for q in range(L):
        m = selected_tokens(s_s[q], q, blk, k_blocks, sink_blocks, recency_blocks)
        pt, ps = p_tau[q, :q + 1][m], p_sigma[q, :q + 1][m]
        if pt.sum() <= 0:
            continue
        out[q] = kl_rows((pt / pt.sum())[None], (ps / ps.sum())[None])[0]
    return out


def training_reductions(Q, K, sm_scale, sel_q, w, sel_k, blk, k_blocks, sink_blocks=0, recency_blocks=0):
    """-> dict(dense_kl [L], sparse_kl [L], teacher_lse [L, H_q], p_tau, p_sigma, s_s)."""
    s_t = backbone_logits(Q, K, sm_scale)
    m = s_t.max(axis=-1)
    lse = (m + np.log(np.exp(s_t - m[..., None]).sum(axis=-1))).T            # [L, H_q]
    p_tau = teacher_distribution(Q, K, sm_scale)
    s_s = student_scores(sel_q, w, sel_k)
    p_sigma = student_distribution(s_s)
    return dict(dense_kl=dense_kl(p_tau, p_sigma),
                sparse_kl=sparse_kl(p_tau, p_sigma, s_s, blk, k_blocks, sink_blocks, recency_blocks),
                teacher_lse=lse, p_tau=p_tau, p_sigma=p_sigma, s_s=s_s)


def training_row(q, Q_row, K_prefix, sm_scale, sel_q_row, w_row, sel_k_prefix, blk, k_blocks, sink_blocks=0, recency_blocks=0):
    """Row q of training_reductions from the causal prefix alone (row q of every quantity above depends on the keys t <= q
    only) -- the same definitions through the same sub-functions, for sampled rows of sequences too long for the L x L
    matrices (pinned against training_reductions on a short sequence, tests/test_oracle_training.py).
    Q_row [H_q, D], K_prefix [q + 1, H_kv, D], sel_q_row [H, d], w_row [H], sel_k_prefix [q + 1, H, d]
    -> dict(dense_kl, sparse_kl, teacher_lse [H_q], s_s [q + 1])."""
    Q_row = np.asarray(Q_row, dtype=np.float64)
    K_prefix = np.asarray(K_prefix, dtype=np.float64)
    assert K_prefix.shape[0] == q + 1
    H_q = Q_row.shape[0]
    G = H_q // K_prefix.shape[1]
    s_t = np.stack([sm_scale * (K_prefix[:, h // G, :] @ Q_row[h]) for h in range(H_q)])      # [H_q, q + 1]
    m = s_t.max(axis=-1)
    lse = m + np.log(np.exp(s_t - m[:, None]).sum(axis=-1))
    p_tau = _row_softmax(s_t).mean(axis=0)                                                     # Eq. 1: softmax, then mean
    s_s = OS.token_scores(sel_q_row, w_row, np.asarray(sel_k_prefix))
    p_sigma = _row_softmax(np.asarray(s_s, dtype=np.float64)[None])[0]                         # Eq. 2
    dkl = kl_rows(p_tau[None], p_sigma[None])[0]                                               # Eq. 3
    msk = selected_tokens(s_s, q, blk, k_blocks, sink_blocks, recency_blocks)                  # R35
    pt, ps = p_tau[msk], p_sigma[msk]
    skl = kl_rows((pt / pt.sum())[None], (ps / ps.sum())[None])[0] if pt.sum() > 0 else 0.0    # Eq. 4, R36
    return dict(dense_kl=dkl, sparse_kl=skl, teacher_lse=lse, s_s=np.asarray(s_s, dtype=np.float64))
