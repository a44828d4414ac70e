"""Upstream step f1 -- selector projections, RoPE, mixing weights (oracle).

TEST INFRASTRUCTURE (see oracle/__init__.py).  fp64.

PAPER.md:39: "q^I_h, k^I_{h,t} are the per-head query/key projections and W_w a small linear map producing the
per-query mixing weights w_h from the hidden state h_q"; 4 heads, head dim 128, "RoPE head dim 64".
The paper gives no more than that; readings R27-R29:

* q^I = W_q h, k^I = W_k h, w = W_w h: no bias, no activation (R27);
* rotary embedding on the first ``rope_dims`` dims of every selector head of q^I and k^I, rotate-half pairing
  (i, i + rope_dims/2), angle = pos * base^(-2 i / rope_dims); the remaining dims pass through (R28);
* everything in exact arithmetic here; the GPU rounds q^I and k^I once to BF16 after the rotation and quantises the
  cache entry from that BF16 value (R29), so tests compare after rounding.
"""
import numpy as np


def rope_angles(pos, rope_dims, base):
    """angle[i] = pos * base^(-2 i / rope_dims), i < rope_dims / 2."""
    i = np.arange(rope_dims // 2, dtype=np.float64)
    return float(pos) * np.power(float(base), -2.0 * i / float(rope_dims))


def rope_rotate(x, pos, rope_dims, base):
    """x [..., d]: rotate the pairs (i, i + rope_dims/2), i < rope_dims/2, of the last axis by angle[i]; dims >=
    rope_dims are returned unchanged."""
    x = np.asarray(x, dtype=np.float64)
    out = x.copy()
    half = rope_dims // 2
    ang = rope_angles(pos, rope_dims, base)
    c, s = np.cos(ang), np.sin(ang)
    x1, x2 = x[..., :half], x[..., half:rope_dims]
    out[..., :half] = x1 * c - x2 * s
    out[..., half:rope_dims] = x2 * c + x1 * s
    return out


def project(h, W_q, W_k, W_w, pos, H_idx, d_idx, rope_dims, base):
    """One token: h [d_model]; W_q, W_k [H_idx*d_idx, d_model]; W_w [H_idx, d_model] -> (q [H_idx, d_idx],
    k [H_idx, d_idx], w [H_idx]), q and k rotated to position ``pos``."""
    h = np.asarray(h, dtype=np.float64)
    q = (np.asarray(W_q, dtype=np.float64) @ h).reshape(H_idx, d_idx)
    k = (np.asarray(W_k, dtype=np.float64) @ h).reshape(H_idx, d_idx)
    w = np.asarray(W_w, dtype=np.float64) @ h
    return rope_rotate(q, pos, rope_dims, base), rope_rotate(k, pos, rope_dims, base), w
