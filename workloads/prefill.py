"""Seeded synthetic chunked-prefill workload (BASELINE.json config 5).

No method arithmetic here.  One sequence of L tokens, causal.  Selector Q and K
are N(0,1) plus a low-rank "topic" component (n_topics random directions, each
span of ``topic_span`` consecutive tokens assigned one topic, amplitude
``topic_amp``) so that tile scores are structured rather than flat: a query
block's mass concentrates on the earlier spans that share its topic, which at
the defaults gives per-query-block densities from about 0.15 to 0.85 at
p = 0.9 (the per-layer K/L range of PAPER.md:166); w_h[q] = (1 + 0.25 u) / (H_idx sqrt(d_idx)),
u ~ U(-1, 1).  Attention Q, K, V ~ N(0,1).  Layouts:

    Q      uint16 [L][H_q][D]           BF16 bits
    K, V   uint16 [H_kv][L][D]          BF16 bits ("HND", batch of one)
    sel_q  uint16 [L][H_idx][d_idx]
    w      float32 [L][H_idx]
    sel_k  uint16 [L][H_idx][d_idx]
"""
from dataclasses import dataclass

import numpy as np

from .bf16 import f32_to_bf16_bits


@dataclass
class PrefillWorkload:
    name: str
    seed: int
    L: int
    H_q: int
    H_kv: int
    D: int
    H_idx: int
    d_idx: int
    blk: int
    q_block: int
    Q: np.ndarray
    K: np.ndarray
    V: np.ndarray
    sel_q: np.ndarray
    w: np.ndarray
    sel_k: np.ndarray
    mode: str = "dual_topp"
    top_k: int = 0
    p: float = 0.90
    sink_blocks: int = 1
    recency_blocks: int = 2
    kmin_blocks: int = 8
    temperature: float = 1.0
    sm_scale: float = 0.0

    def select_kwargs(self):
        return dict(top_k=self.top_k, p=self.p, sink_blocks=self.sink_blocks,
                    recency_blocks=self.recency_blocks, kmin_blocks=self.kmin_blocks,
                    temperature=self.temperature)


def make_prefill_workload(name="cfg5", seed=5005, L=65536, H_q=32, H_kv=8, D=128, H_idx=4,
                          d_idx=64, blk=64, q_block=64, n_topics=16, topic_amp=5.5, topic_span=256,
                          mode="dual_topp", top_k=0, p=0.90, sink_blocks=1, recency_blocks=2,
                          kmin_blocks=8, temperature=1.0, with_kv=True):
    rng = np.random.Generator(np.random.Philox(seed))
    topics = rng.standard_normal((n_topics, H_idx, d_idx), dtype=np.float32)
    topics /= np.linalg.norm(topics, axis=-1, keepdims=True)
    n_span = -(-L // topic_span)
    assign = np.repeat(rng.integers(0, n_topics, size=n_span), topic_span)[:L]
    sq = rng.standard_normal((L, H_idx, d_idx), dtype=np.float32) + topic_amp * topics[assign]
    sk = rng.standard_normal((L, H_idx, d_idx), dtype=np.float32) + topic_amp * topics[assign]
    u = rng.uniform(-1.0, 1.0, size=(L, H_idx)).astype(np.float32)
    w = ((1.0 + 0.25 * u) / np.float32(H_idx * np.sqrt(d_idx))).astype(np.float32)
    if with_kv:
        Q = f32_to_bf16_bits(rng.standard_normal((L, H_q, D), dtype=np.float32))
        K = f32_to_bf16_bits(rng.standard_normal((H_kv, L, D), dtype=np.float32))
        V = f32_to_bf16_bits(rng.standard_normal((H_kv, L, D), dtype=np.float32))
    else:
        Q = K = V = None
    return PrefillWorkload(name=name, seed=seed, L=L, H_q=H_q, H_kv=H_kv, D=D, H_idx=H_idx,
                           d_idx=d_idx, blk=blk, q_block=q_block, Q=Q, K=K, V=V,
                           sel_q=f32_to_bf16_bits(sq), w=w, sel_k=f32_to_bf16_bits(sk),
                           mode=mode, top_k=top_k, p=p, sink_blocks=sink_blocks,
                           recency_blocks=recency_blocks, kmin_blocks=kmin_blocks,
                           temperature=temperature, sm_scale=float(1.0 / np.sqrt(D)))
