"""Seeded synthetic decode workloads (Qwen3-shaped; BASELINE.json configs 1-4).

No method arithmetic here (see workloads/__init__.py): tensors are drawn,
shifted along stated directions and rounded once to BF16 bits.  Layouts:

    q      uint16 [B][H_q][D]            BF16 bits, the decode query
    K, V   uint16 [B][H_kv][L_cap][D]    BF16 bits, backbone KV cache ("HND")
    sel_q  uint16 [B][H_idx][d_idx]      BF16 bits, selector query q^I
    w      float32 [B][H_idx]            per-query mixing weights w_h
    sel_k  uint16 [B][L_cap][H_idx][d_idx]  BF16 bits, per-token selector keys k^I
    seq_len int32 [B]                    valid tokens per sequence (<= L_cap)

Recipes:

* ``planted`` (config 1): everything N(0,1); ``n_planted`` residual blocks get
  their selector keys and attention keys shifted +2.0 along the query
  direction; token 0 gets +4.0 (a high-logit sink).
* ``zipf`` (configs 2-4): background selector keys are N(0,1) with the
  component along each head's query direction projected out, so background
  scores are ~0; every residual block b gets a target logit
  l_b = s * ln(n_res / r_b) (r_b a random rank: a Zipf(s) block distribution
  after softmax) planted on one random peak token through one random owner
  head.  ``zipf_s`` is a float or a (lo, hi) log-uniform range per query
  (config 4's budget heterogeneity).
* ``gauss``: plain N(0,1) everywhere, random-sign w (edge-case tests).
"""
from dataclasses import dataclass, field

import numpy as np

from .bf16 import f32_to_bf16_bits, bf16_bits_to_f32


@dataclass
class DecodeWorkload:
    name: str
    seed: int
    B: int
    L_cap: int
    H_q: int
    H_kv: int
    D: int
    H_idx: int
    d_idx: int
    blk: int
    seq_len: np.ndarray
    q: np.ndarray
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
    planted_blocks: list = field(default_factory=list)

    def select_kwargs(self):
        return dict(top_k=self.top_k, p=self.p, sink_blocks=self.sink_blocks,
                    recency_blocks=self.recency_blocks, kmin_blocks=self.kmin_blocks,
                    temperature=self.temperature)


def _normal_bf16(rng, shape, chunk=1 << 24):
    """N(0,1) float32 -> BF16 bits, generated in chunks to bound temporaries."""
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.uint16)
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        out[s:e] = f32_to_bf16_bits(rng.standard_normal(e - s, dtype=np.float32))
    return out.reshape(shape)


def _unit(v):
    n = np.linalg.norm(v, axis=-1, keepdims=True)
    return v / np.maximum(n, 1e-30)


def make_decode_workload(name, seed, B, L, H_q=32, H_kv=8, D=128, H_idx=4, d_idx=64, blk=64,
                         kind="zipf", zipf_s=1.1, seq_lens=None, n_planted=3,
                         mode="dual_topp", top_k=0, p=0.90, sink_blocks=1, recency_blocks=2,
                         kmin_blocks=8, temperature=1.0, with_kv=True):
    rng = np.random.Generator(np.random.Philox(seed))
    L_cap = L
    seq_len = np.full(B, L, dtype=np.int32) if seq_lens is None else np.asarray(seq_lens, dtype=np.int32)
    assert seq_len.shape == (B,) and seq_len.max() <= L_cap and seq_len.min() >= 1

    q = _normal_bf16(rng, (B, H_q, D))
    sel_q = _normal_bf16(rng, (B, H_idx, d_idx))
    if kind == "gauss":
        w = (rng.standard_normal((B, H_idx)).astype(np.float32) / np.float32(H_idx * np.sqrt(d_idx)))
    else:
        w = np.full((B, H_idx), 1.0 / (H_idx * np.sqrt(d_idx)), dtype=np.float32)

    if with_kv:
        K = _normal_bf16(rng, (B, H_kv, L_cap, D))
        V = _normal_bf16(rng, (B, H_kv, L_cap, D))
    else:
        K = V = None
    sel_k = np.empty((B, L_cap, H_idx, d_idx), dtype=np.uint16)
    planted = []

    for b in range(B):
        Lb = int(seq_len[b])
        n_b = -(-Lb // blk)
        kf = rng.standard_normal((L_cap, H_idx, d_idx), dtype=np.float32)
        qf = bf16_bits_to_f32(sel_q[b])                     # [H_idx, d_idx]
        qhat = _unit(qf)
        if kind == "planted":
            lo, hi = min(1, n_b), max(min(1, n_b), n_b - 3)
            cand = np.arange(lo, hi)
            blocks = sorted(rng.choice(cand, size=min(n_planted, len(cand)), replace=False).tolist()) \
                if len(cand) else []
            planted.append(blocks)
            G = H_q // H_kv
            uf = bf16_bits_to_f32(q[b]).reshape(H_kv, G, D).sum(axis=1)   # per KV head
            uhat = _unit(uf)
            Kf = bf16_bits_to_f32(K[b]) if with_kv else None
            for blkid in blocks:
                t0, t1 = blkid * blk, min((blkid + 1) * blk, Lb)
                kf[t0:t1] += 2.0 * qhat[None]
                if with_kv:
                    Kf[:, t0:t1, :] += 2.0 * uhat[:, None, :]
            kf[0] += 4.0 * qhat
            if with_kv:
                Kf[:, 0, :] += 4.0 * uhat
                K[b] = f32_to_bf16_bits(Kf)
        elif kind == "zipf":
            # project the query direction out of every background key (per head)
            kf -= np.einsum("thd,hd->th", kf, qhat)[..., None] * qhat[None]
            res = np.ones(n_b, dtype=bool)
            res[:min(sink_blocks, n_b)] = False
            res[max(0, n_b - recency_blocks):] = False
            res_idx = np.nonzero(res)[0]
            n_res = len(res_idx)
            if n_res:
                if isinstance(zipf_s, (tuple, list)):
                    s_exp = float(np.exp(rng.uniform(np.log(zipf_s[0]), np.log(zipf_s[1]))))
                else:
                    s_exp = float(zipf_s)
                rank = rng.permutation(n_res) + 1
                logit = (s_exp * np.log(n_res / rank)).astype(np.float32)
                peak = res_idx * blk + rng.integers(0, blk, size=n_res)
                peak = np.minimum(peak, Lb - 1)
                owner = rng.integers(0, H_idx, size=n_res)
                qn = np.linalg.norm(qf, axis=-1)                       # [H_idx]
                amp = logit / (w[b, owner] * qn[owner])
                kf[peak, owner, :] += amp[:, None] * qhat[owner]
        elif kind != "gauss":
            raise ValueError(kind)
        sel_k[b] = f32_to_bf16_bits(kf)

    return DecodeWorkload(name=name, seed=seed, B=B, L_cap=L_cap, H_q=H_q, H_kv=H_kv, D=D,
                          H_idx=H_idx, d_idx=d_idx, blk=blk, seq_len=seq_len, q=q, K=K, V=V,
                          sel_q=sel_q, w=w, sel_k=sel_k, mode=mode, top_k=top_k, p=p,
                          sink_blocks=sink_blocks, recency_blocks=recency_blocks,
                          kmin_blocks=kmin_blocks, temperature=temperature,
                          sm_scale=float(1.0 / np.sqrt(D)), planted_blocks=planted)


# BASELINE.json configs (decode ones) plus reduced "mini" versions the oracle
# finishes in seconds (several tiles, ragged tails).
CONFIGS = {
    "cfg1": dict(seed=1001, B=1, L=4096, kind="planted", mode="topk", top_k=16),
    "cfg2": dict(seed=2002, B=8, L=32768, kind="zipf", zipf_s=1.1),
    "cfg3": dict(seed=3003, B=4, L=131072, kind="zipf", zipf_s=1.1),
    "cfg4_b1": dict(seed=4004, B=1, L=131072, H_q=64, kind="zipf", zipf_s=(1.14, 2.1)),
    "cfg4_b4": dict(seed=4004, B=4, L=131072, H_q=64, kind="zipf", zipf_s=(1.14, 2.1)),
    "cfg4_b16": dict(seed=4004, B=16, L=131072, H_q=64, kind="zipf", zipf_s=(1.14, 2.1)),
    # reduced cases for element-by-element parity
    "mini2": dict(seed=2102, B=3, L=8192, kind="zipf", zipf_s=1.1, seq_lens=[8192, 8000, 5321]),
    "mini3": dict(seed=3103, B=2, L=16384, kind="zipf", zipf_s=1.1, seq_lens=[16384, 12345]),
    "mini4": dict(seed=4104, B=4, L=8192, H_q=64, kind="zipf", zipf_s=(1.14, 2.1),
                  seq_lens=[8192, 8191, 4097, 700]),
}


def make_config(name, **overrides):
    kw = dict(CONFIGS[name])
    kw.update(overrides)
    return make_decode_workload(name, **kw)
