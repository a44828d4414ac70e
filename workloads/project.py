"""Seeded synthetic inputs of the upstream step f1 (selector projections).  No method arithmetic: random tensors only.

    hidden  uint16 [B][d_model]            BF16 bits, N(0, 1)
    w_q/w_k uint16 [H_idx*d_idx][d_model]  BF16 bits, N(0, 1/d_model)  (unit-variance projections)
    w_w     uint16 [H_idx][d_model]        BF16 bits, N(0, 1/d_model)
    pos     int32  [B]                     positions in [0, L)
"""
import numpy as np

from .bf16 import f32_to_bf16_bits


def make_project_workload(seed=6006, B=4, d_model=4096, H_idx=4, d_idx=64, L=131072):
    rng = np.random.Generator(np.random.Philox(seed))
    s = np.float32(1.0 / np.sqrt(d_model))
    return dict(
        hidden=f32_to_bf16_bits(rng.standard_normal((B, d_model), dtype=np.float32)),
        w_q=f32_to_bf16_bits(rng.standard_normal((H_idx * d_idx, d_model), dtype=np.float32) * s),
        w_k=f32_to_bf16_bits(rng.standard_normal((H_idx * d_idx, d_model), dtype=np.float32) * s),
        w_w=f32_to_bf16_bits(rng.standard_normal((H_idx, d_model), dtype=np.float32) * s),
        pos=rng.integers(0, L, size=B).astype(np.int32),
        B=B, d_model=d_model, H_idx=H_idx, d_idx=d_idx, L=L)
