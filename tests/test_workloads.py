"""Host-side checks of the seeded input generators (no GPU): determinism, shapes, and that the
recipes produce the structure DESIGN.md section 5 promises, as seen by the oracle."""
import numpy as np

from oracle import selection as S
from oracle.bf16 import bf16_bits_to_f64
from workloads import make_config, make_decode_workload, make_prefill_workload, f32_to_bf16_bits, bf16_bits_to_f32


def test_bf16_rounding_is_rne():
    x = np.array([1.0, 1.00390625, 1.001953125, 1.005859375, -2.5, 3.0e38, 1e-40], dtype=np.float32)
    b = f32_to_bf16_bits(x)
    back = bf16_bits_to_f32(b)
    assert back[0] == 1.0 and back[1] == 1.0 and back[2] == 1.0        # 1+2^-8 ties to even (down); 1+2^-9 rounds down
    assert back[3] == np.float32(1.0078125)                           # 1+3*2^-9 rounds up
    assert np.array_equal(bf16_bits_to_f64(b), back.astype(np.float64))
    y = np.random.default_rng(0).standard_normal(10000).astype(np.float32)
    assert np.abs(bf16_bits_to_f32(f32_to_bf16_bits(y)) - y).max() <= np.abs(y).max() * 2.0 ** -8


def test_deterministic_and_shapes():
    a = make_config("cfg1")
    b = make_config("cfg1")
    for f in ("q", "K", "V", "sel_q", "w", "sel_k", "seq_len"):
        assert np.array_equal(getattr(a, f), getattr(b, f))
    assert a.K.shape == (1, 8, 4096, 128) and a.sel_k.shape == (1, 4096, 4, 64) and a.q.shape == (1, 32, 128)
    assert a.mode == "topk" and a.top_k == 16 and a.sink_blocks == 1 and a.recency_blocks == 2


def test_config1_planted_blocks_are_selected_by_the_oracle():
    wl = make_config("cfg1")
    s_bar, sel = S.select_decode(bf16_bits_to_f64(wl.sel_q[0]), wl.w[0], bf16_bits_to_f64(wl.sel_k[0]),
                                 int(wl.seq_len[0]), wl.blk, "topk", **wl.select_kwargs())
    assert sel.budget == 16
    assert set(wl.planted_blocks[0]) <= set(sel.indices.tolist())
    assert {0, 62, 63} <= set(sel.indices.tolist())


def test_zipf_recipe_gives_zipf_like_budgets():
    wl = make_decode_workload("z", 77, B=2, L=32768, kind="zipf", zipf_s=1.1, with_kv=False)
    for b in range(2):
        s_bar, sel = S.select_decode(bf16_bits_to_f64(wl.sel_q[b]), wl.w[b], bf16_bits_to_f64(wl.sel_k[b]),
                                     32768, 64, "dual_topp", **wl.select_kwargs())
        # Zipf 1.1 over 509 residual blocks, p = .9 -> about 200 content blocks
        assert 150 <= sel.budget <= 260, sel.budget
        assert 0.10 <= sel.probs.max() <= 0.30
    het = make_decode_workload("h", 78, B=6, L=16384, kind="zipf", zipf_s=(1.14, 2.1), with_kv=False)
    budgets = [S.select_decode(bf16_bits_to_f64(het.sel_q[b]), het.w[b], bf16_bits_to_f64(het.sel_k[b]),
                               16384, 64, "dual_topp", **het.select_kwargs())[1].budget for b in range(6)]
    assert min(budgets) >= 8 and max(budgets) > 2 * min(budgets)


def test_prefill_workload_shapes():
    wl = make_prefill_workload(L=512, with_kv=True)
    assert wl.Q.shape == (512, 32, 128) and wl.K.shape == (8, 512, 128) and wl.sel_k.shape == (512, 4, 64)
    assert wl.w.shape == (512, 4) and wl.w.min() > 0
