"""Randomised parity sweep of the decode path (-m gpu): many small seeded geometries per test -- batch, ragged lengths,
block size 16 / 64, cache format, selector head dim, rule parameters, K/V layout (contiguous, token-major, paged) --
each compared with the fp64 oracle exactly as the targeted tests do (tests/test_gpu_decode.py).  Nothing here is a new
claim; it widens the input space the same assertions are made on."""
import numpy as np
import pytest

from tests import _harness as H
from tests.test_gpu_decode import MAX_ABS, MEAN_ABS, _check_attend, _check_select, torch_cuda  # noqa: F401
from workloads import make_decode_workload

pytestmark = pytest.mark.gpu


def _random_workload(rng, case, with_kv):
    blk = int(rng.choice([16, 64]))
    B = int(rng.integers(1, 6))
    L_cap = int(rng.choice([64, 128, 320, 1024, 2048, 3008, 8192] + ([] if with_kv else [36032])))   # 36032 / 16 > 2048 blocks
    seq_lens = [int(rng.integers(1, L_cap + 1)) for _ in range(B)]
    seq_lens[int(rng.integers(0, B))] = L_cap if rng.random() < 0.5 else seq_lens[0]
    kw = dict(seed=9000 + case, B=B, L=L_cap, seq_lens=seq_lens, blk=blk, d_idx=int(rng.choice([64, 128])),
              kind=str(rng.choice(["gauss", "zipf"])), H_q=int(rng.choice([8, 16, 32, 64])),
              sink_blocks=int(rng.integers(0, 10)), recency_blocks=int(rng.integers(0, 18)),
              kmin_blocks=int(rng.integers(0, 40)), p=float(rng.choice([0.3, 0.7, 0.9, 0.99, 1.0])),
              with_kv=with_kv)
    return make_decode_workload("fuzz%d" % case, **kw)


@pytest.mark.parametrize("chunk", range(4))
def test_fuzz_selection(torch_cuda, chunk):
    rng = np.random.default_rng(4242 + chunk)
    report = []
    for case in range(chunk * 30, chunk * 30 + 30):
        wl = _random_workload(rng, case, with_kv=False)
        fmt = str(rng.choice(["bf16", "mxfp4", "int4_e4m3", "fp8_e4m3"]))
        if case % 5 == 4:                    # f2 formats of round 2 (drawn apart: the older cases keep their formats)
            fmt = ("mxint8", "int4_bf16s")[(case // 5) % 2]
        dd = H.DeviceDecode(wl, fmt, with_kv=False)
        _check_select(dd, fmt, report)
        n_b = dd.n_b_max
        res = wl.sink_blocks + wl.recency_blocks
        _check_select(dd, fmt, report, mode="topk", top_k=int(rng.integers(res, res + n_b + 2)))
        _check_select(dd, fmt, report, temperature=float(rng.choice([0.5, 2.0])))
    non_exact = [r for r in report if r[3] != "exact"]
    print("fuzz near-tie report:", non_exact)
    assert len(non_exact) <= max(2, len(report) // 10)


@pytest.mark.parametrize("chunk", range(3))
def test_fuzz_attention(torch_cuda, chunk):
    torch = torch_cuda
    rng = np.random.default_rng(777 + chunk)
    for case in range(1000 + chunk * 16, 1000 + chunk * 16 + 16):
        wl = _random_workload(rng, case, with_kv=True)
        dd = H.DeviceDecode(wl, "bf16")
        B, Hkv, D, Lc, blk = wl.B, wl.H_kv, wl.D, wl.L_cap, wl.blk
        layout = str(rng.choice(["hld", "lhd", "paged"]))
        if layout == "lhd":                               # [B][L][H_kv][D]
            dd.K = H.dev_u16(np.ascontiguousarray(wl.K.transpose(0, 2, 1, 3)))
            dd.V = H.dev_u16(np.ascontiguousarray(wl.V.transpose(0, 2, 1, 3)))
            dd.kv_strides = (Lc * Hkv * D, Hkv * D, D)
        elif layout == "paged":
            pt = int(rng.choice([16, 32, 64]))
            n_log = -(-Lc // pt)
            n_pages = B * n_log + 3
            table = rng.permutation(n_pages)[:B * n_log].reshape(B, n_log).astype(np.int32)
            poolK = np.zeros((n_pages, Hkv, pt, D), dtype=np.uint16)
            poolV = np.zeros((n_pages, Hkv, pt, D), dtype=np.uint16)
            for b in range(B):
                for lp in range(n_log):
                    t0, t1 = lp * pt, min((lp + 1) * pt, Lc)
                    poolK[table[b, lp], :, :t1 - t0] = wl.K[b, :, t0:t1]
                    poolV[table[b, lp], :, :t1 - t0] = wl.V[b, :, t0:t1]
            dd.K, dd.V = H.dev_u16(poolK), H.dev_u16(poolV)
            dd.kv_strides = (Hkv * pt * D, D, pt * D)
            dd.page_table = torch.from_numpy(table).cuda()
            dd.page_tokens = pt
        lists = []
        for b in range(B):
            n_b = -(-int(wl.seq_len[b]) // blk)
            k = int(rng.integers(0, n_b + 1))
            lists.append(sorted(rng.choice(n_b, size=k, replace=False).tolist()))
        # (an empty list is a legal row -- zeros out, lse = -inf, checked in test_block16_attention -- but the oracle
        # wants at least one block)
        lists = [x if x else [0] for x in lists]
        _check_attend(dd, lists)
        _check_attend(dd, [list(range(-(-int(L) // blk))) for L in wl.seq_len], dense=True)


@pytest.mark.parametrize("chunk", range(2))
def test_fuzz_prefill(torch_cuda, chunk):
    """Chunked prefill: random prompt length, chunk position and size, batch, GQA group, selector head dim, rule
    parameters and cache format; selection against the oracle, attention over the oracle's lists."""
    from tests.test_gpu_prefill import _check_attn_prefill, _check_select_prefill
    from workloads import make_prefill_workload
    rng = np.random.default_rng(31337 + chunk)
    for case in range(chunk * 6, chunk * 6 + 6):
        L = int(rng.choice([256, 640, 1024, 1536]))
        n_blk = L // 64
        qb0 = int(rng.integers(0, n_blk))
        nqb = int(rng.integers(1, min(n_blk - qb0, 6) + 1))
        B = int(rng.integers(1, 3))
        over = dict(p=float(rng.choice([0.5, 0.9, 1.0])), sink_blocks=int(rng.integers(0, 3)),
                    recency_blocks=int(rng.integers(0, 4)), kmin_blocks=int(rng.integers(0, 10)))
        if rng.random() < 0.25:
            over = dict(mode="topk", top_k=int(rng.integers(3, 12)), sink_blocks=1, recency_blocks=2)
        H_q = int(rng.choice([8, 32, 64]))
        d_idx = int(rng.choice([64, 128]))
        wls = [make_prefill_workload(seed=8000 + 13 * case + b, L=L, H_q=H_q, d_idx=d_idx,
                                     topic_span=int(rng.choice([64, 128, 256])))
               for b in range(B)]
        dp = H.DevicePrefill(wls, qb0 * 64, nqb * 64)
        fmt = str(rng.choice(["bf16", "bf16", "mxfp4", "fp8_e4m3"]))
        if case % 3 == 2:                    # round 2: the MXINT8 cache (dequantise pass) and the low-precision tensor-core forms
            fmt = ("mxint8", "mxfp4", "fp8_e4m3")[(case // 3) % 3]
        if fmt != "bf16":
            dp.set_cache_format(fmt)
            if case % 3 == 2 and fmt != "mxint8":
                dp.quantise_queries(fmt)     # q_fmt: MXFP4 x MXFP4 / FP8 x FP8 tile scores straight from the caches
        report = []
        _check_select_prefill(dp, report, **over)
        lists = [[sel.indices.tolist() for _, sel in H.oracle_select_prefill(w, dp.q_start, dp.Tq, **over)] for w in wls]
        paged = rng.random() < 0.4
        if paged:                                        # K/V as a page pool [page][H_kv][page_tokens][D]
            import torch
            pt = int(rng.choice([64, 128]))
            n_log = L // pt
            table = rng.permutation(B * n_log + 2)[:B * n_log].reshape(B, n_log).astype(np.int32)
            wl0 = wls[0]
            poolK = np.zeros((B * n_log + 2, wl0.H_kv, pt, wl0.D), dtype=np.uint16)
            poolV = np.zeros_like(poolK)
            for b, w in enumerate(wls):
                for lp in range(n_log):
                    poolK[table[b, lp]] = w.K[:, lp * pt:(lp + 1) * pt]
                    poolV[table[b, lp]] = w.V[:, lp * pt:(lp + 1) * pt]
            dp.K, dp.V = H.dev_u16(poolK), H.dev_u16(poolV)
            dp.kv_strides = (wl0.H_kv * pt * wl0.D, wl0.D, pt * wl0.D)
            dp.page_table, dp.page_tokens = torch.from_numpy(table).cuda(), pt
        _check_attn_prefill(dp, lists)
        print("fuzz prefill case %d: L=%d q_start=%d Tq=%d B=%d H_q=%d d_idx=%d %s%s near-ties %s"
              % (case, L, dp.q_start, dp.Tq, B, H_q, d_idx, fmt, " paged" if paged else "", report))


def test_fuzz_prefill_block16(torch_cuda):
    """f3: chunked prefill over 16-token key blocks -- random chunk geometries, reserved tiers, selector widths, cache
    formats, contiguous and paged K/V (recency >= 4 blocks keeps the whole diagonal 64 tokens in every list, so every
    query row sees at least itself)."""
    from tests.test_gpu_prefill import _check_attn_prefill, _check_select_prefill
    from workloads import make_prefill_workload
    rng = np.random.default_rng(1616)
    for case in range(8):
        L = int(rng.choice([256, 640, 1024, 1536]))
        n_blk = L // 64
        qb0 = int(rng.integers(0, n_blk))
        nqb = int(rng.integers(1, min(n_blk - qb0, 6) + 1))
        B = int(rng.integers(1, 3))
        over = dict(p=float(rng.choice([0.5, 0.9, 1.0])), sink_blocks=int(rng.integers(0, 9)),
                    recency_blocks=int(rng.integers(4, 17)), kmin_blocks=int(rng.integers(0, 40)))
        if rng.random() < 0.25:
            over = dict(mode="topk", top_k=int(rng.integers(24, 60)), sink_blocks=8, recency_blocks=16)
        H_q = int(rng.choice([8, 32, 64]))
        d_idx = int(rng.choice([64, 128]))
        wls = [make_prefill_workload(seed=16000 + 13 * case + b, L=L, H_q=H_q, d_idx=d_idx, blk=16,
                                     topic_span=int(rng.choice([64, 128, 256])))
               for b in range(B)]
        dp = H.DevicePrefill(wls, qb0 * 64, nqb * 64)
        fmt = str(rng.choice(["bf16", "bf16", "mxfp4", "fp8_e4m3"]))
        if case % 3 == 2:                    # round 2: the MXINT8 cache (dequantise pass) and the low-precision tensor-core forms
            fmt = ("mxint8", "mxfp4", "fp8_e4m3")[(case // 3) % 3]
        if fmt != "bf16":
            dp.set_cache_format(fmt)
            if case % 3 == 2 and fmt != "mxint8":
                dp.quantise_queries(fmt)     # q_fmt: MXFP4 x MXFP4 / FP8 x FP8 tile scores straight from the caches
        report = []
        _check_select_prefill(dp, report, **over)
        lists = [[sel.indices.tolist() for _, sel in H.oracle_select_prefill(w, dp.q_start, dp.Tq, **over)] for w in wls]
        paged = rng.random() < 0.4
        if paged:
            import torch
            pt = int(rng.choice([64, 128]))
            n_log = L // pt
            table = rng.permutation(B * n_log + 2)[:B * n_log].reshape(B, n_log).astype(np.int32)
            wl0 = wls[0]
            poolK = np.zeros((B * n_log + 2, wl0.H_kv, pt, wl0.D), dtype=np.uint16)
            poolV = np.zeros_like(poolK)
            for b, w in enumerate(wls):
                for lp in range(n_log):
                    poolK[table[b, lp]] = w.K[:, lp * pt:(lp + 1) * pt]
                    poolV[table[b, lp]] = w.V[:, lp * pt:(lp + 1) * pt]
            dp.K, dp.V = H.dev_u16(poolK), H.dev_u16(poolV)
            dp.kv_strides = (wl0.H_kv * pt * wl0.D, wl0.D, pt * wl0.D)
            dp.page_table, dp.page_tokens = torch.from_numpy(table).cuda(), pt
        _check_attn_prefill(dp, lists)
        print("fuzz prefill blk16 case %d: L=%d q_start=%d Tq=%d B=%d H_q=%d d_idx=%d %s%s near-ties %s"
              % (case, L, dp.q_start, dp.Tq, B, H_q, d_idx, fmt, " paged" if paged else "", report))
