"""GPU parity, chunked-prefill path (-m gpu): tcgen05 tile scoring (a1'), selection per query block (a2) and
block-sparse causal attention (a3') against the fp64 oracle on the same seeded bits.

Tile scores: fp32 tensor-core accumulation of exact BF16 products vs fp64 -> rtol/atol 2e-5.  Index lists and
budgets follow the decode protocol (exact, or a reported near-tie at the cut).  Attention: max-abs 2e-2 /
mean-abs 2e-3 on the oracle's selected set (BASELINE.json north_star)."""
import numpy as np
import pytest

from tests import _harness as H
from workloads import make_prefill_workload

pytestmark = pytest.mark.gpu

MAX_ABS, MEAN_ABS, PROB_ABS = 2e-2, 2e-3, 1e-3


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_22874_b200 import _lib
    _lib.load()
    return torch


def _neg_weights(wl, seed):
    """flip the sign of ~1/4 of the mixing weights (R13: w_h may be negative)"""
    rng = np.random.Generator(np.random.Philox(seed))
    flip = rng.random(wl.w.shape) < 0.25
    wl.w = np.where(flip, -wl.w, wl.w).astype(np.float32)
    return wl


def _check_select_prefill(dp, report, **over):
    idx, bud, scores, probs = dp.select(**over)
    p = over.get("p", dp.wl.p)
    mode = over.get("mode", dp.wl.mode)
    for b, wl in enumerate(dp.wls):
        ora = H.oracle_select_prefill(wl, dp.q_start, dp.Tq, **over)
        for i, (s_bar, sel) in enumerate(ora):
            row = b * dp.n_q + i
            n_b = len(s_bar)
            np.testing.assert_allclose(scores[row, :n_b], s_bar, rtol=2e-5, atol=2e-5,
                                       err_msg="tile scores, seq %d query block %d" % (b, i))
            cls = H.classify_selection(s_bar, sel, idx[row], int(bud[row]), p if mode == "dual_topp" else None)
            assert not cls.startswith("FAIL"), "seq %d query block %d: %s" % (b, i, cls)
            if cls != "exact":
                report.append((b, i, cls))
            assert np.all(idx[row, int(bud[row]):] == -1)
            if mode == "dual_topp" and cls == "exact":
                assert np.abs(probs[row, :n_b] - sel.probs).max() <= PROB_ABS
    return idx, bud


@pytest.mark.parametrize("L,q_start,Tq,B,over", [
    (1024, 0, 1024, 1, {}),                                   # whole prompt in one chunk
    (1024, 512, 320, 2, {}),                                  # later chunk, odd number of query blocks, batch of 2
    (4608, 0, 4608, 1, {}),                                   # 72 key blocks: three 32-block chunks per query tile
    (1024, 256, 256, 1, {"recency_blocks": 0, "sink_blocks": 0}),   # diagonal tile is residual: causal mask inside
    (1024, 0, 512, 1, {"mode": "topk", "top_k": 6}),
    (1024, 0, 64, 1, {"p": 1.0}),
])
def test_prefill_scores_and_selection(torch_cuda, L, q_start, Tq, B, over):
    wls = [_neg_weights(make_prefill_workload(seed=5005 + 7 * b, L=L, with_kv=False), 90 + b) for b in range(B)]
    dp = H.DevicePrefill(wls, q_start, Tq, with_kv=False)
    report = []
    _check_select_prefill(dp, report, **over)
    print("prefill select L=%d q_start=%d Tq=%d: %d near-tie rows %s" % (L, q_start, Tq, len(report), report[:4]))


def test_prefill_over_int4_with_bf16_scales_is_refused(torch_cuda):
    """R39: the keys of SPOT_SELK_INT4_BF16S are not BF16 numbers, and the prefill form would score their BF16 view --
    spot_select / spot_score_blocks say UNSUPPORTED for q_block = 64 instead of rounding silently."""
    torch = torch_cuda
    from paper_2606_22874_b200 import api
    wls = [make_prefill_workload(seed=6100, L=256, with_kv=False)]
    dp = H.DevicePrefill(wls, 0, 256, with_kv=False)
    dp.set_cache_format("mxint8")            # a cache of the right size class; the call must refuse before reading it
    dp.sel_k = torch.zeros(api.spot_selector_k_bytes("int4_bf16s", 1, 256, dp.wl.H_idx, dp.wl.d_idx), dtype=torch.uint8,
                           device="cuda")
    dp.fmt = "int4_bf16s"
    with pytest.raises(RuntimeError, match="UNSUPPORTED"):
        dp.select()


@pytest.mark.parametrize("fmt", ["mxfp4", "int4_e4m3", "fp8_e4m3", "mxint8"])
def test_prefill_selection_over_a_quantised_cache(torch_cuda, fmt):
    """f2: a later chunk (batch of 2, odd number of query blocks) scored against a quantised selector cache -- the
    library dequantises the visible prefix into its workspace and runs the BF16 tile-score GEMM; the oracle scores the
    oracle-quantised keys.  spot_score_blocks takes the same path and needs the same workspace."""
    torch = torch_cuda
    from paper_2606_22874_b200 import api
    wls = [_neg_weights(make_prefill_workload(seed=6006 + 7 * b, L=1024, with_kv=False), 70 + b) for b in range(2)]
    dp = H.DevicePrefill(wls, 512, 320, with_kv=False)
    dp.set_cache_format(fmt)
    report = []
    idx, bud = _check_select_prefill(dp, report)
    _check_select_prefill(dp, report, mode="topk", top_k=6)
    print("quantised prefill select (%s): near-tie rows %s" % (fmt, report[:4]))
    # score-only entry: same scores; too small a workspace is reported, not overrun
    wl = dp.wl
    nb_stride = (dp.n_b_max + 3) & ~3
    scores = torch.full((dp.B * dp.n_q, nb_stride), float("nan"), device="cuda")
    sp = api.make_select_params(dp.sel_q, dp.w, dp.sel_k, fmt, dp.L, None, 0, dp.B, dp.Tq, wl.H_idx, wl.d_idx,
                                q_start=dp.q_start, blk=wl.blk, q_block=wl.q_block, block_scores=scores,
                                nb_stride=nb_stride)
    with pytest.raises(RuntimeError, match="WORKSPACE"):
        api.spot_score_blocks(sp)
    # a score-only block (no indices / budgets / cap) sizes its own workspace: the dequantised prefix
    need = api.spot_select_workspace_bytes(sp)
    assert need >= dp.B * (dp.q_start + dp.Tq) * wl.H_idx * wl.d_idx * 2
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    sp.workspace, sp.workspace_bytes = ws.data_ptr(), ws.numel()
    api.spot_score_blocks(sp)
    torch.cuda.synchronize()
    got = scores.cpu().numpy()
    for b, w in enumerate(dp.wls):
        for i, (s_bar, _) in enumerate(H.oracle_select_prefill(w, dp.q_start, dp.Tq)):
            np.testing.assert_allclose(got[b * dp.n_q + i, :len(s_bar)], s_bar, rtol=2e-5, atol=2e-5)


@pytest.mark.parametrize("L,q_start,Tq,B", [(1024, 0, 1024, 1), (1024, 512, 320, 2), (4608, 0, 4608, 1), (1024, 256, 64, 1)])
def test_prefill_selection_with_the_papers_selector_width(torch_cuda, L, q_start, Tq, B):
    """d_idx = 128: a head is two 64-wide planes, the K ring is staged per head (4608 tokens: three
    32-block chunks per query tile, many trips around the 3-stage ring)."""
    wls = [_neg_weights(make_prefill_workload(seed=7007 + 7 * b, L=L, d_idx=128, with_kv=False), 50 + b) for b in range(B)]
    dp = H.DevicePrefill(wls, q_start, Tq, with_kv=False)
    report = []
    _check_select_prefill(dp, report)
    _check_select_prefill(dp, report, mode="topk", top_k=6)
    print("prefill select d_idx=128 L=%d q_start=%d Tq=%d: near-tie rows %s" % (L, q_start, Tq, report[:4]))


def _check_attn_prefill(dp, lists_per_seq, want_lse=False):
    """lists_per_seq[b][i] = selected key blocks of query block i of sequence b (the oracle's lists on both sides)."""
    wl = dp.wl
    rows = dp.B * dp.n_q
    cap = max(max(len(l) for l in ls) for ls in lists_per_seq)
    idx = np.full((rows, cap), -1, dtype=np.int32)
    bud = np.zeros(rows, dtype=np.int32)
    for b, ls in enumerate(lists_per_seq):
        for i, l in enumerate(ls):
            idx[b * dp.n_q + i, :len(l)] = l
            bud[b * dp.n_q + i] = len(l)
    out, lse = dp.attend(idx, bud, want_lse=want_lse)
    worst = (0.0, 0.0)
    for b, w in enumerate(dp.wls):
        want = H.oracle_attend_prefill(w, dp.q_start, dp.Tq, lists_per_seq[b])
        err = np.abs(out[b] - want)
        assert err.max() <= MAX_ABS and err.mean() <= MEAN_ABS, (b, err.max(), err.mean())
        worst = (max(worst[0], err.max()), max(worst[1], err.mean()))
    return out, lse, worst


@pytest.mark.parametrize("L,q_start,Tq,B,H_q,over", [
    (1024, 0, 256, 1, 32, {}),                     # first chunk: short lists, diagonal mask in every row
    (1024, 640, 192, 2, 32, {"p": 0.7}),           # later chunk, odd number of query blocks, batch of 2
    (1024, 512, 128, 1, 64, {}),                   # GQA 8: four 128-row tiles per KV head
    (1024, 768, 64, 1, 8, {"p": 1.0}),             # MHA-shaped group (G = 1, half of the tile idle), all blocks
])
def test_prefill_attention_on_oracle_lists(torch_cuda, L, q_start, Tq, B, H_q, over):
    wls = [make_prefill_workload(seed=5105 + 11 * b, L=L, H_q=H_q) for b in range(B)]
    dp = H.DevicePrefill(wls, q_start, Tq)
    lists = [[sel.indices.tolist() for _, sel in H.oracle_select_prefill(w, q_start, Tq, **over)] for w in wls]
    _, _, worst = _check_attn_prefill(dp, lists)
    print("prefill attn L=%d q_start=%d Tq=%d H_q=%d: max-abs %.2e mean-abs %.2e" % ((L, q_start, Tq, H_q) + worst))


def test_prefill_attention_all_blocks_is_dense_causal(torch_cuda):
    """indices == NULL (every visible block) and the explicit full lists both equal dense causal attention, which
    the oracle computes from the same definition with every block listed; LSE checked too."""
    L, q_start, Tq = 768, 256, 256
    wl = make_prefill_workload(seed=5205, L=L)
    dp = H.DevicePrefill([wl], q_start, Tq)
    full = [list(range((q_start + 64 * (i + 1) - 1) // 64 + 1)) for i in range(Tq // 64)]
    out_l, lse, _ = _check_attn_prefill(dp, [full], want_lse=True)
    # dense form through the same entry point
    import torch
    api = dp.api
    out = torch.zeros((1, Tq, wl.H_q, wl.D), dtype=torch.int16, device="cuda")
    ap = api.make_attn_params(dp.Q, dp.K, dp.V, dp.kv_strides, None, 0, None, None, 0, 1, Tq, wl.H_q, wl.H_kv, wl.D,
                              q_start=q_start, blk=wl.blk, sm_scale=wl.sm_scale, out=out)
    api.spot_sparse_attn_prefill(ap)
    torch.cuda.synchronize()
    got = H.bf16_bits_to_f64(H.to_np_u16(out))
    assert np.array_equal(got, out_l)
    # LSE against a direct fp64 evaluation for a few (query, head) pairs
    Kf = H.bf16_bits_to_f64(wl.K)
    Qf = H.bf16_bits_to_f64(wl.Q)
    G = wl.H_q // wl.H_kv
    for qq, h in [(0, 0), (63, 5), (100, 17), (255, 31)]:
        pos = q_start + qq
        logits = wl.sm_scale * (Kf[h // G, :pos + 1] @ Qf[pos, h])
        want = logits.max() + np.log(np.exp(logits - logits.max()).sum())
        assert abs(lse[0, qq, h] - want) <= 2e-3, (qq, h, lse[0, qq, h], want)


def test_prefill_attention_token_major_kv_layout(torch_cuda):
    """K/V as [B][L][H_kv][D] (strides passed) give the same bits as the head-major layout."""
    import torch
    L, q_start, Tq = 512, 256, 128
    wl = make_prefill_workload(seed=5305, L=L)
    dp = H.DevicePrefill([wl], q_start, Tq)
    lists = [sel.indices.tolist() for _, sel in H.oracle_select_prefill(wl, q_start, Tq)]
    out_hnd, _, _ = _check_attn_prefill(dp, [lists])
    Kt = dp.K.view(1, wl.H_kv, L, wl.D).permute(0, 2, 1, 3).contiguous()
    Vt = dp.V.view(1, wl.H_kv, L, wl.D).permute(0, 2, 1, 3).contiguous()
    dp.K, dp.V = Kt, Vt
    dp.kv_strides = (L * wl.H_kv * wl.D, wl.H_kv * wl.D, wl.D)
    out_nhd, _, _ = _check_attn_prefill(dp, [lists])
    assert np.array_equal(out_hnd, out_nhd)


def test_prefill_attention_argument_errors(torch_cuda):
    import torch
    from paper_2606_22874_b200 import api
    wl = make_prefill_workload(seed=5405, L=256)
    dp = H.DevicePrefill([wl], 0, 128)
    out = torch.zeros((1, 128, wl.H_q, wl.D), dtype=torch.int16, device="cuda")

    def params(**kw):
        base = dict(q_start=0, Tq=128)
        base.update(kw)
        return api.make_attn_params(dp.Q, dp.K, dp.V, dp.kv_strides, None, 0, None, None, 0, 1, base["Tq"], wl.H_q,
                                    wl.H_kv, wl.D, q_start=base["q_start"], blk=wl.blk, sm_scale=wl.sm_scale, out=out)
    for bad in (dict(q_start=32), dict(Tq=96)):                  # R26: chunk alignment
        with pytest.raises(api.SpotError) as e:
            api.spot_sparse_attn_prefill(params(**bad))
        assert "INVALID_ARG" in str(e.value)


def test_full_size_cfg5_in_the_bench_configuration(torch_cuda):
    """BASELINE.json config 5 at full size (L=65536, whole prompt as one chunk), launched as bench.py launches it.
    Sampled outputs the oracle can compute one by one: a seeded sample of 32 query blocks plus
    the first and the last -- for each, the whole selection row (tile scores, index list, budget) and the attention
    output over the oracle's list.  For attention the oracle runs on the gathered selected blocks with the query re-based
    onto the last of them (all other selected blocks are fully visible, so the causal structure is unchanged); the
    oracle's prefill attention costs ~1.5 s per (query, 32 heads) at a budget of 500 blocks, so the first two query blocks
    are checked on every query row and the others on four rows each (the block's first and last row -- the two ends of
    the diagonal mask -- and two seeded ones; eight rows for the last block), every head of each."""
    torch = torch_cuda
    from oracle import attention as OA
    from paper_2606_22874_b200 import api
    L = 65536
    n_qb = L // 64
    wl = make_prefill_workload(seed=5005, L=L, with_kv=False)
    dp = H.DevicePrefill([wl], 0, L, with_kv=False)
    idx, bud, scores, probs = dp.select(want_probs=False)
    rng = np.random.Generator(np.random.Philox(55005))
    sample = sorted(set([0, 1, n_qb - 1]) | set(rng.choice(np.arange(2, n_qb - 1), size=32, replace=False).tolist()))
    assert len(sample) >= 34
    full_rows = {0, 1}
    sels, near = {}, []
    for i in sample:
        (s_bar, sel), = H.oracle_select_prefill(wl, i * 64, 64)
        np.testing.assert_allclose(scores[i, :len(s_bar)], s_bar, rtol=2e-5, atol=2e-5)
        cls = H.classify_selection(s_bar, sel, idx[i], int(bud[i]), wl.p)
        assert not cls.startswith("FAIL"), "query block %d: %s" % (i, cls)
        if cls != "exact":
            near.append((i, cls))
        idx[i] = -1
        idx[i, :sel.budget] = sel.indices
        bud[i] = sel.budget
        sels[i] = sel
    print("cfg5: %d sampled query blocks, budgets %s, near-tie rows %s"
          % (len(sample), [sels[i].budget for i in sample], near))
    assert len(near) <= 1
    dev = torch.device("cuda")
    gen = torch.Generator(device=dev)
    gen.manual_seed(wl.seed + 17)
    Hq, Hkv, D = wl.H_q, wl.H_kv, wl.D
    Q = torch.randn((1, L, Hq, D), generator=gen, device=dev, dtype=torch.bfloat16)
    K = torch.randn((1, Hkv, L, D), generator=gen, device=dev, dtype=torch.bfloat16)
    V = torch.randn((1, Hkv, L, D), generator=gen, device=dev, dtype=torch.bfloat16)
    out = torch.zeros((1, L, Hq, D), dtype=torch.int16, device=dev)
    d_idx, d_bud = torch.from_numpy(idx).to(dev), torch.from_numpy(bud).to(dev)
    ap = api.make_attn_params(Q, K, V, (Hkv * L * D, D, L * D), None, 0, d_idx, d_bud, idx.shape[1], 1, L, Hq, Hkv, D,
                              q_start=0, blk=64, sm_scale=wl.sm_scale, out=out)
    api.spot_sparse_attn_prefill(ap)
    torch.cuda.synchronize()
    worst = (0.0, 0.0)
    for i in sample:
        blocks = sels[i].indices.astype(np.int64)
        assert blocks[-1] == i                                   # the diagonal block is reserved (recency tier)
        n = len(blocks)
        bl = torch.from_numpy(blocks).to(dev)
        Kg = K[0].view(Hkv, L // 64, 64, D)[:, bl].reshape(Hkv, n * 64, D)
        Vg = V[0].view(Hkv, L // 64, 64, D)[:, bl].reshape(Hkv, n * 64, D)
        Kh = H.bf16_bits_to_f64(H.to_np_u16(Kg.contiguous().view(torch.int16))).transpose(1, 0, 2)
        Vh = H.bf16_bits_to_f64(H.to_np_u16(Vg.contiguous().view(torch.int16))).transpose(1, 0, 2)
        Qh = H.bf16_bits_to_f64(H.to_np_u16(Q[0, i * 64:(i + 1) * 64].contiguous().view(torch.int16)))
        got = H.bf16_bits_to_f64(H.to_np_u16(out[0, i * 64:(i + 1) * 64]))
        if i in full_rows:
            want = OA.sparse_attn_prefill(Qh, Kh, Vh, [list(range(n))], (n - 1) * 64, 64, 64, wl.sm_scale)
            err = np.abs(got - want)
        else:
            extra = 6 if i == n_qb - 1 else 2
            rows = sorted({0, 63} | set(rng.choice(np.arange(1, 63), size=extra, replace=False).tolist()))
            # one query at a time: the oracle's prefill form with q_block = 1 at the query's (re-based) position
            want = np.stack([OA.sparse_attn_prefill(Qh[r:r + 1], Kh, Vh, [list(range(n))], (n - 1) * 64 + r, 1, 64,
                                                    wl.sm_scale)[0] for r in rows])
            err = np.abs(got[rows] - want)
        assert err.max() <= MAX_ABS and err.mean() <= MEAN_ABS, (i, err.max(), err.mean())
        worst = (max(worst[0], err.max()), max(worst[1], err.mean()))
    print("cfg5: attention over the oracle's lists of %d query blocks, worst max-abs %.2e mean-abs %.2e"
          % (len(sample), worst[0], worst[1]))


@pytest.mark.parametrize("page_tokens,layout", [(64, "phd"), (128, "pthd"), (256, "phd")])
def test_prefill_attention_over_paged_kv(torch_cuda, page_tokens, layout):
    """f3 / R32: K/V in a page pool shared by the batch behind a per-sequence page table (pages placed at random,
    finite garbage in the unused ones); the oracle reads the pool back through the table and attends as usual."""
    torch = torch_cuda
    from oracle import attention as OA
    L, q_start, Tq, B = 1024, 512, 320, 2
    wls = [make_prefill_workload(seed=9100 + 11 * b, L=L) for b in range(B)]
    dp = H.DevicePrefill(wls, q_start, Tq)
    wl = dp.wl
    pt, Hkv, D = page_tokens, wl.H_kv, wl.D
    n_log = L // pt
    rng = np.random.default_rng(41)
    n_pages = B * n_log + 5
    table = rng.permutation(n_pages)[:B * n_log].reshape(B, n_log).astype(np.int32)
    poolK = rng.integers(0, 1 << 16, size=(n_pages, pt, Hkv, D), dtype=np.uint16) & 0x3fff
    poolV = rng.integers(0, 1 << 16, size=(n_pages, pt, Hkv, D), dtype=np.uint16) & 0x3fff
    for b, w in enumerate(wls):
        Kb, Vb = w.K.transpose(1, 0, 2), w.V.transpose(1, 0, 2)                      # [L][H_kv][D]
        for lp in range(n_log):
            poolK[table[b, lp]] = Kb[lp * pt:(lp + 1) * pt]
            poolV[table[b, lp]] = Vb[lp * pt:(lp + 1) * pt]
        assert np.array_equal(OA.gather_paged_kv(poolK, table[b], L, pt), Kb)
        assert np.array_equal(OA.gather_paged_kv(poolV, table[b], L, pt), Vb)
    if layout == "phd":          # [page][H_kv][page_tokens][D]
        dp.K = H.dev_u16(np.ascontiguousarray(poolK.transpose(0, 2, 1, 3)))
        dp.V = H.dev_u16(np.ascontiguousarray(poolV.transpose(0, 2, 1, 3)))
        dp.kv_strides = (Hkv * pt * D, D, pt * D)
    else:                        # [page][page_tokens][H_kv][D]
        dp.K, dp.V = H.dev_u16(poolK), H.dev_u16(poolV)
        dp.kv_strides = (pt * Hkv * D, Hkv * D, D)
    dp.page_table = torch.from_numpy(table).cuda()
    dp.page_tokens = pt
    lists = [[sel.indices.tolist() for _, sel in H.oracle_select_prefill(w, q_start, Tq)] for w in wls]
    _check_attn_prefill(dp, lists)
    dense = [[list(range((q_start + 64 * i) // 64 + 1)) for i in range(Tq // 64)] for _ in wls]
    _check_attn_prefill(dp, dense)


# ---------------------------------------------------------------- f3: the paper's 16-token key blocks in prefill
F3 = dict(blk=16, sink_blocks=8, recency_blocks=16, kmin_blocks=32)


@pytest.mark.parametrize("L,q_start,Tq,B,d_idx,over", [
    (1024, 0, 1024, 1, 64, {}),
    (1024, 512, 320, 2, 64, {}),
    (4608, 0, 4608, 1, 64, {}),                                # 288 blocks per 64-key chunk boundary, three chunks
    (1024, 256, 256, 1, 128, {}),
    (1024, 256, 256, 1, 64, {"recency_blocks": 0, "sink_blocks": 0, "kmin_blocks": 0}),   # diagonal quarters residual
    (1024, 0, 512, 1, 64, {"mode": "topk", "top_k": 40}),
])
def test_prefill_block16_scores_and_selection(torch_cuda, L, q_start, Tq, B, d_idx, over):
    """Four tile scores per 64-key block (one per 16-token quarter, the causal mask applied token-wise inside the
    diagonal block), selection rows of 4x the entries, the paper's 8 / 16 / 32 reserved blocks."""
    wls = [_neg_weights(make_prefill_workload(seed=8008 + 7 * b, L=L, d_idx=d_idx, with_kv=False, **F3), 30 + b)
           for b in range(B)]
    dp = H.DevicePrefill(wls, q_start, Tq, with_kv=False)
    report = []
    _check_select_prefill(dp, report, **over)
    print("prefill blk16 select L=%d q_start=%d Tq=%d d_idx=%d: near-tie rows %s" % (L, q_start, Tq, d_idx, report[:4]))
    assert len(report) <= 1


def test_prefill_block16_selection_over_a_quantised_cache(torch_cuda):
    wls = [_neg_weights(make_prefill_workload(seed=8108, L=1024, with_kv=False, **F3), 31)]
    dp = H.DevicePrefill(wls, 512, 320, with_kv=False)
    dp.set_cache_format("mxfp4")
    report = []
    _check_select_prefill(dp, report)
    assert len(report) <= 1


def test_prefill_block16_attention(torch_cuda):
    """Block-sparse causal attention over lists of 16-token blocks: the oracle's lists (a later chunk, batch of 2), dense
    (indices NULL), and hand-made lists -- tiles that are not full (lists of 1, 3, 9, 17 entries), entries that lie wholly
    in the future of the first rows of the query block (quarters 1-3 of the diagonal block without quarter 0), a list
    whose only past block is the sink."""
    L, q_start, Tq, B = 1024, 512, 320, 2
    wls = [make_prefill_workload(seed=8208 + 11 * b, L=L, **F3) for b in range(B)]
    dp = H.DevicePrefill(wls, q_start, Tq)
    lists = [[sel.indices.tolist() for _, sel in H.oracle_select_prefill(w, q_start, Tq)] for w in wls]
    _check_attn_prefill(dp, lists, want_lse=True)
    n_q = Tq // 64
    dense = [[list(range(((q_start + 64 * (i + 1)) // 16))) for i in range(n_q)] for _ in wls]
    _check_attn_prefill(dp, dense)
    out_dense, _, _ = _check_attn_prefill_indices_none(dp, dense)
    d0 = lambda i: (q_start + 64 * i) // 16                     # first 16-token block of query block i's diagonal
    hand = [[[0], [0, 5, d0(1) + 1], [0, 1, 2, 3, 9, 10, 11, d0(2) + 1, d0(2) + 3],
             [0] + list(range(17, 32)) + [d0(3) + 2], [0, d0(4), d0(4) + 1, d0(4) + 2, d0(4) + 3]] for _ in wls]
    _check_attn_prefill(dp, hand)


def _check_attn_prefill_indices_none(dp, dense_lists):
    """indices == NULL (every causally visible block) must equal the explicit dense lists bit for bit."""
    import torch
    wl, api = dp.wl, dp.api
    out = torch.zeros((dp.B, dp.Tq, wl.H_q, wl.D), dtype=torch.int16, device="cuda")
    ap = api.make_attn_params(dp.Q, dp.K, dp.V, dp.kv_strides, None, 0, None, None, 0, dp.B, dp.Tq, wl.H_q, wl.H_kv, wl.D,
                              q_start=dp.q_start, blk=wl.blk, sm_scale=wl.sm_scale, out=out)
    api.spot_sparse_attn_prefill(ap)
    torch.cuda.synchronize()
    rows = dp.B * dp.n_q
    cap = max(max(len(l) for l in ls) for ls in dense_lists)
    idx = np.full((rows, cap), -1, dtype=np.int32)
    bud = np.zeros(rows, dtype=np.int32)
    for b, ls in enumerate(dense_lists):
        for i, l in enumerate(ls):
            idx[b * dp.n_q + i, :len(l)] = l
            bud[b * dp.n_q + i] = len(l)
    want, _ = dp.attend(idx, bud)
    got = H.bf16_bits_to_f64(H.to_np_u16(out))
    assert np.array_equal(got, want)
    return got, None, None


def test_prefill_block16_attention_over_paged_kv(torch_cuda):
    torch = torch_cuda
    L, q_start, Tq = 1024, 256, 256
    wl = make_prefill_workload(seed=8308, L=L, **F3)
    dp = H.DevicePrefill([wl], q_start, Tq)
    lists = [[sel.indices.tolist() for _, sel in H.oracle_select_prefill(wl, q_start, Tq)]]
    _check_attn_prefill(dp, lists)
    pt, Hkv, D = 64, wl.H_kv, wl.D
    n_log = L // pt
    rng = np.random.default_rng(43)
    table = rng.permutation(n_log + 3)[:n_log].reshape(1, n_log).astype(np.int32)
    poolK = rng.integers(0, 1 << 16, size=(n_log + 3, Hkv, pt, D), dtype=np.uint16) & 0x3fff
    poolV = rng.integers(0, 1 << 16, size=(n_log + 3, Hkv, pt, D), dtype=np.uint16) & 0x3fff
    for lp in range(n_log):
        poolK[table[0, lp]] = wl.K[:, lp * pt:(lp + 1) * pt]
        poolV[table[0, lp]] = wl.V[:, lp * pt:(lp + 1) * pt]
    dp.K, dp.V = H.dev_u16(poolK), H.dev_u16(poolV)
    dp.kv_strides = (Hkv * pt * D, D, pt * D)
    dp.page_table, dp.page_tokens = torch.from_numpy(table).cuda(), pt
    _check_attn_prefill(dp, lists)


# ---------------------------------------------------------------- f2: FP8 x FP8 tile scores on the tensor cores
@pytest.mark.parametrize("d_idx,L,q_start,Tq,B,blk", [(64, 1024, 0, 1024, 1, 64), (128, 1024, 512, 320, 2, 64),
                                                      (128, 4608, 0, 4608, 1, 64), (64, 1024, 256, 256, 1, 16)])
def test_prefill_fp8_queries_and_keys_on_the_tensor_cores(torch_cuda, d_idx, L, q_start, Tq, B, blk):
    """PAPER.md:115 / :186 quantise the selector's queries as well as its key cache.  With both in FP8-E4M3 the tile
    scores are FP8 x FP8 products accumulated in fp32 by tcgen05.mma kind::f8f6f4 straight from the cache layout (q_fmt):
    no dequantise pass.  The oracle scores the two dequantised images (R33).  Every product of two E4M3 values has at most
    8 significant bits, so the products are exact and the only error is the fp32 accumulation over d_idx -- the same
    2e-5 tolerance as the BF16 GEMM, and exact index lists."""
    geo = dict(blk=16, sink_blocks=8, recency_blocks=16, kmin_blocks=32) if blk == 16 else {}
    wls = [_neg_weights(make_prefill_workload(seed=6606 + 7 * b, L=L, d_idx=d_idx, with_kv=False, **geo), 60 + b)
           for b in range(B)]
    dp = H.DevicePrefill(wls, q_start, Tq, with_kv=False)
    dp.set_cache_format("fp8_e4m3")
    dp.quantise_queries("fp8_e4m3")
    report = []
    _check_select_prefill(dp, report)
    _check_select_prefill(dp, report, mode="topk", top_k=40 if blk == 16 else 6)
    print("fp8 x fp8 prefill select d_idx=%d L=%d: near-tie rows %s" % (d_idx, L, report[:4]))
    assert len(report) <= 1


# ---------------------------------------------------------------- f2: MXFP4 x MXFP4 block-scaled tile scores
@pytest.mark.parametrize("d_idx,L,q_start,Tq,B,blk", [(64, 1024, 0, 1024, 1, 64), (128, 1024, 512, 320, 2, 64),
                                                      (128, 4608, 0, 4608, 1, 64), (64, 1024, 256, 256, 1, 16),
                                                      (64, 2112, 1024, 1088, 2, 64), (128, 448, 0, 448, 3, 16)])
def test_prefill_mxfp4_queries_and_keys_block_scaled_on_the_tensor_cores(torch_cuda, d_idx, L, q_start, Tq, B, blk):
    """PAPER.md:115 / :184-188: queries and key cache in FP4 "group-32 microscale".  With both in MXFP4 the tile scores are
    E2M1 x E2M1 products times the two groups' UE8M0 scales, accumulated in fp32 by tcgen05.mma kind::mxf4.block_scale
    straight from the opaque cache layout (q_fmt = mxfp4): no dequantise pass, the scales go through tensor memory.  The
    oracle scores the two dequantised images (R33).  Products and power-of-two scales are exact; the error is the fp32
    accumulation over d_idx terms -- the BF16 GEMM's 2e-5 tolerance, exact index lists.  Odd numbers of query blocks and of
    visible key blocks exercise the half-filled tiles (scale rows that are never loaded must stay out of every result)."""
    geo = dict(blk=16, sink_blocks=8, recency_blocks=16, kmin_blocks=32) if blk == 16 else {}
    wls = [_neg_weights(make_prefill_workload(seed=6806 + 7 * b, L=L, d_idx=d_idx, with_kv=False, **geo), 50 + b)
           for b in range(B)]
    dp = H.DevicePrefill(wls, q_start, Tq, with_kv=False)
    dp.set_cache_format("mxfp4")
    dp.quantise_queries("mxfp4")
    report = []
    _check_select_prefill(dp, report)
    _check_select_prefill(dp, report, mode="topk", top_k=40 if blk == 16 else 6)
    print("mxfp4 x mxfp4 prefill select d_idx=%d L=%d: near-tie rows %s" % (d_idx, L, report[:4]))
    assert len(report) <= 1


@pytest.mark.parametrize("fmt,d_idx", [("mxfp4", 64), ("mxfp4", 128), ("fp8_e4m3", 128)])
def test_full_size_cfg5_low_precision_tile_scores(torch_cuda, fmt, d_idx):
    """The low-precision tensor-core forms of the tile-score GEMM at config 5's full size (L = 65536, one chunk), launched as
    `bench.py --workload cfg5 --fmt X --qfmt X` launches them: a seeded sample of query blocks (the first two, the last, an odd
    one and five others), each checked on its whole selection row -- tile scores at 2e-5 and the index list / budget against
    the oracle run on the two dequantised images (R33)."""
    L = 65536
    n_qb = L // 64
    wl = make_prefill_workload(seed=5005, L=L, d_idx=d_idx, with_kv=False)
    dp = H.DevicePrefill([wl], 0, L, with_kv=False)
    dp.set_cache_format(fmt)
    dp.quantise_queries(fmt)
    idx, bud, scores, probs = dp.select(want_probs=False)
    rng = np.random.Generator(np.random.Philox(65005 + d_idx))
    sample = sorted(set([0, 1, 513, n_qb - 1]) | set(rng.choice(np.arange(2, n_qb - 1), size=5, replace=False).tolist()))
    near = []
    for i in sample:
        (s_bar, sel), = H.oracle_select_prefill(wl, i * 64, 64)
        np.testing.assert_allclose(scores[i, :len(s_bar)], s_bar, rtol=2e-5, atol=2e-5)
        cls = H.classify_selection(s_bar, sel, idx[i], int(bud[i]), wl.p)
        assert not cls.startswith("FAIL"), "query block %d: %s" % (i, cls)
        if cls != "exact":
            near.append((i, cls))
    print("cfg5 %s x %s d_idx %d: %d sampled query blocks, near-tie rows %s" % (fmt, fmt, d_idx, len(sample), near))
    assert len(near) <= 1


def test_q_fmt_argument_errors(torch_cuda):
    """spot.h, q_fmt: FP8 queries need an FP8 cache and the prefill form; any other value is an invalid argument.  Nothing
    is written to the outputs by a refused call."""
    from paper_2606_22874_b200 import api
    wl = make_prefill_workload(seed=6707, L=256, with_kv=False)
    dp = H.DevicePrefill([wl], 0, 128, with_kv=False)
    dp.q_fmt = "fp8_e4m3"                                         # BF16 cache, FP8 query flag
    with pytest.raises(api.SpotError) as e:
        dp.select()
    assert "UNSUPPORTED" in str(e.value)
    dp.set_cache_format("mxfp4")
    with pytest.raises(api.SpotError) as e:
        dp.select()
    assert "UNSUPPORTED" in str(e.value)
    dp.set_cache_format("fp8_e4m3")
    dp.q_fmt = "mxfp4"
    with pytest.raises(api.SpotError) as e:
        dp.select()
    assert "UNSUPPORTED" in str(e.value) or "INVALID_ARG" in str(e.value)
    import torch
    scores = torch.zeros((2, 4), dtype=torch.float32, device="cuda")
    sp = api.make_select_params(dp.sel_q, dp.w, dp.sel_k, "fp8_e4m3", 256, None, 0, 1, 128, wl.H_idx, wl.d_idx,
                                q_start=0, blk=wl.blk, q_block=64, mode=wl.mode, p=wl.p, block_scores=scores, nb_stride=4)
    sp.q_fmt = 77
    with pytest.raises(api.SpotError) as e:
        api.spot_score_blocks(sp)
    assert "INVALID_ARG" in str(e.value)
    # the decode form takes BF16 queries only
    sp = api.make_select_params(dp.sel_q, dp.w, dp.sel_k, "fp8_e4m3", 256, None, 0, 1, 1, wl.H_idx, wl.d_idx,
                                blk=wl.blk, q_block=1, q_fmt="fp8_e4m3", mode=wl.mode, p=wl.p, block_scores=scores,
                                nb_stride=4)
    with pytest.raises(api.SpotError) as e:
        api.spot_score_blocks(sp)
    assert "UNSUPPORTED" in str(e.value)
    assert float(scores.abs().sum()) == 0.0
