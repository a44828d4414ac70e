"""Tiny invocations of every kernel family, for compute-sanitizer (memcheck / racecheck / synccheck) on the GPU box:

    compute-sanitizer --tool <tool> python tests/sanitize_smoke.py [decode|prefill|all]

decode : one spot_decode_step (score -> select -> attend -> merge, the pipelined launch) and the separate calls, for every
         selector-cache format, 64- and 16-token blocks, contiguous and paged K/V, the dense comparator, the quantisers and
         the projection + append step;
prefill: one chunk of tcgen05 tile scoring + selection + block-sparse causal attention for d_idx 64 and 128, a quantised
         cache (dequantise pass), contiguous and paged K/V.
guarded: the decode step with every written buffer between canary guard bands, and run-to-run bit equality (what is
         left to check with when compute-sanitizer is unavailable).
Sizes are a few tiles (the tools slow kernels down 10-100x); results are checked for finiteness only -- parity is the
job of the pytest suite.  Exit code 0 = every call returned SPOT_OK and produced finite output."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def decode_cases():
    import torch
    from paper_2606_22874_b200 import api
    from tests import _harness as H
    from workloads import make_decode_workload
    F3 = dict(blk=16, sink_blocks=8, recency_blocks=16, kmin_blocks=32)
    for fmt in ("bf16", "mxfp4", "int4_e4m3", "fp8_e4m3", "mxint8", "int4_bf16s"):
        for over in ({}, F3):
            wl = make_decode_workload("san", 7, B=3, L=1280, kind="zipf", seq_lens=[1280, 1000, 333], **over)
            dd = H.DeviceDecode(wl, fmt)
            dp = dd.step_params(garbage=0x3C)
            api.spot_decode_step(dp)
            api.spot_decode_step(dp)
            idx, bud, out, lse = dd.step_results()
            assert np.isfinite(out).all() and (bud > 0).all(), (fmt, over)
            idx2, bud2, _, _ = dd.select()
            assert np.array_equal(bud, bud2)
            out2, _ = dd.attend(idx2, bud2)
            assert np.isfinite(out2).all()
            print("decode", fmt, "blk", wl.blk, "budgets", bud.tolist())
    # d_idx 128, dense comparator, paged K/V
    wl = make_decode_workload("san128", 9, B=2, L=640, kind="zipf", seq_lens=[640, 600], d_idx=128)
    for fmt in ("bf16", "mxfp4"):
        dd = H.DeviceDecode(wl, fmt)
        dp = dd.step_params()
        api.spot_decode_step(dp)
        idx, bud, out, _ = dd.step_results()
        assert np.isfinite(out).all()
    dd = H.DeviceDecode(wl, "bf16")
    out, _ = dd.attend(dense=True)
    assert np.isfinite(out).all()
    pt, B, Hkv, D, Lc = 64, wl.B, wl.H_kv, wl.D, wl.L_cap
    n_log = Lc // pt
    table = np.random.default_rng(3).permutation(B * n_log).reshape(B, n_log).astype(np.int32)
    pool = np.zeros((B * n_log, Hkv, pt, D), dtype=np.uint16)
    poolv = np.zeros_like(pool)
    for b in range(B):
        for lp in range(n_log):
            pool[table[b, lp]] = wl.K[b][:, lp * pt:(lp + 1) * pt]
            poolv[table[b, lp]] = wl.V[b][:, lp * pt:(lp + 1) * pt]
    dd.K, dd.V = H.dev_u16(pool), H.dev_u16(poolv)
    dd.kv_strides = (Hkv * pt * D, D, pt * D)
    dd.page_table, dd.page_tokens = torch.from_numpy(table).cuda(), pt
    dp = dd.step_params()
    api.spot_decode_step(dp)
    _, bud, out, _ = dd.step_results()
    assert np.isfinite(out).all()
    print("decode d_idx 128 / dense / paged ok")
    # projection + RoPE + append (f1)
    from workloads import make_project_workload
    pw = make_project_workload(seed=5, B=2, d_model=512, H_idx=4, d_idx=64, L=128)
    dev = {k: H.dev_u16(pw[k]) for k in ("hidden", "w_q", "w_k", "w_w")}
    pos = torch.tensor([5, 77], dtype=torch.int32, device="cuda")
    for fmt in ("bf16", "mxfp4", "fp8_e4m3"):
        cache = torch.zeros(api.spot_selector_k_bytes(fmt, 2, 128, 4, 64), dtype=torch.uint8, device="cuda")
        sq = torch.zeros((2, 4, 64), dtype=torch.int16, device="cuda")
        ww = torch.zeros((2, 4), device="cuda")
        pp = api.make_project_params(dev["hidden"], dev["w_q"], dev["w_k"], dev["w_w"], pos, 2, 512, 4, 64, rope_dims=64,
                                     rope_base=1e6, sel_q=sq, w=ww, sel_k=cache, fmt=fmt, cache_stride_tokens=128)
        ws = torch.empty(max(16, api.spot_selector_project_append_workspace_bytes(pp)), dtype=torch.uint8, device="cuda")
        pp.workspace, pp.workspace_bytes = ws.data_ptr(), ws.numel()
        api.spot_selector_project_append(pp)
        torch.cuda.synchronize()
        assert torch.isfinite(ww).all()
    print("project + append ok")


def prefill_cases():
    import torch
    from tests import _harness as H
    from workloads import make_prefill_workload
    for d_idx, fmt in ((64, "bf16"), (128, "bf16"), (64, "mxfp4")):
        wl = make_prefill_workload(seed=31 + d_idx, L=512, d_idx=d_idx)
        dp = H.DevicePrefill([wl], 128, 256)
        if fmt != "bf16":
            dp.set_cache_format(fmt)
        idx, bud, scores, _ = dp.select()
        assert (bud > 0).all() and np.isfinite(scores[:, :2]).all()
        out, _ = dp.attend(idx, bud, want_lse=True)
        assert np.isfinite(out).all()
        print("prefill d_idx", d_idx, fmt, "budgets", bud.tolist())
    wl = make_prefill_workload(seed=77, L=512)
    dp = H.DevicePrefill([wl], 0, 256)
    idx, bud, _, _ = dp.select()
    pt, Hkv, D, L = 64, wl.H_kv, wl.D, 512
    table = np.random.default_rng(4).permutation(L // pt).reshape(1, L // pt).astype(np.int32)
    pool = np.zeros((L // pt, Hkv, pt, D), dtype=np.uint16)
    poolv = np.zeros_like(pool)
    for lp in range(L // pt):
        pool[table[0, lp]] = wl.K[:, lp * pt:(lp + 1) * pt]
        poolv[table[0, lp]] = wl.V[:, lp * pt:(lp + 1) * pt]
    dp.K, dp.V = H.dev_u16(pool), H.dev_u16(poolv)
    dp.kv_strides = (Hkv * pt * D, D, pt * D)
    dp.page_table, dp.page_tokens = torch.from_numpy(table).cuda(), pt
    out, _ = dp.attend(idx, bud)
    assert np.isfinite(out).all()
    print("prefill paged ok")


class Arena:
    """Guard bands by hand (compute-sanitizer is closed on this GPU pool): every buffer a kernel WRITES is carved out of one
    arena filled with a canary pattern, 64 KiB of canary on both sides; check() fails if any guard byte changed."""
    PAD = 64 << 10

    def __init__(self, nbytes):
        import torch
        self.buf = torch.full((nbytes,), 0xC5, dtype=torch.uint8, device="cuda")
        self.off, self.spans = self.PAD, []

    def take(self, nbytes, dtype, shape):
        import torch
        n = (nbytes + 255) & ~255
        view = self.buf[self.off:self.off + nbytes]
        self.spans.append((self.off, self.off + nbytes))
        self.off += n + self.PAD
        assert self.off <= self.buf.numel()
        return view.view(dtype).reshape(shape)

    def check(self, what):
        import torch
        keep = torch.ones(self.buf.numel(), dtype=torch.bool, device="cuda")
        for a, b in self.spans:
            keep[a:b] = False
        bad = int(((self.buf != 0xC5) & keep).sum())
        assert bad == 0, "%s: %d guard bytes overwritten" % (what, bad)


def guarded_cases():
    """Out-of-bounds WRITES: the decode step and the prefill pass with every output and workspace between guard bands;
    and run-to-run determinism (a data race would show as differing bits): every case three times, bit-equal."""
    import torch
    from paper_2606_22874_b200 import api
    from tests import _harness as H
    from workloads import make_decode_workload, make_prefill_workload
    for fmt, over in (("bf16", {}), ("mxfp4", {}), ("int4_e4m3", dict(blk=16, sink_blocks=8, recency_blocks=16, kmin_blocks=32)),
                      ("fp8_e4m3", {}), ("mxint8", {}), ("int4_bf16s", dict(blk=16, sink_blocks=8, recency_blocks=16, kmin_blocks=32))):
        wl = make_decode_workload("guard", 13, B=5, L=2048 + 64, kind="zipf", seq_lens=[2112, 2048, 1999, 65, 1], **over)
        dd = H.DeviceDecode(wl, fmt)
        dp = dd.step_params()
        ar = Arena(64 << 20)
        B, cap = wl.B, dd.cap
        dd.indices = ar.take(B * cap * 4, torch.int32, (B, cap))
        dd.budgets = ar.take(B * 4, torch.int32, (B,))
        dd.out = ar.take(B * wl.H_q * wl.D * 2, torch.int16, (B, wl.H_q, wl.D))
        dd.lse = ar.take(B * wl.H_q * 4, torch.float32, (B, wl.H_q))
        ws_sel = ar.take(dd.ws_sel.numel(), torch.uint8, (dd.ws_sel.numel(),))
        ws_att = ar.take(dd.ws_att.numel(), torch.uint8, (dd.ws_att.numel(),))
        ws_step = ar.take(dd.ws_step.numel(), torch.uint8, (dd.ws_step.numel(),))
        for blk_ in (dp.select, dp.attn):
            blk_.indices, blk_.budgets = dd.indices.data_ptr(), dd.budgets.data_ptr()
        dp.attn.out, dp.attn.lse = dd.out.data_ptr(), dd.lse.data_ptr()
        dp.select.workspace, dp.attn.workspace, dp.workspace = ws_sel.data_ptr(), ws_att.data_ptr(), ws_step.data_ptr()
        runs = []
        for _ in range(3):
            api.spot_decode_step(dp)
            torch.cuda.synchronize()
            runs.append((dd.indices.clone(), dd.budgets.clone(), dd.out.clone()))
        ar.check("decode step %s blk %d" % (fmt, wl.blk))
        for r in runs[1:]:
            assert all(torch.equal(x, y) for x, y in zip(r, runs[0])), "decode step %s: runs differ" % fmt
        print("guarded decode step", fmt, "blk", wl.blk, "ok, budgets", dd.budgets.tolist())
    for d_idx, qfmt in ((64, None), (128, None), (64, "mxfp4"), (128, "mxfp4"), (128, "fp8_e4m3")):
        wl = make_prefill_workload(seed=90 + d_idx, L=1024, d_idx=d_idx)
        dpf = H.DevicePrefill([wl], 256, 448)
        if qfmt:                              # low-precision tensor-core tile scores: quantised cache AND queries (q_fmt)
            dpf.set_cache_format(qfmt)
            dpf.quantise_queries(qfmt)
        outs = []
        for _ in range(3):
            idx, bud, scores, _ = dpf.select()
            out, lse = dpf.attend(idx, bud, want_lse=True)
            outs.append((idx.copy(), bud.copy(), scores[:, :4].copy(), out.copy()))
        for r in outs[1:]:
            assert all(np.array_equal(x, y) for x, y in zip(r, outs[0])), "prefill d_idx %d %s: runs differ" % (d_idx, qfmt)
        print("deterministic prefill d_idx", d_idx, qfmt or "bf16", "ok")


if __name__ == "__main__":
    what = sys.argv[1] if len(sys.argv) > 1 else "all"
    from paper_2606_22874_b200 import _lib
    _lib.load()
    if what in ("decode", "all"):
        decode_cases()
    if what in ("prefill", "all"):
        prefill_cases()
    if what in ("guarded", "all"):
        guarded_cases()
    print("sanitize_smoke: ok")
