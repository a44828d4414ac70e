"""Test-side glue: moves a seeded workload to the GPU, calls the C ABI through the Python binding, and runs the
fp64 oracle on the same bits.  Holds the parity protocol for index lists."""
import numpy as np

from oracle import attention as OA
from oracle import quant as OQ
from oracle import selection as OS
from oracle.bf16 import bf16_bits_to_f64, f64_to_bf16_bits_exact


def dev_u16(arr):
    import torch
    return torch.from_numpy(np.ascontiguousarray(arr).view(np.int16)).cuda()


def to_np_u16(t):
    return t.cpu().numpy().view(np.uint16)


class DeviceDecode:
    """A DecodeWorkload resident on the GPU, selector cache in one format."""

    def __init__(self, wl, fmt="bf16", with_kv=True):
        import torch
        from paper_2606_22874_b200 import api
        self.wl, self.fmt, self.api = wl, fmt, api
        self.sel_q = dev_u16(wl.sel_q)
        self.w = torch.from_numpy(wl.w).cuda()
        self.seq_len = torch.from_numpy(wl.seq_len).cuda()
        self.max_seq_len = int(wl.seq_len.max())
        self.L_cap = wl.L_cap
        sel_k_bf16 = dev_u16(wl.sel_k)
        if fmt == "bf16":
            self.sel_k = sel_k_bf16
        else:
            assert wl.L_cap % 64 == 0
            nbytes = api.spot_selector_k_bytes(fmt, wl.B, wl.L_cap, wl.H_idx, wl.d_idx)
            self.sel_k = torch.zeros(nbytes, dtype=torch.uint8, device="cuda")
            api.spot_quantize_selector_k(sel_k_bf16, self.sel_k, fmt, wl.B, wl.L_cap, 0, wl.L_cap, wl.H_idx, wl.d_idx)
        if with_kv and wl.K is not None:
            self.q = dev_u16(wl.q)
            self.K = dev_u16(wl.K)
            self.V = dev_u16(wl.V)
            self.kv_strides = (wl.H_kv * wl.L_cap * wl.D, wl.D, wl.L_cap * wl.D)   # [B][H_kv][L][D]
        self.n_b_max = -(-self.max_seq_len // wl.blk)

    def select(self, cap=None, want_scores=True, want_probs=True, **over):
        import torch
        wl, api = self.wl, self.api
        kw = dict(mode=wl.mode, top_k=wl.top_k, p=wl.p, sink_blocks=wl.sink_blocks,
                  recency_blocks=wl.recency_blocks, kmin_blocks=wl.kmin_blocks, temperature=wl.temperature)
        kw.update(over)
        cap = self.n_b_max if cap is None else cap
        self.cap = cap
        self.indices = torch.full((wl.B, cap), -7, dtype=torch.int32, device="cuda")
        self.budgets = torch.full((wl.B,), -7, dtype=torch.int32, device="cuda")
        nb_stride = (self.n_b_max + 3) & ~3
        scores = torch.full((wl.B, nb_stride), float("nan"), device="cuda") if want_scores else None
        probs = torch.full((wl.B, nb_stride), float("nan"), device="cuda") if want_probs else None
        sp = api.make_select_params(self.sel_q, self.w, self.sel_k, self.fmt, self.L_cap, self.seq_len,
                                    self.max_seq_len, wl.B, 1, wl.H_idx, wl.d_idx, blk=wl.blk, q_block=1,
                                    indices=self.indices, cap=cap, budgets=self.budgets, block_scores=scores,
                                    block_probs=probs, nb_stride=nb_stride, **kw)
        ws = torch.empty(max(api.spot_select_workspace_bytes(sp), 16), dtype=torch.uint8, device="cuda")
        sp.workspace, sp.workspace_bytes = ws.data_ptr(), ws.numel()
        api.spot_select(sp)
        torch.cuda.synchronize()
        return (self.indices.cpu().numpy(), self.budgets.cpu().numpy(),
                None if scores is None else scores.cpu().numpy(), None if probs is None else probs.cpu().numpy())

    def attend(self, indices_np=None, budgets_np=None, dense=False, want_lse=True):
        import torch
        wl, api = self.wl, self.api
        out = torch.zeros((wl.B, wl.H_q, wl.D), dtype=torch.int16, device="cuda")
        lse = torch.zeros((wl.B, wl.H_q), device="cuda") if want_lse else None
        if dense:
            idx = bud = None
            cap = 0
        else:
            idx = torch.from_numpy(np.ascontiguousarray(indices_np, dtype=np.int32)).cuda()
            bud = torch.from_numpy(np.ascontiguousarray(budgets_np, dtype=np.int32)).cuda()
            cap = idx.shape[1]
        ap = api.make_attn_params(self.q, self.K, self.V, self.kv_strides, self.seq_len, self.max_seq_len, idx, bud,
                                  cap, wl.B, 1, wl.H_q, wl.H_kv, wl.D, blk=wl.blk, sm_scale=wl.sm_scale, out=out,
                                  lse=lse, page_table=getattr(self, "page_table", None),
                                  page_tokens=getattr(self, "page_tokens", 0))
        fn_ws = api.spot_dense_attn_decode_workspace_bytes if dense else api.spot_sparse_attn_decode_workspace_bytes
        ws = torch.empty(max(fn_ws(ap), 16), dtype=torch.uint8, device="cuda")
        ap.workspace, ap.workspace_bytes = ws.data_ptr(), ws.numel()
        (api.spot_dense_attn_decode if dense else api.spot_sparse_attn_decode)(ap)
        torch.cuda.synchronize()
        return bf16_bits_to_f64(to_np_u16(out)), (None if lse is None else lse.cpu().numpy())


    def step_params(self, cap=None, garbage=None, want_lse=True, **over):
        """Parameter block of spot_decode_step (a1 + a2 + a3 in one call) over this workload, with every buffer it
        needs kept alive on `self`.  garbage: byte value the workspaces are filled with first (they need not be
        initialised)."""
        import torch
        wl, api = self.wl, self.api
        kw = dict(mode=wl.mode, top_k=wl.top_k, p=wl.p, sink_blocks=wl.sink_blocks,
                  recency_blocks=wl.recency_blocks, kmin_blocks=wl.kmin_blocks, temperature=wl.temperature)
        kw.update(over)
        cap = self.n_b_max if cap is None else cap
        self.cap = cap
        self.indices = torch.full((wl.B, cap), -7, dtype=torch.int32, device="cuda")
        self.budgets = torch.full((wl.B,), -7, dtype=torch.int32, device="cuda")
        self.out = torch.zeros((wl.B, wl.H_q, wl.D), dtype=torch.int16, device="cuda")
        self.lse = torch.zeros((wl.B, wl.H_q), device="cuda") if want_lse else None

        def ws(n):
            t = torch.empty(max(n, 16), dtype=torch.uint8, device="cuda")
            if garbage is not None:
                t.fill_(garbage)
            return t
        sp = api.make_select_params(self.sel_q, self.w, self.sel_k, self.fmt, self.L_cap, self.seq_len,
                                    self.max_seq_len, wl.B, 1, wl.H_idx, wl.d_idx, blk=wl.blk, q_block=1,
                                    indices=self.indices, cap=cap, budgets=self.budgets, **kw)
        self.ws_sel = ws(api.spot_select_workspace_bytes(sp))
        sp.workspace, sp.workspace_bytes = self.ws_sel.data_ptr(), self.ws_sel.numel()
        ap = api.make_attn_params(self.q, self.K, self.V, self.kv_strides, self.seq_len, self.max_seq_len, self.indices,
                                  self.budgets, cap, wl.B, 1, wl.H_q, wl.H_kv, wl.D, blk=wl.blk, sm_scale=wl.sm_scale,
                                  out=self.out, lse=self.lse, page_table=getattr(self, "page_table", None),
                                  page_tokens=getattr(self, "page_tokens", 0))
        self.ws_att = ws(api.spot_sparse_attn_decode_workspace_bytes(ap))
        ap.workspace, ap.workspace_bytes = self.ws_att.data_ptr(), self.ws_att.numel()
        dp = api.make_decode_step_params(sp, ap)
        self.ws_step = ws(api.spot_decode_step_workspace_bytes(dp))
        dp.workspace, dp.workspace_bytes = self.ws_step.data_ptr(), self.ws_step.numel()
        return dp

    def step_results(self):
        import torch
        torch.cuda.synchronize()
        return (self.indices.cpu().numpy(), self.budgets.cpu().numpy(), bf16_bits_to_f64(to_np_u16(self.out)),
                None if self.lse is None else self.lse.cpu().numpy())


# ------------------------------------------------------------------------------------------------------
# oracle side
# ------------------------------------------------------------------------------------------------------

def oracle_dequantised_view(fmt, k_bits):
    """What spot_dequantize_selector_k must return for BF16 keys k_bits stored in format fmt, as float64: the oracle's
    dequantised keys -- exactly BF16 numbers for every format but int4_bf16s, whose exact values q * s the call returns
    rounded to nearest-even BF16 (R39; the rounding is the workloads' converter, no method arithmetic)."""
    from workloads import f32_to_bf16_bits
    want = OQ.quantize_dequantize(fmt, k_bits)
    if fmt == "int4_bf16s":
        w32 = want.astype(np.float32)
        assert np.array_equal(w32.astype(np.float64), want)
        want = bf16_bits_to_f64(f32_to_bf16_bits(w32))
    return want


def oracle_keys(wl, fmt, b):
    """fp64 selector keys of sequence b as the given cache format stores them."""
    return OQ.quantize_dequantize(fmt, wl.sel_k[b])


def oracle_select(wl, fmt, b, **over):
    kw = wl.select_kwargs()
    kw.update(over)
    mode = kw.pop("mode", wl.mode)
    return OS.select_decode(bf16_bits_to_f64(wl.sel_q[b]), wl.w[b].astype(np.float64), oracle_keys(wl, fmt, b),
                            int(wl.seq_len[b]), wl.blk, mode, **kw)


def oracle_attend(wl, b, blocks):
    K = bf16_bits_to_f64(wl.K[b]).transpose(1, 0, 2)    # [L][H_kv][D]
    V = bf16_bits_to_f64(wl.V[b]).transpose(1, 0, 2)
    return OA.sparse_attn_decode(bf16_bits_to_f64(wl.q[b]), K, V, blocks, int(wl.seq_len[b]), wl.blk, wl.sm_scale)


# ------------------------------------------------------------------------------------------------------
# parity protocol for index lists (north_star: bit-exact "except where two block scores differ by less than 1e-6
# relative at the cut, which is reported"; DESIGN.md section 6 adds the mass-near-cut class)
# ------------------------------------------------------------------------------------------------------

def classify_selection(s_bar, sel, gpu_idx, gpu_budget, p=None, rel=1e-6):
    """-> 'exact' | 'score-near-tie' | 'mass-near-cut' | 'FAIL: ...'."""
    want = sel.indices.tolist()
    got = [int(x) for x in gpu_idx[:gpu_budget]]
    if got != sorted(set(got)) or any(x < 0 for x in got):
        return "FAIL: index list not strictly ascending / negative"
    if got == want and gpu_budget == sel.budget:
        return "exact"
    diff = set(got) ^ set(want)
    order = sel.order.tolist()
    if sel.n_taken == 0 or sel.n_taken > len(order):
        return "FAIL: sets differ %s" % sorted(diff)
    cut_score = s_bar[order[sel.n_taken - 1]]
    tol = rel * max(abs(cut_score), 1e-30)
    if len(got) == len(want) and all(abs(s_bar[b] - cut_score) <= tol for b in diff):
        return "score-near-tie"
    if p is not None and sel.cum is not None and abs(len(got) - len(want)) == 1 and sel.n_taken == sel.n_star:
        n = sel.n_star
        below = sel.cum[n - 2] if n >= 2 else 0.0
        margin = min(p - below, sel.cum[n - 1] - p)
        rank_pos = {b: r for r, b in enumerate(order)}
        if margin < rel and all(abs(rank_pos.get(b, -99) - (n - 1)) <= 1 for b in diff):
            return "mass-near-cut"
    return "FAIL: sets differ %s (budget %d vs %d)" % (sorted(diff)[:8], gpu_budget, sel.budget)


# ------------------------------------------------------------------------------------------------------
# prefill form
# ------------------------------------------------------------------------------------------------------

class DevicePrefill:
    """One or more PrefillWorkloads (same shapes, one per batch entry) resident on the GPU; the chunk of queries
    [q_start, q_start + Tq) is scored against the BF16 selector K-cache of capacity L."""

    def __init__(self, wls, q_start, Tq, with_kv=True):
        import torch
        from paper_2606_22874_b200 import api
        self.api, self.wls, self.q_start, self.Tq = api, wls, q_start, Tq
        wl = wls[0]
        self.wl, self.B, self.L = wl, len(wls), wl.L
        self.sel_q = dev_u16(np.stack([x.sel_q[q_start:q_start + Tq] for x in wls]))
        self.w = torch.from_numpy(np.stack([x.w[q_start:q_start + Tq] for x in wls])).cuda()
        self.sel_k = dev_u16(np.stack([x.sel_k for x in wls]))
        self.n_q = Tq // wl.q_block
        self.n_b_max = (q_start + Tq - 1) // wl.blk + 1
        if with_kv and wl.K is not None:
            self.Q = dev_u16(np.stack([x.Q[q_start:q_start + Tq] for x in wls]))     # [B][Tq][H_q][D]
            self.K = dev_u16(np.stack([x.K for x in wls]))                           # [B][H_kv][L][D]
            self.V = dev_u16(np.stack([x.V for x in wls]))
            self.kv_strides = (wl.H_kv * wl.L * wl.D, wl.D, wl.L * wl.D)

    def select(self, cap=None, want_scores=True, want_probs=True, **over):
        import torch
        wl, api = self.wl, self.api
        kw = dict(mode=wl.mode, top_k=wl.top_k, p=wl.p, sink_blocks=wl.sink_blocks,
                  recency_blocks=wl.recency_blocks, kmin_blocks=wl.kmin_blocks, temperature=wl.temperature)
        kw.update(over)
        cap = self.n_b_max if cap is None else cap
        rows = self.B * self.n_q
        indices = torch.full((rows, cap), -7, dtype=torch.int32, device="cuda")
        budgets = torch.full((rows,), -7, dtype=torch.int32, device="cuda")
        nb_stride = (self.n_b_max + 3) & ~3
        scores = torch.full((rows, nb_stride), float("nan"), device="cuda") if want_scores else None
        probs = torch.full((rows, nb_stride), float("nan"), device="cuda") if want_probs else None
        sp = api.make_select_params(self.sel_q, self.w, self.sel_k, getattr(self, "fmt", "bf16"), self.L, None, 0,
                                    self.B, self.Tq,
                                    wl.H_idx, wl.d_idx, q_start=self.q_start, blk=wl.blk, q_block=wl.q_block,
                                    indices=indices, cap=cap, budgets=budgets, block_scores=scores,
                                    block_probs=probs, nb_stride=nb_stride, q_fmt=getattr(self, "q_fmt", "bf16"), **kw)
        ws = torch.empty(max(api.spot_select_workspace_bytes(sp), 16), dtype=torch.uint8, device="cuda")
        sp.workspace, sp.workspace_bytes = ws.data_ptr(), ws.numel()
        api.spot_select(sp)
        torch.cuda.synchronize()
        return (indices.cpu().numpy(), budgets.cpu().numpy(),
                None if scores is None else scores.cpu().numpy(), None if probs is None else probs.cpu().numpy())

    def set_cache_format(self, fmt):
        """Re-store the selector cache in a quantised format (f2); the workloads' BF16 keys are replaced by the ORACLE
        quantiser's image of them (exactly BF16 numbers), so the oracle side needs no other change."""
        import torch
        from workloads import f32_to_bf16_bits
        wl, api = self.wl, self.api
        if not hasattr(self, "_sel_k_bf16"):              # a second call re-quantises the ORIGINAL BF16 keys, not the
            self._sel_k_bf16 = self.sel_k                 # previous call's cache (which is not a BF16 tensor any more)
            self._host_sel_k = [x.sel_k for x in self.wls]
        self.sel_k = torch.zeros(api.spot_selector_k_bytes(fmt, self.B, self.L, wl.H_idx, wl.d_idx), dtype=torch.uint8,
                                 device="cuda")
        api.spot_quantize_selector_k(self._sel_k_bf16, self.sel_k, fmt, self.B, self.L, 0, self.L, wl.H_idx, wl.d_idx)
        self.fmt = fmt
        for x, k0 in zip(self.wls, self._host_sel_k):
            x.sel_k = f32_to_bf16_bits(OQ.quantize_dequantize(fmt, k0).astype(np.float32))

    def quantise_queries(self, fmt="fp8_e4m3"):
        """f2: the chunk's selector queries through the cache quantiser (a cache of Tq tokens), kept in the quantised
        layout for the tensor-core path (q_fmt); the workloads' BF16 queries are replaced by the ORACLE quantiser's image of
        them, so the oracle scores (quantised q) x (quantised k)."""
        import torch
        from workloads import f32_to_bf16_bits
        wl, api = self.wl, self.api
        q8 = torch.zeros(api.spot_selector_k_bytes(fmt, self.B, self.Tq, wl.H_idx, wl.d_idx), dtype=torch.uint8, device="cuda")
        api.spot_quantize_selector_k(self.sel_q, q8, fmt, self.B, self.Tq, 0, self.Tq, wl.H_idx, wl.d_idx)
        self.sel_q, self.q_fmt = q8, fmt
        for x in self.wls:
            img = OQ.quantize_dequantize(fmt, x.sel_q[self.q_start:self.q_start + self.Tq])
            x.sel_q = x.sel_q.copy()
            x.sel_q[self.q_start:self.q_start + self.Tq] = f32_to_bf16_bits(img.astype(np.float32))

    def attend(self, indices_np, budgets_np, want_lse=False):
        import torch
        wl, api = self.wl, self.api
        out = torch.zeros((self.B, self.Tq, wl.H_q, wl.D), dtype=torch.int16, device="cuda")
        lse = torch.zeros((self.B, self.Tq, wl.H_q), device="cuda") if want_lse else None
        idx = torch.from_numpy(np.ascontiguousarray(indices_np, dtype=np.int32)).cuda()
        bud = torch.from_numpy(np.ascontiguousarray(budgets_np, dtype=np.int32)).cuda()
        ap = api.make_attn_params(self.Q, self.K, self.V, self.kv_strides, None, 0, idx, bud, idx.shape[1], self.B,
                                  self.Tq, wl.H_q, wl.H_kv, wl.D, q_start=self.q_start, blk=wl.blk,
                                  sm_scale=wl.sm_scale, out=out, lse=lse, page_table=getattr(self, "page_table", None),
                                  page_tokens=getattr(self, "page_tokens", 0))
        ws = torch.empty(max(api.spot_sparse_attn_prefill_workspace_bytes(ap), 16), dtype=torch.uint8, device="cuda")
        ap.workspace, ap.workspace_bytes = ws.data_ptr(), ws.numel()
        api.spot_sparse_attn_prefill(ap)
        torch.cuda.synchronize()
        return bf16_bits_to_f64(to_np_u16(out)), (None if lse is None else lse.cpu().numpy())


def oracle_select_prefill(wl, q_start, Tq, **over):
    """-> list over query blocks of (s_bar_i, Selection_i) for the chunk [q_start, q_start + Tq)."""
    kw = wl.select_kwargs()
    kw.update(over)
    mode = kw.pop("mode", wl.mode)
    return OS.select_prefill(bf16_bits_to_f64(wl.sel_q[q_start:q_start + Tq]),
                             wl.w[q_start:q_start + Tq].astype(np.float64), bf16_bits_to_f64(wl.sel_k),
                             q_start, wl.q_block, wl.blk, mode, **kw)


def oracle_attend_prefill(wl, q_start, Tq, block_lists):
    K = bf16_bits_to_f64(wl.K).transpose(1, 0, 2)
    V = bf16_bits_to_f64(wl.V).transpose(1, 0, 2)
    return OA.sparse_attn_prefill(bf16_bits_to_f64(wl.Q[q_start:q_start + Tq]), K, V, block_lists, q_start,
                                  wl.q_block, wl.blk, wl.sm_scale)
