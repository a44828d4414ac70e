#!/usr/bin/env python
"""bench.py -- one decode layer-step of the SpotAttention hot path (selector scoring -> dual top-p -> block-sparse
GQA attention) on synthetic Qwen3-shaped inputs, through the C ABI of include/spot.h.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--fmt bf16|mxfp4|int4_e4m3|fp8_e4m3|mxint8|int4_bf16s] [--p 0.9]
    python bench.py --impl reference ...       # the fp64 CPU oracle on a bounded sample (rank 0 only)

Prints ONE JSON line (rank 0).  A "step" = spot_decode_step (= spot_select + spot_sparse_attn_decode in one call) over
one batch (all of SURVEY.md section 8(a)'s decode rows: a1 score + block max, a2 distribution + selection, a3 sparse attention; a0 runs once, before
the timed region, because the cache is quantised when tokens are appended, not per step).  The L2 is flushed (a
read sweep over a 512 MiB buffer) before every timed step; each step is timed with its own CUDA-event pair on the
launching stream and the flush sits outside the pairs.  DESIGN.md section 7 states the byte accounting."""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "decode us/layer-step (selector+sparse attn) @L=128K; % of HBM roofline"
N_LAYERS = {32: 36, 64: 64}       # Qwen3-8B-shaped: 36 layers; 32B-shaped: 64 (model card)


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self._stop = index, [], threading.Event()
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                parts = [x.strip() for x in out.strip().split(",")]
                if len(parts) >= 7:
                    self.rows.append(parts)
            except Exception:
                pass
            self._stop.wait(0.02)

    def __enter__(self):
        self.t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self.t.join(timeout=6)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        sm = sorted(float(r[0]) for r in self.rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]), "reasons": reasons,
                "samples": len(self.rows)}


# ------------------------------------------------------------------------------------------------------
def build_workload(name, overrides):
    from workloads import make_config
    return make_config(name, with_kv=False, **overrides)


def oracle_step_sample(wl, fmt, K0, V0, q0, p):
    """The oracle's decode layer-step for sequence 0 (select + attend), as it stands.  Returns seconds, budget."""
    from oracle import attention as OA
    from oracle import quant as OQ
    from oracle import selection as OS
    from oracle.bf16 import bf16_bits_to_f64
    t0 = time.perf_counter()
    keys = OQ.quantize_dequantize(fmt, wl.sel_k[0])
    kw = wl.select_kwargs()
    kw["p"] = p
    s_bar, sel = OS.select_decode(bf16_bits_to_f64(wl.sel_q[0]), wl.w[0].astype(np.float64), keys,
                                  int(wl.seq_len[0]), wl.blk, wl.mode, **kw)
    OA.sparse_attn_decode(bf16_bits_to_f64(q0), bf16_bits_to_f64(K0).transpose(1, 0, 2),
                          bf16_bits_to_f64(V0).transpose(1, 0, 2), sel.indices, int(wl.seq_len[0]), wl.blk, wl.sm_scale)
    return time.perf_counter() - t0, sel.budget


def host_kv_for_seq0(wl, seed):
    """Sequence 0's K/V/q as BF16 bits on the host, N(0,1) (used by the reference arm, which has no GPU copy)."""
    from workloads import f32_to_bf16_bits
    rng = np.random.Generator(np.random.Philox(seed + 17))
    K0 = f32_to_bf16_bits(rng.standard_normal((wl.H_kv, wl.L_cap, wl.D), dtype=np.float32))
    V0 = f32_to_bf16_bits(rng.standard_normal((wl.H_kv, wl.L_cap, wl.D), dtype=np.float32))
    return K0, V0, wl.q[0]


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = build_workload(args.workload, dict(D_IDX_OVERRIDE))
    K0, V0, q0 = host_kv_for_seq0(wl, wl.seed)
    times = []
    budget = 0
    for i in range(args.warmup + args.steps):
        dt, budget = oracle_step_sample(wl, args.fmt, K0, V0, q0, args.p)
        if i >= args.warmup:
            times.append(dt)
    per_seq = float(np.mean(times))
    us = per_seq * wl.B * 1e6
    cores = len(os.sched_getaffinity(0))
    line = {
        "impl": "reference", "metric": METRIC, "value": us, "unit": "us/layer-step", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": us / 1e3, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "fmt": args.fmt, "p": args.p, "B": wl.B, "L": wl.L_cap},
        "cpu_baseline": {"value": us, "unit": "us/layer-step", "cores": cores, "kind": "oracle",
                         "sample": "sequence 0 of %d (select + attend, budget %d blocks), time x B" % (wl.B, budget)},
        "e2e": {"value": us, "unit": "us/layer-step", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


D_IDX_OVERRIDE = {}


def rank_workload(name, rank):
    """Every rank runs the same-shaped batch of independent sequences with its own seed (rank 0: the config's seed):
    the path shards by sequence, weak scaling, no data-path collective."""
    if rank == 0:
        return build_workload(name, dict(D_IDX_OVERRIDE))
    from workloads import CONFIGS, make_decode_workload
    kw = dict(CONFIGS[name])
    kw.update(D_IDX_OVERRIDE)
    kw["seed"] = kw["seed"] + 1000 * rank
    return make_decode_workload(name, with_kv=False, **kw)


def max_over_ranks(value, device, world):
    """The step time the contract reports: the slowest rank's."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())



def traffic_entry(key):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from profiles/traffic.json (ncu --set full captures named in
    profiles/traffic.json.md), or None when that kernel / workload has not been captured."""
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        with open(tpath) as f:
            return json.load(f).get(key)
    return None


def prefill_gemm_roofline(dev, steps, warmup, clocks_index):
    """BASELINE.json's second target, in the default run: the chunked-prefill selector GEMM of config 5 (a1', L = 65536,
    one chunk, BF16 4 x 64) timed ALONE through spot_score_blocks -> fraction of the measured BF16 tensor peak."""
    import torch
    from paper_2606_22874_b200 import api
    from workloads import make_prefill_workload
    L = 65536
    wl = make_prefill_workload(seed=5005, L=L, with_kv=False)
    n_qb = L // 64
    sel_q = torch.from_numpy(wl.sel_q.view(np.int16)).to(dev)
    w = torch.from_numpy(wl.w).to(dev)
    sel_k = torch.from_numpy(wl.sel_k.view(np.int16)).to(dev)
    nb_stride = (n_qb + 3) & ~3
    scores = torch.empty((n_qb, nb_stride), dtype=torch.float32, device=dev)
    sp = api.make_select_params(sel_q, w, sel_k, "bf16", L, None, 0, 1, L, wl.H_idx, wl.d_idx, q_start=0, blk=64,
                                q_block=64, block_scores=scores, nb_stride=nb_stride)
    stream = torch.cuda.current_stream()
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev).zero_()
    ts = []
    with ClockSampler(clocks_index) as clk:
        for i in range(steps + warmup):
            flush.view(torch.int64).sum()
            a_, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a_.record(stream)
            api.spot_score_blocks(sp, stream)
            b_.record(stream)
            torch.cuda.synchronize()
            if i >= warmup:
                ts.append(a_.elapsed_time(b_))
    burst, sustained, peak_src = tensor_peaks()
    tiles = n_qb * (n_qb + 1) // 2
    flop = 2.0 * 64 * 64 * wl.d_idx * wl.H_idx * tiles
    achieved = flop / (float(np.mean(ts)) * 1e-3) / 1e12
    # f2 (round 2): the same GEMM with queries AND keys in a quantised cache format, straight from the caches on the
    # low-precision tensor-core paths (q_fmt: FP8 x FP8 kind::f8f6f4, MXFP4 x MXFP4 kind::mxf4.block_scale), timed the same way
    low = {}
    for fmt in ("fp8_e4m3", "mxfp4"):
        k_f = torch.zeros(api.spot_selector_k_bytes(fmt, 1, L, wl.H_idx, wl.d_idx), dtype=torch.uint8, device=dev)
        q_f = torch.zeros_like(k_f)
        api.spot_quantize_selector_k(sel_k, k_f, fmt, 1, L, 0, L, wl.H_idx, wl.d_idx)
        api.spot_quantize_selector_k(sel_q, q_f, fmt, 1, L, 0, L, wl.H_idx, wl.d_idx)
        sp_f = api.make_select_params(q_f, w, k_f, fmt, L, None, 0, 1, L, wl.H_idx, wl.d_idx, q_start=0, blk=64,
                                      q_block=64, q_fmt=fmt, block_scores=scores, nb_stride=nb_stride)
        tf = []
        for i in range(max(3, steps // 2) + 2):
            flush.view(torch.int64).sum()
            a_, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a_.record(stream)
            api.spot_score_blocks(sp_f, stream)
            b_.record(stream)
            torch.cuda.synchronize()
            if i >= 2:
                tf.append(a_.elapsed_time(b_))
        low[fmt] = {"ms": float(np.mean(tf)), "tflops_equivalent": flop / (float(np.mean(tf)) * 1e-3) / 1e12,
                    "operand_bytes": int(k_f.numel() + q_f.numel()),
                    "traffic": traffic_entry("cfg5/%s+q/score_prefill_kernel" % fmt)}
        del k_f, q_f
    return {"bound": "tensor", "kernel": "score_prefill_kernel", "workload": "cfg5 (L=65536, one chunk, selector 4x64 bf16)",
            "low_precision_q_and_k": low,
            "ms": float(np.mean(ts)), "achieved": achieved, "peak": burst, "unit": "TFLOP/s", "frac": achieved / burst,
            "frac_of_sustained": achieved / sustained, "algorithmic_flops": flop,
            "traffic": traffic_entry("cfg5/bf16/score_prefill_kernel"), "peak_source": peak_src,
            "launches": steps, "clocks": clk.summary()}


# ------------------------------------------------------------------------------------------------------
def run_ours(args):
    import ctypes as C

    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_2606_22874_b200 import _lib, api
    from paper_2606_22874_b200 import build as B
    B.build()
    _lib.load()                                   # no fallback: raises if the CUDA library is missing

    wl = rank_workload(args.workload, rank)
    dev = torch.device("cuda", local_rank)
    Bn, L, Hq, Hkv, D = wl.B, wl.L_cap, wl.H_q, wl.H_kv, wl.D
    gen = torch.Generator(device=dev)
    gen.manual_seed(wl.seed + 17)
    K = torch.randn((Bn, Hkv, L, D), generator=gen, device=dev, dtype=torch.bfloat16)
    V = torch.randn((Bn, Hkv, L, D), generator=gen, device=dev, dtype=torch.bfloat16)
    q = torch.from_numpy(wl.q.view(np.int16)).to(dev)
    sel_q = torch.from_numpy(wl.sel_q.view(np.int16)).to(dev)
    w = torch.from_numpy(wl.w).to(dev)
    seq_len = torch.from_numpy(wl.seq_len).to(dev)
    sel_k_bf16 = torch.from_numpy(wl.sel_k.view(np.int16)).to(dev)
    sel_bytes = api.spot_selector_k_bytes(args.fmt, Bn, L, wl.H_idx, wl.d_idx)
    if args.fmt == "bf16":
        sel_k = sel_k_bf16
    else:
        sel_k = torch.zeros(sel_bytes, dtype=torch.uint8, device=dev)
        api.spot_quantize_selector_k(sel_k_bf16, sel_k, args.fmt, Bn, L, 0, L, wl.H_idx, wl.d_idx)
        del sel_k_bf16
    n_b = -(-L // wl.blk)
    cap = n_b
    indices = torch.empty((Bn, cap), dtype=torch.int32, device=dev)
    budgets = torch.empty((Bn,), dtype=torch.int32, device=dev)
    out = torch.empty((Bn, Hq, D), dtype=torch.int16, device=dev)
    sp = api.make_select_params(sel_q, w, sel_k, args.fmt, L, seq_len, L, Bn, 1, wl.H_idx, wl.d_idx, blk=wl.blk,
                                q_block=1, mode=wl.mode, top_k=wl.top_k, p=args.p, sink_blocks=wl.sink_blocks,
                                recency_blocks=wl.recency_blocks, kmin_blocks=wl.kmin_blocks,
                                temperature=wl.temperature, indices=indices, cap=cap, budgets=budgets)
    ws_sel = torch.empty(max(16, api.spot_select_workspace_bytes(sp)), dtype=torch.uint8, device=dev)
    sp.workspace, sp.workspace_bytes = ws_sel.data_ptr(), ws_sel.numel()
    kv_strides = (Hkv * L * D, D, L * D)
    paging = {}
    if args.paged:
        # the same bytes read as a page pool [page][H_kv][page_tokens][D] behind a random page table (f3, R32)
        pt = args.paged
        n_log = -(-L // pt)
        table = torch.randperm(Bn * n_log, generator=gen, device=dev).to(torch.int32).reshape(Bn, n_log)
        kv_strides = (Hkv * pt * D, D, pt * D)
        paging = dict(page_table=table, page_tokens=pt)
    ap = api.make_attn_params(q, K, V, kv_strides, seq_len, L, indices, budgets, cap, Bn, 1, Hq, Hkv, D, blk=wl.blk,
                              sm_scale=wl.sm_scale, out=out, **paging)
    ws_att = torch.empty(max(16, api.spot_sparse_attn_decode_workspace_bytes(ap)), dtype=torch.uint8, device=dev)
    ap.workspace, ap.workspace_bytes = ws_att.data_ptr(), ws_att.numel()
    apd = api.make_attn_params(q, K, V, kv_strides, seq_len, L, None, None, 0, Bn, 1, Hq, Hkv, D, blk=wl.blk,
                               sm_scale=wl.sm_scale, out=torch.empty_like(out), **paging)
    ws_den = torch.empty(max(16, api.spot_dense_attn_decode_workspace_bytes(apd)), dtype=torch.uint8, device=dev)
    apd.workspace, apd.workspace_bytes = ws_den.data_ptr(), ws_den.numel()

    # the step: a1 + a2 + a3 in ONE call (spot_decode_step: the same kernels as spot_select + spot_sparse_attn_decode,
    # launched so that they overlap -- include/spot.h)
    dp = api.make_decode_step_params(sp, ap)
    ws_step = torch.empty(max(16, api.spot_decode_step_workspace_bytes(dp)), dtype=torch.uint8, device=dev)
    dp.workspace, dp.workspace_bytes = ws_step.data_ptr(), ws_step.numel()

    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev).zero_()
    stream = torch.cuda.current_stream()

    def flush_l2():
        flush.view(torch.int64).sum()             # read sweep: leaves the L2 full of clean lines

    def step():
        api.spot_decode_step(dp, stream)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        flush_l2()
        step()
    barrier()

    # the step: both calls back to back, one event pair around them (the four kernels chain through programmatic
    # dependent launch, which an event between the calls would break)
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(args.steps)]
    # clocks / throttle reasons are sampled from here to the end of the e2e loop: the timed loop alone lasts ~10 ms,
    # less than one nvidia-smi query, and the loops that follow run the same kernels on the same data
    clk = ClockSampler(local_rank)
    clk.__enter__()
    for i in range(args.steps):
        flush_l2()
        ev[i][0].record(stream)
        api.spot_decode_step(dp, stream)
        ev[i][1].record(stream)
    barrier()
    step_ms = np.array([e[0].elapsed_time(e[1]) for e in ev])

    def time_alone(fn, n):
        ts = []
        for i in range(n + 2):
            flush_l2()
            a_, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a_.record(stream)
            fn()
            b_.record(stream)
            torch.cuda.synchronize()
            if i >= 2:
                ts.append(a_.elapsed_time(b_))
        return np.array(ts)

    # the two calls timed alone (breakdown, and the live duration of the dominant kernel for the roofline object), and
    # back to back as separate calls (what the one-call step is compared with)
    n_alone = max(3, min(args.steps, 20))
    sel_ms = time_alone(lambda: api.spot_select(sp, stream), n_alone)
    att_ms = time_alone(lambda: api.spot_sparse_attn_decode(ap, stream), n_alone)
    sep_ms = time_alone(lambda: (api.spot_select(sp, stream), api.spot_sparse_attn_decode(ap, stream)), n_alone)

    # the same step replayed from a CUDA graph (the calls never synchronise, so a caller may capture them)
    graph_us = None
    try:
        cap_stream = torch.cuda.Stream()
        gph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(gph, stream=cap_stream):
            api.spot_decode_step(dp, torch.cuda.current_stream())
        graph_us = float(time_alone(gph.replay, n_alone).mean()) * 1e3
    except Exception as e:                                    # reported, never fatal for the headline number
        graph_us = "capture failed: %s" % (str(e).splitlines()[0] if str(e) else type(e).__name__)

    # dense comparator (same shapes, every block)
    den = time_alone(lambda: api.spot_dense_attn_decode(apd, stream), max(3, min(args.steps, 10)))

    # the step right before the path, timed alone and reported beside the step, not inside it: selector
    # projections + RoPE + mixing weights + append of the new token's key to the cache (synthetic Qwen3-8B-sized weights)
    from workloads import make_project_workload
    d_model = 4096 if Hq == 32 else 5120
    pw = make_project_workload(seed=wl.seed + 29, B=Bn, d_model=d_model, H_idx=wl.H_idx, d_idx=wl.d_idx, L=L)
    p_dev = {k: torch.from_numpy(pw[k].view(np.int16)).to(dev) for k in ("hidden", "w_q", "w_k", "w_w")}
    p_pos = torch.full((Bn,), 63, dtype=torch.int32, device=dev)
    p_q = torch.empty_like(sel_q)
    p_w = torch.empty_like(w)
    # (a 64-token scratch cache of the same format: the append touches one slot per sequence whatever the cache size,
    # and the step's real cache stays as the generator made it)
    p_cache = torch.zeros(api.spot_selector_k_bytes(args.fmt, Bn, 64, wl.H_idx, wl.d_idx), dtype=torch.uint8, device=dev)
    pp = api.make_project_params(p_dev["hidden"], p_dev["w_q"], p_dev["w_k"], p_dev["w_w"], p_pos, Bn, d_model, wl.H_idx,
                                 wl.d_idx, rope_dims=min(64, wl.d_idx), rope_base=1.0e6, sel_q=p_q, w=p_w, sel_k=p_cache,
                                 fmt=args.fmt, cache_stride_tokens=64)
    ws_p = torch.empty(api.spot_selector_project_append_workspace_bytes(pp), dtype=torch.uint8, device=dev)
    pp.workspace, pp.workspace_bytes = ws_p.data_ptr(), ws_p.numel()
    f1_ms = time_alone(lambda: api.spot_selector_project_append(pp, stream), max(3, min(args.steps, 10)))
    f1_bytes = (2 * wl.H_idx * wl.d_idx + wl.H_idx + Bn) * d_model * 2

    # e2e: host buffers through spot_decode_step_host (H2D of the step's q / q^I / w, D2H of out + budgets)
    # The step's inputs sit back to back in one pinned buffer (sel_q | w | q) and so do their device staging areas, the
    # outputs likewise (out | budgets): spot_decode_step_host then moves each group in a single transfer.
    hp = api.DecodeStepHostParams()
    n_selq, n_w, n_q = wl.sel_q.nbytes, wl.w.nbytes, wl.q.nbytes
    n_out, n_bud = Bn * Hq * D * 2, Bn * 4
    h_in = torch.empty(n_selq + n_w + n_q, dtype=torch.uint8).pin_memory()
    h_in[:n_selq] = torch.from_numpy(wl.sel_q.view(np.uint8).reshape(-1))
    h_in[n_selq:n_selq + n_w] = torch.from_numpy(wl.w.view(np.uint8).reshape(-1))
    h_in[n_selq + n_w:] = torch.from_numpy(wl.q.view(np.uint8).reshape(-1))
    h_res = torch.empty(n_out + n_bud, dtype=torch.uint8).pin_memory()
    d_in = torch.empty(n_selq + n_w + n_q, dtype=torch.uint8, device=dev)
    d_res = torch.empty(n_out + n_bud, dtype=torch.uint8, device=dev)
    sp_e = type(sp).from_buffer_copy(sp)
    ap_e = type(ap).from_buffer_copy(ap)
    sp_e.sel_q, sp_e.w = d_in.data_ptr(), d_in.data_ptr() + n_selq
    ap_e.q = d_in.data_ptr() + n_selq + n_w
    ap_e.out, sp_e.budgets, ap_e.budgets = d_res.data_ptr(), d_res.data_ptr() + n_out, d_res.data_ptr() + n_out
    hp.sel_q_host, hp.w_host, hp.q_host = h_in.data_ptr(), h_in.data_ptr() + n_selq, h_in.data_ptr() + n_selq + n_w
    hp.out_host, hp.budgets_host = h_res.data_ptr(), h_res.data_ptr() + n_out
    hp.select, hp.attn = sp_e, ap_e
    ws_step_e = torch.empty(ws_step.numel(), dtype=torch.uint8, device=dev)
    hp.step_workspace, hp.step_workspace_bytes = ws_step_e.data_ptr(), ws_step_e.numel()
    h_bud = h_res[n_out:].view(torch.int32)
    h2d = n_selq + n_w + n_q
    d2h = n_out + n_bud
    e2e = []
    for i in range(args.steps + 2):
        flush_l2()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        api.spot_decode_step_host(hp, stream)
        torch.cuda.synchronize()
        if i >= 2:
            e2e.append((time.perf_counter() - t0) * 1e3)
    bud_host = h_bud.numpy().copy()
    clk.__exit__(None, None, None)
    clocks = clk.summary()

    step_mean = max_over_ranks(step_ms.mean(), dev, world)
    if rank != 0:
        return

    peak, peak_src = measured_peaks()

    def bytes_per_token(fmt):
        n = wl.H_idx * wl.d_idx
        return {"bf16": n * 2, "fp8_e4m3": n, "mxint8": n + n // 32, "int4_bf16s": n // 2 + n // 16}.get(
            fmt, n // 2 + n // 32)

    # config 3's own subject, in the default run: the same step with the selector K-cache quantised (INT4 + E4M3 scale,
    # MXFP4), beside the BF16 control above; and BASELINE.json's second target, the prefill selector GEMM, timed alone
    formats, prefill_roofline = None, None
    if args.extras and args.fmt == "bf16" and args.workload == "cfg3" and not args.paged and wl.blk == 64:
        formats = {"bf16": {"us": step_mean * 1e3, "selector_cache_bytes": int(sel_bytes), "bytes_per_token": bytes_per_token("bf16")}}
        # (round 2: all five quantised precisions the paper lists -- FP4, INT4 with an E4M3 or a 16-bit scale, FP8, INT8)
        for fmt in ("mxfp4", "int4_e4m3", "int4_bf16s", "fp8_e4m3", "mxint8"):
            n_f = max(3, min(args.steps, 10))
            sel_k_f = torch.zeros(api.spot_selector_k_bytes(fmt, Bn, L, wl.H_idx, wl.d_idx), dtype=torch.uint8, device=dev)
            api.spot_quantize_selector_k(sel_k, sel_k_f, fmt, Bn, L, 0, L, wl.H_idx, wl.d_idx)
            sp_f = type(sp).from_buffer_copy(sp)
            sp_f.sel_k, sp_f.fmt = sel_k_f.data_ptr(), api.FORMATS[fmt]
            ws_f = torch.empty(max(16, api.spot_select_workspace_bytes(sp_f)), dtype=torch.uint8, device=dev)
            sp_f.workspace, sp_f.workspace_bytes = ws_f.data_ptr(), ws_f.numel()
            dp_f = api.make_decode_step_params(sp_f, ap)
            dp_f.workspace, dp_f.workspace_bytes = ws_step.data_ptr(), ws_step.numel()
            for _ in range(3):
                flush_l2()
                api.spot_decode_step(dp_f, stream)
            torch.cuda.synchronize()
            ev_f = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(n_f)]
            for i in range(n_f):
                flush_l2()
                ev_f[i][0].record(stream)
                api.spot_decode_step(dp_f, stream)
                ev_f[i][1].record(stream)
            torch.cuda.synchronize()
            us_f = float(np.mean([e[0].elapsed_time(e[1]) for e in ev_f])) * 1e3
            sel_ms_f = time_alone(lambda: api.spot_select(sp_f, stream), max(3, min(args.steps, 10)))
            bud_f = budgets.cpu().numpy().astype(np.int64)
            sel_alg_f = float(np.sum(wl.seq_len.astype(np.int64)) * bytes_per_token(fmt))
            kv_alg_f = float(bud_f.sum() * wl.blk * Hkv * D * 2 * 2)
            formats[fmt] = {
                "us": us_f, "steps": n_f, "budgets": bud_f.tolist(),
                "selector_cache_bytes": int(sel_k_f.numel()), "bytes_per_token": bytes_per_token(fmt),
                "shrink_vs_bf16": float(sel_bytes) / float(sel_k_f.numel()),
                "select_call_us": float(sel_ms_f.mean()) * 1e3,
                "selector_gbs": sel_alg_f / (float(sel_ms_f.mean()) * 1e-3) / 1e9,
                "step_bytes": sel_alg_f + kv_alg_f,
                "step_frac": (sel_alg_f + kv_alg_f) / (us_f * 1e-6) / 1e9 / peak,
                "step_frac_of_8TBs": (sel_alg_f + kv_alg_f) / (us_f * 1e-6) / 1e9 / 8000.0,
                "selector_kernel_traffic": traffic_entry("%s/%s/score_decode_kernel" % (args.workload, fmt)),
            }
            del sel_k_f, ws_f
        api.spot_decode_step(dp, stream)            # leave indices / budgets as the BF16 control selected them
        torch.cuda.synchronize()
        prefill_roofline = prefill_gemm_roofline(dev, max(3, min(args.steps, 10)), 3, local_rank)

    bytes_per_tok = bytes_per_token(args.fmt)
    sel_alg = float(np.sum(wl.seq_len.astype(np.int64)) * bytes_per_tok)
    kv_alg = float(np.sum(bud_host.astype(np.int64)) * wl.blk * Hkv * D * 2 * 2)
    att_s = float(att_ms.mean()) * 1e-3
    achieved = kv_alg / att_s / 1e9
    traffic = traffic_entry("%s/%s/attn_decode_kernel" % (args.workload, args.fmt))
    us = step_mean * 1e3
    n_layers = N_LAYERS.get(Hq, 36)

    # oracle on the host cores, bounded sample: sequence 0 (needs its K/V bits back on the host)
    K0 = K[0].view(torch.int16).cpu().numpy().view(np.uint16)
    V0 = V[0].view(torch.int16).cpu().numpy().view(np.uint16)
    cpu_t, cpu_budget = oracle_step_sample(wl, args.fmt, K0, V0, wl.q[0], args.p)
    line = {
        "metric": METRIC, "value": us, "unit": "us/layer-step", "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": step_mean, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": args.workload, "B": Bn, "L": L, "H_q": Hq, "H_kv": Hkv, "D": D,
                   "selector": "%dx%d %s" % (wl.H_idx, wl.d_idx, args.fmt), "blk": wl.blk,
                   "kv_layout": ("paged, %d tokens per page, random table" % args.paged) if args.paged else "[B][H_kv][L][D]",
                   "mode": wl.mode,
                   "p": args.p, "sink/recency/kmin": [wl.sink_blocks, wl.recency_blocks, wl.kmin_blocks],
                   "budgets": bud_host.tolist(), "l2": "flushed by a 512 MiB read sweep before every timed step",
                   "kv": "N(0,1) BF16 generated on the device (seeded); selector side from workloads/"},
        "tokens_per_s": world * Bn / (n_layers * step_mean * 1e-3),
        "breakdown_us": {"select (score+select kernels)": float(sel_ms.mean()) * 1e3,
                         "sparse attention (attn+merge kernels)": float(att_ms.mean()) * 1e3,
                         "spot_select + spot_sparse_attn_decode as two calls": float(sep_ms.mean()) * 1e3,
                         "dense flash-decode comparator": float(np.mean(den)) * 1e3,
                         "step replayed from a CUDA graph": graph_us,
                         "upstream f1 alone (projection + RoPE + append; not in the step)": float(np.mean(f1_ms)) * 1e3},
        "upstream_f1": {"us": float(np.mean(f1_ms)) * 1e3, "weight_bytes": f1_bytes, "d_model": d_model,
                        "note": "latency-bound: %.1f MiB of weights = %.2f us at the measured copy peak"
                                % (f1_bytes / 2 ** 20, f1_bytes / peak / 1e3)},
        "step_roofline": {"bytes": sel_alg + kv_alg, "achieved_gbs": (sel_alg + kv_alg) / (step_mean * 1e-3) / 1e9,
                          "frac_of_measured": (sel_alg + kv_alg) / (step_mean * 1e-3) / 1e9 / peak,
                          "frac_of_8TBs": (sel_alg + kv_alg) / (step_mean * 1e-3) / 1e9 / 8000.0,
                          "selector_bytes": sel_alg, "selected_kv_bytes": kv_alg,
                          "selector_gbs": sel_alg / (float(sel_ms.mean()) * 1e-3) / 1e9},
        "roofline": {"bound": "hbm", "kernel": "attn_decode_kernel", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                     "algorithmic_bytes": kv_alg},
        "cpu_baseline": {"value": cpu_t * Bn * 1e6, "unit": "us/layer-step", "cores": len(os.sched_getaffinity(0)),
                         "kind": "oracle",
                         "sample": "sequence 0 of %d (select + attend, budget %d blocks), time x B" % (Bn, cpu_budget)},
        "e2e": {"value": float(np.mean(e2e)) * 1e3, "unit": "us/layer-step", "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h},
        "gpu_launches": 4 * args.steps,          # score, select, attn, merge per step (timed loop only)
        "clocks": clocks,
        "formats": formats,
        "prefill_roofline": prefill_roofline,
        "traffic_source": "profiles/traffic.json: dram__bytes_read.sum + dram__bytes_write.sum per launch from the ncu --set full "
                          "captures named in profiles/traffic.json.md (null: that kernel / format has no capture there)",
        "paper_context": "paper: 3.9x FlashAttention / 1.8x Twilight end-to-end at L=128K, Qwen3-8B, one B200, Triton "
                         "kernels (PAPER.md:146); other shapes, context only",
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------------
# chunked prefill (BASELINE.json config 5): a1' tile scoring on tcgen05 -> a2 per query block -> a3' sparse attention
# ------------------------------------------------------------------------------------------------------
PF_METRIC = "prefill ms/layer (selector GEMM + dual top-p + block-sparse causal attn) @L=64K; % of tensor-pipe peak"


def tensor_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return float(d["bf16_tflops"]), float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), \
            "measured (MEASURED_PEAKS.json bf16_tflops, burst: the kernel is timed alone)"
    return 1700.0, 1700.0, "fallback (B200_PROFILING.md)"


def oracle_prefill_sample(wl, K, V, Q, blocks, p, fmt="bf16"):
    """The oracle's prefill layer pass on a few query blocks (scoring, selection, attention).  K/V/Q: BF16 bits on the
    host.  Returns (seconds, scored tiles, attended (query block, key block) pairs)."""
    from oracle import attention as OA
    from oracle import quant as OQ
    from oracle import selection as OS
    from oracle.bf16 import bf16_bits_to_f64
    t0 = time.perf_counter()
    keys = OQ.quantize_dequantize(fmt, wl.sel_k[:(max(blocks) + 1) * 64])        # fp64, as the cache format stores them
    tiles = pairs = 0
    kw = wl.select_kwargs()
    kw["p"] = p
    for i in blocks:
        q0 = i * 64
        n_tok = q0 + 64
        res = OS.select_prefill(bf16_bits_to_f64(wl.sel_q[q0:q0 + 64]), wl.w[q0:q0 + 64].astype(np.float64),
                                keys[:n_tok], q0, wl.q_block, wl.blk, wl.mode, **kw)
        s_bar, sel = res[0]
        OA.sparse_attn_prefill(bf16_bits_to_f64(Q[q0:q0 + 64]), bf16_bits_to_f64(K[:, :n_tok]).transpose(1, 0, 2),
                               bf16_bits_to_f64(V[:, :n_tok]).transpose(1, 0, 2), [sel.indices.tolist()], q0,
                               wl.q_block, wl.blk, wl.sm_scale)
        tiles += i + 1
        pairs += sel.budget
    return time.perf_counter() - t0, tiles, pairs


def run_prefill(args):
    import torch
    from workloads import make_prefill_workload, f32_to_bf16_bits
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    L = args.L or 65536
    assert args.fmt != "int4_bf16s", ("--fmt int4_bf16s is a decode-row format: its keys q * s are not BF16 numbers and prefill "
                                      "selection over it returns SPOT_ERR_UNSUPPORTED (DESIGN.md R39)")
    geo = dict(D_IDX_OVERRIDE)
    if args.blk == 16:                # the paper's 16-token key blocks with its 8 / 16 / 32 reserved blocks (f3)
        geo.update(blk=16, sink_blocks=8, recency_blocks=16, kmin_blocks=32)
    wl = make_prefill_workload(seed=5005 + 1000 * rank, L=L, with_kv=False, **geo)
    wl.p = args.p
    n_qb = L // 64
    blk = wl.blk
    n_kb = L // blk
    Hq, Hkv, D = wl.H_q, wl.H_kv, wl.D

    if args.impl == "reference":
        if rank != 0:
            return
        rng = np.random.Generator(np.random.Philox(wl.seed + 17))
        n_tok = min(L, 4096)                       # the sampled query blocks all sit below this position
        Kh = f32_to_bf16_bits(rng.standard_normal((Hkv, n_tok, D), dtype=np.float32))
        Vh = f32_to_bf16_bits(rng.standard_normal((Hkv, n_tok, D), dtype=np.float32))
        Qh = f32_to_bf16_bits(rng.standard_normal((n_tok, Hq, D), dtype=np.float32))
        blocks = [0, n_tok // 128, n_tok // 64 - 1]
        ts = []
        for i in range(args.warmup + args.steps):
            dt, tiles, pairs = oracle_prefill_sample(wl, Kh, Vh, Qh, blocks, args.p, args.fmt)
            if i >= args.warmup:
                ts.append(dt)
        full_tiles = n_qb * (n_qb + 1) // 2
        ms = float(np.mean(ts)) / tiles * full_tiles * 1e3
        cores = len(os.sched_getaffinity(0))
        sample = ("query blocks %s of %d (score + select + attend; %d tiles, %d attended block pairs), time scaled "
                  "linearly in scored tiles to the full lower triangle (%d tiles)" % (blocks, n_qb, tiles, pairs, full_tiles))
        print(json.dumps({
            "impl": "reference", "metric": PF_METRIC, "value": ms, "unit": "ms/layer", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "cfg5", "L": L, "p": args.p},
            "cpu_baseline": {"value": ms, "unit": "ms/layer", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": ms, "unit": "ms/layer", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))
        return

    torch.cuda.set_device(local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_2606_22874_b200 import _lib, api
    from paper_2606_22874_b200 import build as B
    B.build()
    _lib.load()
    dev = torch.device("cuda", local_rank)
    gen = torch.Generator(device=dev)
    gen.manual_seed(wl.seed + 17)
    Q = torch.randn((1, L, Hq, D), generator=gen, device=dev, dtype=torch.bfloat16)
    K = torch.randn((1, Hkv, L, D), generator=gen, device=dev, dtype=torch.bfloat16)
    V = torch.randn((1, Hkv, L, D), generator=gen, device=dev, dtype=torch.bfloat16)
    h_selq = torch.from_numpy(wl.sel_q.view(np.int16)).pin_memory()
    h_w = torch.from_numpy(wl.w).pin_memory()
    h_selk = torch.from_numpy(wl.sel_k.view(np.int16)).pin_memory()
    sel_q, w, sel_k = h_selq.to(dev), h_w.to(dev), h_selk.to(dev)
    sel_k_bf16 = sel_k
    if args.fmt != "bf16":
        # f2: the selector cache in a quantised format; spot_select dequantises the visible prefix into its workspace
        sel_k = torch.zeros(api.spot_selector_k_bytes(args.fmt, 1, L, wl.H_idx, wl.d_idx), dtype=torch.uint8, device=dev)
        api.spot_quantize_selector_k(sel_k_bf16, sel_k, args.fmt, 1, L, 0, L, wl.H_idx, wl.d_idx)
    sel_q_in, q_fmt = sel_q, "bf16"
    if args.qfmt != "bf16":
        # f2: the queries quantised too -- FP8 x FP8 tile scores on the tensor cores, no dequantise pass (spot.h, q_fmt)
        assert args.fmt == args.qfmt and args.qfmt in ("fp8_e4m3", "mxfp4"), "--qfmt X needs --fmt X (fp8_e4m3 or mxfp4)"
        sel_q_in = torch.zeros(api.spot_selector_k_bytes(args.qfmt, 1, L, wl.H_idx, wl.d_idx), dtype=torch.uint8, device=dev)
        api.spot_quantize_selector_k(sel_q, sel_q_in, args.qfmt, 1, L, 0, L, wl.H_idx, wl.d_idx)
        q_fmt = args.qfmt
    f8 = q_fmt != "bf16"
    tc_ratio = {"bf16": 1.0, "fp8_e4m3": 2.0, "mxfp4": 4.0}[q_fmt]         # a contraction takes the peak of its own dtype
    cap = n_kb
    nb_stride = (n_kb + 3) & ~3
    indices = torch.empty((n_qb, cap), dtype=torch.int32, device=dev)
    budgets = torch.empty((n_qb,), dtype=torch.int32, device=dev)
    scores = torch.empty((n_qb, nb_stride), dtype=torch.float32, device=dev)
    out = torch.empty((1, L, Hq, D), dtype=torch.int16, device=dev)
    sp = api.make_select_params(sel_q_in, w, sel_k, args.fmt, L, None, 0, 1, L, wl.H_idx, wl.d_idx, q_start=0, blk=blk,
                                q_fmt=q_fmt, q_block=64, mode=wl.mode, top_k=wl.top_k, p=args.p, sink_blocks=wl.sink_blocks,
                                recency_blocks=wl.recency_blocks, kmin_blocks=wl.kmin_blocks,
                                temperature=wl.temperature, indices=indices, cap=cap, budgets=budgets,
                                block_scores=scores, nb_stride=nb_stride)
    ws = torch.empty(max(16, api.spot_select_workspace_bytes(sp)), dtype=torch.uint8, device=dev)
    sp.workspace, sp.workspace_bytes = ws.data_ptr(), ws.numel()
    kv_strides, paging = (Hkv * L * D, D, L * D), {}
    if args.paged:
        # the same bytes read as a page pool [page][H_kv][page_tokens][D] behind a random page table (f3, R32)
        pt = max(args.paged, 64)
        gen_t = torch.Generator(device=dev)
        gen_t.manual_seed(wl.seed + 23)
        table = torch.randperm(L // pt, generator=gen_t, device=dev).to(torch.int32).reshape(1, L // pt)
        kv_strides, paging = (Hkv * pt * D, D, pt * D), dict(page_table=table, page_tokens=pt)
    ap = api.make_attn_params(Q, K, V, kv_strides, None, 0, indices, budgets, cap, 1, L, Hq, Hkv, D,
                              q_start=0, blk=blk, sm_scale=wl.sm_scale, out=out, **paging)
    stream = torch.cuda.current_stream()
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev).zero_()

    def flush_l2():
        flush.view(torch.int64).sum()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
            torch.cuda.synchronize()

    W = max(args.warmup, 3)
    # the selector GEMM kernel alone (spot_score_blocks = a1' only), live, for the roofline object -- timed FIRST, after
    # W warm-up launches of its own and before any attention pass: its denominator is the burst peak of a kernel timed
    # alone (B200_PROFILING.md), and tens of ms of attention per step push the part into its power cap (SM clock
    # 1800 instead of 1965 MHz: the same kernel then takes 1.28 instead of 1.17 ms)
    sc = []
    for i in range(args.steps + W):
        flush_l2()
        a_, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a_.record(stream)
        api.spot_score_blocks(sp, stream)
        b_.record(stream)
        torch.cuda.synchronize()
        if i >= W:
            sc.append(a_.elapsed_time(b_))
    for _ in range(W):
        flush_l2()
        api.spot_select(sp, stream)
        api.spot_sparse_attn_prefill(ap, stream)
    barrier()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    clk = ClockSampler(local_rank)
    clk.__enter__()
    for i in range(args.steps):
        flush_l2()
        ev[i][0].record(stream)
        api.spot_select(sp, stream)
        ev[i][1].record(stream)
        api.spot_sparse_attn_prefill(ap, stream)
        ev[i][2].record(stream)
    barrier()
    sel_ms = np.array([e[0].elapsed_time(e[1]) for e in ev])
    att_ms = np.array([e[1].elapsed_time(e[2]) for e in ev])
    step_ms = np.array([e[0].elapsed_time(e[2]) for e in ev])
    # dense causal comparator (indices NULL) -- a few iterations only
    apd = api.make_attn_params(Q, K, V, kv_strides, None, 0, None, None, 0, 1, L, Hq, Hkv, D,
                               q_start=0, blk=blk, sm_scale=wl.sm_scale, out=out, **paging)
    den = []
    for i in range(3):
        a_, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a_.record(stream)
        api.spot_sparse_attn_prefill(apd, stream)
        b_.record(stream)
        torch.cuda.synchronize()
        if i >= 1:
            den.append(a_.elapsed_time(b_))
    api.spot_select(sp, stream)
    torch.cuda.synchronize()
    bud_host = budgets.cpu().numpy().astype(np.int64)
    # e2e: the selector-side inputs of the chunk cross PCIe inside the timed region, budgets come back
    e2e = []
    h_bud = torch.empty((n_qb,), dtype=torch.int32).pin_memory()
    for i in range(min(args.steps, 5) + 1):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        sel_q.copy_(h_selq, non_blocking=True)
        w.copy_(h_w, non_blocking=True)
        sel_k_bf16.copy_(h_selk, non_blocking=True)
        if args.fmt != "bf16":             # the cache is produced from the fresh keys inside the step
            api.spot_quantize_selector_k(sel_k_bf16, sel_k, args.fmt, 1, L, 0, L, wl.H_idx, wl.d_idx, stream)
        if q_fmt != "bf16":
            api.spot_quantize_selector_k(sel_q, sel_q_in, q_fmt, 1, L, 0, L, wl.H_idx, wl.d_idx, stream)
        api.spot_select(sp, stream)
        api.spot_sparse_attn_prefill(ap, stream)
        h_bud.copy_(budgets, non_blocking=True)
        torch.cuda.synchronize()
        if i >= 1:
            e2e.append((time.perf_counter() - t0) * 1e3)
    clk.__exit__(None, None, None)
    clocks = clk.summary()

    step_mean = max_over_ranks(step_ms.mean(), dev, world)
    if rank != 0:
        return
    burst, sustained, peak_src = tensor_peaks()
    tiles = n_qb * (n_qb + 1) // 2
    gemm_flop = 2.0 * 64 * 64 * wl.d_idx * wl.H_idx * tiles
    att_flop = 4.0 * 64 * blk * D * Hq * float(bud_host.sum())
    score_s = float(np.mean(sc)) * 1e-3
    achieved = gemm_flop / score_s / 1e12
    traffic = traffic_entry("cfg5/%s/score_prefill_kernel" % (args.fmt if q_fmt == "bf16" else args.fmt + "+q"))
    # oracle on the host cores: three query blocks below position 4096
    n_tok = min(L, 4096)
    Kh = K[0, :, :n_tok].contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
    Vh = V[0, :, :n_tok].contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
    Qh = Q[0, :n_tok].contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
    blocks = [0, n_tok // 128, n_tok // 64 - 1]
    cpu_t, cpu_tiles, cpu_pairs = oracle_prefill_sample(wl, Kh, Vh, Qh, blocks, args.p, args.fmt)
    line = {
        "metric": PF_METRIC, "value": step_mean, "unit": "ms/layer", "n_gpus": world, "steps": args.steps,
        "warmup": W, "ms_per_step": step_mean, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16" if not f8 else "bf16 (attention), %s x %s -> fp32 (tile scores)" % (q_fmt, q_fmt), "data": "synthetic",
        "config": {"workload": "cfg5", "B": 1, "L": L, "H_q": Hq, "H_kv": Hkv, "D": D,
                   "selector": "%dx%d %s" % (wl.H_idx, wl.d_idx, args.fmt), "selector_queries": q_fmt, "blk": blk, "q_block": 64,
                   "kv_layout": ("paged, %d tokens per page, random table" % max(args.paged, 64)) if args.paged else "[B][H_kv][L][D]", "mode": wl.mode, "p": args.p,
                   "sink/recency/kmin": [wl.sink_blocks, wl.recency_blocks, wl.kmin_blocks],
                   "mean_budget": float(bud_host.mean()), "density": float(bud_host.sum()) * blk / 64.0 / tiles,
                   "l2": "flushed by a 512 MiB read sweep before every timed step"},
        "tokens_per_s": world * L / (step_mean * 1e-3),
        "breakdown_ms": {"select (tile-score GEMM + selection kernels)": float(sel_ms.mean()),
                         "tile-score GEMM alone (spot_score_blocks)": float(np.mean(sc)),
                         "sparse causal attention": float(att_ms.mean()),
                         "dense causal attention (same kernel, every block)": float(np.mean(den))},
        "attention_tflops": att_flop / (float(att_ms.mean()) * 1e-3) / 1e12,
        "roofline": {"bound": "tensor", "kernel": "score_prefill_kernel" + ("<.., %s x %s>" % (q_fmt, q_fmt) if f8 else ""),
                     "achieved": achieved, "peak": burst * tc_ratio, "unit": "TFLOP/s", "frac": achieved / (burst * tc_ratio),
                     "frac_of_sustained": achieved / (sustained * tc_ratio), "traffic": traffic,
                     "peak_source": peak_src + ((" x %g: the guide's nominal %s : bf16 ratio (%g : 2.25 PFLOP/s); no such "
                                                 "peak is measured on this pool") % (tc_ratio, q_fmt, 2.25 * tc_ratio) if f8 else ""),
                     "algorithmic_flops": gemm_flop},
        "cpu_baseline": {"value": cpu_t / cpu_tiles * tiles * 1e3, "unit": "ms/layer",
                         "cores": len(os.sched_getaffinity(0)), "kind": "oracle",
                         "sample": "query blocks %s of %d (score + select + attend; %d tiles, %d attended block pairs), "
                                   "time scaled linearly in scored tiles to %d" % (blocks, n_qb, cpu_tiles, cpu_pairs, tiles)},
        "e2e": {"value": float(np.mean(e2e)), "unit": "ms/layer",
                "h2d_bytes_per_step": h_selq.numel() * 2 + h_w.numel() * 4 + h_selk.numel() * 2,
                "d2h_bytes_per_step": h_bud.numel() * 4},
        "gpu_launches": 3 * args.steps,
        "clocks": clocks,
    }
    print(json.dumps(line))



# ------------------------------------------------------------------------------------------------------
# f4: the training-side reductions at the paper's training length (L = 16384, K_train = 8192 tokens = 512 blocks
# of 16) on the synthetic prefill workload's tensors
# ------------------------------------------------------------------------------------------------------
TR_METRIC = "training reductions ms/layer (teacher Eq.1 + DenseKL Eq.3 + SparseKL Eq.4) @L=16K; % of tensor-pipe peak"


def oracle_train_sample(wl, n):
    from oracle import training as OT
    from oracle.bf16 import bf16_bits_to_f64
    t0 = time.perf_counter()
    OT.training_reductions(bf16_bits_to_f64(wl.Q[:n]), bf16_bits_to_f64(wl.K[:, :n]).transpose(1, 0, 2), wl.sm_scale,
                           bf16_bits_to_f64(wl.sel_q[:n]), wl.w[:n].astype(np.float64), bf16_bits_to_f64(wl.sel_k[:n]),
                           wl.blk, max(1, n // 32))
    return time.perf_counter() - t0


def run_train(args):
    from workloads import make_prefill_workload
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    L = args.L or 16384
    top_k = max(1, L // 32)                      # K_train = 0.5 L tokens = L / 32 blocks of 16 (Table 3)
    wl = make_prefill_workload(seed=7007 + 1000 * rank, L=L, blk=16, **{k: v for k, v in D_IDX_OVERRIDE.items() if k == "d_idx"})
    cores = len(os.sched_getaffinity(0))
    n_cpu = 384
    pairs_full, pairs_cpu = L * (L + 1) / 2, n_cpu * (n_cpu + 1) / 2
    if args.impl == "reference":
        if rank != 0:
            return
        ts = [oracle_train_sample(wl, n_cpu) for _ in range(args.warmup + args.steps)][args.warmup:]
        ms = float(np.mean(ts)) * pairs_full / pairs_cpu * 1e3
        sample = "the first %d tokens of the sequence (%d of %d causal pairs), time scaled by the pair count" % (n_cpu, pairs_cpu, pairs_full)
        print(json.dumps({"impl": "reference", "metric": TR_METRIC, "value": ms, "unit": "ms/layer", "n_gpus": args.gpus,
                          "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": False,
                          "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                          "config": {"workload": "train", "L": L, "top_k_blocks": top_k},
                          "cpu_baseline": {"value": ms, "unit": "ms/layer", "cores": cores, "kind": "oracle", "sample": sample},
                          "e2e": {"value": ms, "unit": "ms/layer", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))
        return
    import torch
    torch.cuda.set_device(local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_2606_22874_b200 import _lib, api
    from paper_2606_22874_b200 import build as B
    B.build()
    _lib.load()
    dev = torch.device("cuda", local_rank)
    pin = lambda a_: torch.from_numpy(np.ascontiguousarray(a_).view(np.int16)).pin_memory()
    h = {k: pin(getattr(wl, k)) for k in ("Q", "K", "sel_q", "sel_k")}
    h_w = torch.from_numpy(wl.w).pin_memory()
    d = {k: v.to(dev) for k, v in h.items()}
    w = h_w.to(dev)
    dkl = torch.empty((L,), device=dev)
    skl = torch.empty((L,), device=dev)
    tp = api.make_train_params(d["Q"], d["K"], (wl.D, L * wl.D), d["sel_q"], w, d["sel_k"], L, wl.H_q, wl.H_kv, wl.D,
                               wl.H_idx, wl.d_idx, blk=16, top_k=top_k, sm_scale=wl.sm_scale, dense_kl=dkl, sparse_kl=skl)
    ws = torch.empty(api.spot_train_kl_workspace_bytes(tp), dtype=torch.uint8, device=dev)
    tp.workspace, tp.workspace_bytes = ws.data_ptr(), ws.numel()
    stream = torch.cuda.current_stream()
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev).zero_()
    W = max(args.warmup, 3)
    for _ in range(W):
        api.spot_train_kl(tp, stream)
    torch.cuda.synchronize()
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(args.steps)]
    with ClockSampler(local_rank) as clk:
        for i in range(args.steps):
            flush.view(torch.int64).sum()
            ev[i][0].record(stream)
            api.spot_train_kl(tp, stream)
            ev[i][1].record(stream)
        torch.cuda.synchronize()
        e2e = []
        h_out = torch.empty((2, L), dtype=torch.float32).pin_memory()
        for i in range(min(args.steps, 5) + 1):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for k_ in h:
                d[k_].copy_(h[k_], non_blocking=True)
            w.copy_(h_w, non_blocking=True)
            api.spot_train_kl(tp, stream)
            h_out[0].copy_(dkl, non_blocking=True)
            h_out[1].copy_(skl, non_blocking=True)
            torch.cuda.synchronize()
            if i >= 1:
                e2e.append((time.perf_counter() - t0) * 1e3)
    ms = max_over_ranks(float(np.mean([e[0].elapsed_time(e[1]) for e in ev])), dev, world)
    if rank != 0:
        return
    burst, sustained, peak_src = tensor_peaks()
    flop = 2.0 * (2.0 * pairs_full * wl.H_q * wl.D) + 2.0 * (2.0 * pairs_full * wl.H_idx * wl.d_idx)   # two passes: teacher + selector
    achieved = flop / (ms * 1e-3) / 1e12
    cpu_t = oracle_train_sample(wl, n_cpu)
    print(json.dumps({
        "metric": TR_METRIC, "value": ms, "unit": "ms/layer", "n_gpus": world, "steps": args.steps, "warmup": W,
        "ms_per_step": ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": "train", "L": L, "H_q": wl.H_q, "H_kv": wl.H_kv, "D": wl.D,
                   "selector": "%dx%d bf16" % (wl.H_idx, wl.d_idx), "blk": 16, "top_k_blocks": top_k,
                   "l2": "flushed by a 512 MiB read sweep before every timed step"},
        "losses": {"dense_kl_mean": float(dkl.mean()), "sparse_kl_mean": float(skl.mean())},
        "tokens_per_s": world * L / (ms * 1e-3),
        "roofline": {"bound": "tensor", "kernel": "the whole call: attn_prefill_tc_kernel<64, STATS> + student_pass1_kernel (pass 1), select, train_pass_kernel<2> (pass 2, mma.sync)", "achieved": achieved,
                     "peak": sustained, "unit": "TFLOP/s", "frac": achieved / sustained, "traffic": None,
                     "peak_source": peak_src + "; sustained figure: the two passes run for milliseconds",
                     "algorithmic_flops": flop},
        "cpu_baseline": {"value": cpu_t * pairs_full / pairs_cpu * 1e3, "unit": "ms/layer", "cores": cores, "kind": "oracle",
                         "sample": "the first %d tokens of the sequence, time scaled by the causal pair count" % n_cpu},
        "e2e": {"value": float(np.mean(e2e)), "unit": "ms/layer",
                "h2d_bytes_per_step": int(sum(v.numel() * 2 for v in h.values()) + h_w.numel() * 4), "d2h_bytes_per_step": 8 * L},
        "gpu_launches": 6 * args.steps, "clocks": clk.summary()}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--fmt", default="bf16", choices=["bf16", "mxfp4", "int4_e4m3", "fp8_e4m3", "mxint8", "int4_bf16s"])
    ap.add_argument("--qfmt", default="bf16", choices=["bf16", "fp8_e4m3", "mxfp4"],
                    help="cfg5 only: format of the selector QUERIES (fp8_e4m3 with --fmt fp8_e4m3: FP8 x FP8 tensor-core scoring)")
    ap.add_argument("--p", type=float, default=0.90)
    ap.add_argument("--L", type=int, default=0, help="cfg5 only: prompt length (default 65536)")
    ap.add_argument("--d-idx", type=int, default=0, choices=[0, 64, 128],
                    help="selector head dim (default: the config's 64; 128 = the paper's geometry, PAPER.md:363)")
    ap.add_argument("--paged", type=int, default=0, choices=[0, 16, 64, 256],
                    help="K/V as a page pool of this many tokens per page behind a random page table (prefill: >= 64)")
    ap.add_argument("--blk", type=int, default=64, choices=[64, 16],
                    help="decode only: selection block size (16 = the paper's geometry with its 8/16/32 reserved "
                         "sink/recency/K_min blocks, PAPER.md:362-365, :400-402)")
    ap.add_argument("--no-extras", dest="extras", action="store_false",
                    help="skip the quantised-cache steps and the prefill selector GEMM that the default cfg3 / bf16 run "
                         "reports beside the headline (keys formats, prefill_roofline)")
    args = ap.parse_args()
    if args.d_idx:
        D_IDX_OVERRIDE["d_idx"] = args.d_idx
    if args.blk == 16 and args.workload != "cfg5":
        D_IDX_OVERRIDE.update(blk=16, sink_blocks=8, recency_blocks=16, kmin_blocks=32)
    if args.workload == "train":
        run_train(args)
    elif args.workload == "cfg5":
        run_prefill(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
