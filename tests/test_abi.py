"""C-ABI checks that need no GPU (-m "not gpu"): libspot.so builds and loads, exports every symbol include/spot.h
declares, the ctypes structs match the compiled layout, the size query matches the byte counts the paper prints
(PAPER.md:188), and every argument error of SURVEY.md section 8(b) is rejected on the host before any launch.
No compute call is made here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_22874_b200 import build as B
    from paper_2606_22874_b200 import _lib
    B.build()
    return _lib.load()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "spot.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(spot_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported_and_bound(lib):
    from paper_2606_22874_b200 import _lib, api
    names = declared_symbols()
    assert len(names) >= 17 and "spot_quantize_selector_k" in names and "spot_sparse_attn_prefill" in names
    for n in names:
        assert hasattr(lib, n), "libspot.so does not export %s" % n
        assert n in _lib.PROTOTYPES, "binding has no prototype for %s" % n
    for n in ("spot_quantize_selector_k", "spot_dequantize_selector_k", "spot_select", "spot_score_blocks",
              "spot_sparse_attn_decode", "spot_sparse_attn_decode_static", "spot_sparse_attn_prefill", "spot_dense_attn_decode",
              "spot_decode_step_host", "spot_selector_k_bytes"):
        assert callable(getattr(api, n)), "python binding lacks %s" % n


def test_struct_layout_and_strings(lib):
    from paper_2606_22874_b200 import _lib
    assert lib.spot_struct_size(0) == C.sizeof(_lib.SelectParams)
    assert lib.spot_struct_size(1) == C.sizeof(_lib.AttnParams)
    assert lib.spot_struct_size(2) == C.sizeof(_lib.DecodeStepHostParams)
    assert lib.spot_struct_size(3) == C.sizeof(_lib.ProjectParams)
    assert lib.spot_struct_size(4) == C.sizeof(_lib.DecodeStepParams)
    assert lib.spot_struct_size(5) == C.sizeof(_lib.TrainParams)
    assert lib.spot_struct_size(6) == 0
    assert [lib.spot_status_string(i) for i in range(5)] == [
        b"SPOT_OK", b"SPOT_ERR_INVALID_ARG", b"SPOT_ERR_UNSUPPORTED", b"SPOT_ERR_WORKSPACE_TOO_SMALL", b"SPOT_ERR_CUDA"]
    assert re.match(rb"\d+\.\d+$", lib.spot_version())


def test_selector_k_bytes_matches_the_papers_footprint(lib):
    """4.50 GiB BF16 for 128K tokens x 36 layers x 4 x 128 -> 1.20 GiB at 4.25 bit/element."""
    from paper_2606_22874_b200 import api
    n_tok = 131072 * 36
    bf16 = api.spot_selector_k_bytes("bf16", 1, n_tok, 4, 128)
    fp4 = api.spot_selector_k_bytes("mxfp4", 1, n_tok, 4, 128)
    int4 = api.spot_selector_k_bytes("int4_e4m3", 1, n_tok, 4, 128)
    assert bf16 == n_tok * 4 * 128 * 2 and abs(bf16 / 2 ** 30 - 4.50) < 1e-9
    assert fp4 == int4 == n_tok * 4 * 128 // 2 + n_tok * 4 * 128 // 32
    assert round(fp4 / 2 ** 30, 2) == 1.20
    # the measured geometry: 4 x 64, 136 B per token
    assert api.spot_selector_k_bytes("mxfp4", 4, 131072, 4, 64) == 4 * 131072 * 136
    assert api.spot_selector_k_bytes("fp8_e4m3", 1, n_tok, 4, 128) * 2 == bf16           # f2: the paper's 0.5x
    assert api.spot_selector_k_bytes("mxint8", 1, n_tok, 4, 128) * 32 == bf16 // 2 * 33   # 8.25 bit/elt (R38)
    assert api.spot_selector_k_bytes("int4_bf16s", 1, n_tok, 4, 128) * 32 == bf16 * 9     # 4.5 bit/elt: PAPER.md:188 (R39)
    # invalid: unknown format, d_idx not a multiple of 32, capacity not a multiple of the 64-token tile
    assert lib.spot_selector_k_bytes(7, 1, 64, 4, 64) == 0
    assert api.spot_selector_k_bytes("mxfp4", 1, 64, 4, 48) == 0
    assert api.spot_selector_k_bytes("mxfp4", 1, 100, 4, 64) == 0


def _select_params(**over):
    """A syntactically valid decode spot_select_params built from fake (aligned, never dereferenced) addresses."""
    from paper_2606_22874_b200 import _lib
    sp = _lib.SelectParams()
    sp.sel_q, sp.w, sp.sel_k, sp.seq_len = 0x1000, 0x2000, 0x3000, 0x4000
    sp.fmt, sp.cache_stride_tokens, sp.max_seq_len = 0, 4096, 4096
    sp.B, sp.Tq, sp.H_idx, sp.d_idx, sp.q_start, sp.blk, sp.q_block = 2, 1, 4, 64, 0, 64, 1
    sp.mode, sp.top_k, sp.p, sp.sink_blocks, sp.recency_blocks, sp.kmin_blocks, sp.temperature = 1, 0, 0.9, 1, 2, 8, 1.0
    sp.indices, sp.cap, sp.budgets, sp.nb_stride = 0x5000, 64, 0x6000, 64
    for k, v in over.items():
        setattr(sp, k, v)
    return sp


def test_select_argument_errors_are_caught_on_the_host(lib):
    INVALID, UNSUPPORTED = 1, 2
    assert lib.spot_select_workspace_bytes(C.byref(_select_params())) >= 2 * 64 * 4
    bad = [dict(sel_q=None), dict(w=None), dict(sel_k=None), dict(indices=None), dict(budgets=None),
           dict(seq_len=None), dict(sel_q=0x1008), dict(B=0), dict(max_seq_len=0), dict(max_seq_len=8192),
           dict(d_idx=48), dict(fmt=9), dict(mode=5), dict(p=0.0), dict(p=1.5), dict(temperature=0.0),
           dict(cap=63), dict(mode=0, top_k=2), dict(q_block=7), dict(sink_blocks=-1),
           dict(fmt=2, cache_stride_tokens=4100, max_seq_len=4096),
           dict(q_block=64, Tq=96, seq_len=None), dict(q_block=64, Tq=128, q_start=32, seq_len=None),
           dict(block_scores=0x7000, nb_stride=32)]
    for o in bad:
        sp = _select_params(**o)
        assert lib.spot_select(C.byref(sp), None) == INVALID, o
        assert lib.spot_select_workspace_bytes(C.byref(sp)) == 0, o
    assert lib.spot_select(C.byref(_select_params(blk=32)), None) == UNSUPPORTED
    # 16-token blocks (f3) are a decode geometry: accepted there (4x the blocks), not for 64-query prefill rows
    assert lib.spot_select_workspace_bytes(C.byref(_select_params(blk=16, cap=256, nb_stride=256))) >= 2 * 256 * 4
    assert lib.spot_select_workspace_bytes(C.byref(_select_params(blk=16, cap=256, nb_stride=256, q_block=64, Tq=64,
                                                                  seq_len=None))) > 0            # f3: prefill rows too
    # INT4 with BF16 group scales (f2, R39) is a decode-row format: its keys are not BF16 numbers, prefill rows are refused
    assert lib.spot_select_workspace_bytes(C.byref(_select_params(fmt=5))) > 0
    assert lib.spot_select(C.byref(_select_params(fmt=5, q_block=64, Tq=128, seq_len=None)), None) == UNSUPPORTED
    assert lib.spot_select(None, None) == INVALID
    assert lib.spot_score_blocks(C.byref(_select_params()), None) == INVALID        # block_scores is required
    # a score-only block (what spot_score_blocks reads: no indices / budgets / cap) can size its own workspace -- a
    # quantised cache in prefill needs the dequantised prefix (spot.h), a BF16 one nothing beyond the alignment slack
    so = dict(indices=None, budgets=None, cap=0, block_scores=0x7000, nb_stride=64, q_block=64, Tq=128, q_start=1024,
              seq_len=None)
    assert lib.spot_select_workspace_bytes(C.byref(_select_params(fmt=2, **so))) >= 2 * (1024 + 128) * 4 * 64 * 2
    assert 0 < lib.spot_select_workspace_bytes(C.byref(_select_params(fmt=0, **so))) <= 4096


def _attn_params(**over):
    from paper_2606_22874_b200 import _lib
    ap = _lib.AttnParams()
    ap.q, ap.k, ap.v, ap.out, ap.seq_len = 0x1000, 0x2000, 0x3000, 0x4000, 0x5000
    ap.kv_stride_batch, ap.kv_stride_token, ap.kv_stride_head = 8 * 4096 * 128, 128, 4096 * 128
    ap.max_seq_len, ap.indices, ap.budgets, ap.cap = 4096, 0x6000, 0x7000, 64
    ap.B, ap.Tq, ap.H_q, ap.H_kv, ap.D, ap.q_start, ap.blk, ap.sm_scale = 1, 1, 32, 8, 128, 0, 64, 0.088
    for k, v in over.items():
        setattr(ap, k, v)
    return ap


def test_attention_argument_errors_are_caught_on_the_host(lib):
    INVALID, UNSUPPORTED = 1, 2
    assert lib.spot_sparse_attn_decode_workspace_bytes(C.byref(_attn_params())) > 0
    for o in (dict(q=None), dict(out=None), dict(k=0x2004), dict(H_q=30), dict(B=0), dict(budgets=None),
              dict(seq_len=None), dict(max_seq_len=0), dict(kv_stride_token=100), dict(kv_stride_head=4)):
        ap = _attn_params(**o)
        assert lib.spot_sparse_attn_decode(C.byref(ap), None) == INVALID, o
        assert lib.spot_sparse_attn_decode_workspace_bytes(C.byref(ap)) == 0, o
    for o in (dict(D=64), dict(blk=32), dict(H_q=8 * 17)):
        assert lib.spot_sparse_attn_decode(C.byref(_attn_params(**o)), None) == UNSUPPORTED, o
    # prefill: chunk alignment (R26)
    for o in (dict(Tq=96), dict(Tq=128, q_start=32), dict(Tq=0)):
        assert lib.spot_sparse_attn_prefill(C.byref(_attn_params(**o)), None) == INVALID, o
    assert lib.spot_sparse_attn_decode_workspace_bytes(C.byref(_attn_params(blk=16))) > 0          # f3
    assert lib.spot_sparse_attn_prefill(C.byref(_attn_params(Tq=64, blk=32)), None) == UNSUPPORTED
    # paged K/V (f3): decode only; page size a multiple of 16, the table must cover max_seq_len, page stride a multiple
    # of the token stride
    paged = dict(page_table=0x8000, page_table_stride=64, page_tokens=64, kv_stride_batch=8 * 64 * 128)
    assert lib.spot_sparse_attn_decode_workspace_bytes(C.byref(_attn_params(**paged))) > 0
    for o in (dict(page_tokens=0), dict(page_tokens=40), dict(page_table_stride=63), dict(kv_stride_batch=8 * 64 * 128 + 8)):
        assert lib.spot_sparse_attn_decode(C.byref(_attn_params(**dict(paged, **o))), None) == INVALID, o
    assert lib.spot_sparse_attn_prefill_workspace_bytes(C.byref(_attn_params(Tq=64, **paged))) >= 0
    assert lib.spot_sparse_attn_prefill(C.byref(_attn_params(Tq=64, **dict(paged, page_tokens=32))), None) == UNSUPPORTED
    assert lib.spot_sparse_attn_prefill(C.byref(_attn_params(Tq=128, q_start=4096, **paged)), None) == INVALID   # table too short
    assert lib.spot_decode_step_host(None, None) == INVALID


def test_quantize_argument_errors(lib):
    INVALID = 1
    f = lib.spot_quantize_selector_k
    assert f(None, 0x2000, 2, 1, 64, 0, 64, 4, 64, None) == INVALID
    assert f(0x1000, 0x2000, 2, 1, 64, 0, 64, 4, 48, None) == INVALID           # d_idx % 32
    assert f(0x1000, 0x2000, 2, 1, 64, 64, 64, 4, 64, None) == INVALID          # past the capacity
    assert f(0x1000, 0x2000, 6, 1, 64, 0, 64, 4, 64, None) == INVALID           # unknown format
    assert lib.spot_dequantize_selector_k(0x1000, None, 2, 1, 64, 0, 64, 4, 64, None) == INVALID


def test_project_argument_errors(lib):
    from paper_2606_22874_b200 import _lib
    INVALID, WS = 1, 3

    def params(**over):
        pp = _lib.ProjectParams()
        pp.hidden, pp.w_q, pp.w_k, pp.w_w, pp.pos = 0x1000, 0x2000, 0x3000, 0x4000, 0x5000
        pp.B, pp.d_model, pp.H_idx, pp.d_idx, pp.rope_dims, pp.rope_base = 4, 4096, 4, 64, 64, 1e6
        pp.sel_q, pp.w, pp.sel_k, pp.fmt, pp.cache_stride_tokens = 0x6000, 0x7000, 0x8000, 2, 4096
        for k, v in over.items():
            setattr(pp, k, v)
        return pp
    assert lib.spot_selector_project_append_workspace_bytes(C.byref(params())) >= 4 * 4 * 64 * 2
    for o in (dict(hidden=None), dict(w_w=None), dict(pos=None), dict(sel_k=None), dict(w_q=0x2004), dict(B=0),
              dict(d_model=4000), dict(d_idx=48), dict(rope_dims=33), dict(rope_dims=128), dict(rope_base=0.0),
              dict(fmt=7), dict(cache_stride_tokens=100)):
        pp = params(**o)
        assert lib.spot_selector_project_append(C.byref(pp), None) == INVALID, o
        assert lib.spot_selector_project_append_workspace_bytes(C.byref(pp)) == 0, o
    assert lib.spot_selector_project_append(None, None) == INVALID


def test_binding_fails_loudly_without_the_library(monkeypatch):
    from paper_2606_22874_b200 import _lib
    monkeypatch.setattr(_lib, "_lib", None)
    monkeypatch.setattr(_lib, "LIB_PATH", os.path.join(ROOT, "no_such_dir", "libspot.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        _lib.load()


def test_header_is_plain_c99():
    """include/spot.h is the boundary: it must compile as C99 (no C++, no torch, no CUDA types in the signatures)."""
    import shutil
    import subprocess
    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("no gcc on this machine")
    hdr = os.path.join(ROOT, "include", "spot.h")
    r = subprocess.run([gcc, "-std=c99", "-Wall", "-Wextra", "-Werror", "-fsyntax-only", "-x", "c", hdr],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    src = open(hdr).read()
    assert "torch" not in src and "cuda_runtime" not in src and "cudaStream_t stream" not in src
