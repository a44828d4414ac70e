"""Thin Python binding of the C ABI in include/spot.h -- same names, argument marshalling only.

torch supplies device memory (`tensor.data_ptr()`) and the stream; every step of the path runs in libspot.so.
BF16 tensors may be torch.bfloat16 or raw bit patterns (torch.uint16 / int16)."""
import ctypes as C

import torch

from . import _lib as L
from ._lib import (AttnParams, DecodeStepHostParams, DecodeStepParams, ProjectParams, SelectParams, TrainParams,  # noqa: F401
                   FORMATS, MODES)


class SpotError(RuntimeError):
    def __init__(self, status, where):
        lib = L.load()
        name = lib.spot_status_string(status).decode()
        extra = ""
        if status == L.SPOT_ERR_CUDA:
            extra = " (cudaError %d)" % lib.spot_last_cuda_error()
        super().__init__("%s: %s%s" % (where, name, extra))
        self.status = status


def _check(status, where):
    if status != L.SPOT_OK:
        raise SpotError(status, where)


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _fmt(fmt):
    return FORMATS[fmt] if isinstance(fmt, str) else int(fmt)


def spot_version():
    return L.load().spot_version().decode()


def spot_selector_k_bytes(fmt, B, cache_stride_tokens, H_idx, d_idx):
    return int(L.load().spot_selector_k_bytes(_fmt(fmt), B, cache_stride_tokens, H_idx, d_idx))


def spot_quantize_selector_k(k_bf16, k_cache, fmt, B, n_tokens, token_offset, cache_stride_tokens, H_idx, d_idx,
                             stream=None):
    _check(L.load().spot_quantize_selector_k(_ptr(k_bf16), _ptr(k_cache), _fmt(fmt), B, n_tokens, token_offset,
                                             cache_stride_tokens, H_idx, d_idx, _stream(stream)),
           "spot_quantize_selector_k")


def spot_dequantize_selector_k(k_cache, k_bf16_out, fmt, B, n_tokens, token_offset, cache_stride_tokens, H_idx,
                               d_idx, stream=None):
    _check(L.load().spot_dequantize_selector_k(_ptr(k_cache), _ptr(k_bf16_out), _fmt(fmt), B, n_tokens, token_offset,
                                               cache_stride_tokens, H_idx, d_idx, _stream(stream)),
           "spot_dequantize_selector_k")


def make_select_params(sel_q, w, sel_k, fmt, cache_stride_tokens, seq_len, max_seq_len, B, Tq, H_idx, d_idx, *,
                       q_start=0, blk=64, q_block=1, mode="dual_topp", top_k=0, p=0.9, sink_blocks=1,
                       recency_blocks=2, kmin_blocks=8, temperature=1.0, indices=None, cap=0, budgets=None,
                       block_scores=None, block_probs=None, nb_stride=0, workspace=None, q_fmt="bf16"):
    sp = SelectParams()
    sp.q_fmt = _fmt(q_fmt)
    sp.sel_q, sp.w, sp.sel_k = sel_q.data_ptr(), w.data_ptr(), sel_k.data_ptr()
    sp.fmt = _fmt(fmt)
    sp.cache_stride_tokens = cache_stride_tokens
    sp.seq_len = seq_len.data_ptr() if seq_len is not None else None
    sp.max_seq_len = max_seq_len
    sp.B, sp.Tq, sp.H_idx, sp.d_idx = B, Tq, H_idx, d_idx
    sp.q_start, sp.blk, sp.q_block = q_start, blk, q_block
    sp.mode = MODES[mode] if isinstance(mode, str) else int(mode)
    sp.top_k, sp.p = top_k, float(p)
    sp.sink_blocks, sp.recency_blocks, sp.kmin_blocks = sink_blocks, recency_blocks, kmin_blocks
    sp.temperature = float(temperature)
    sp.indices = indices.data_ptr() if indices is not None else None
    sp.cap = cap
    sp.budgets = budgets.data_ptr() if budgets is not None else None
    sp.block_scores = block_scores.data_ptr() if block_scores is not None else None
    sp.block_probs = block_probs.data_ptr() if block_probs is not None else None
    sp.nb_stride = nb_stride
    if workspace is not None:
        sp.workspace, sp.workspace_bytes = workspace.data_ptr(), workspace.numel() * workspace.element_size()
    return sp


def spot_select_workspace_bytes(sp):
    return int(L.load().spot_select_workspace_bytes(C.byref(sp)))


def spot_select(sp, stream=None):
    _check(L.load().spot_select(C.byref(sp), _stream(stream)), "spot_select")


def spot_score_blocks(sp, stream=None):
    _check(L.load().spot_score_blocks(C.byref(sp), _stream(stream)), "spot_score_blocks")


def make_attn_params(q, k, v, kv_strides, seq_len, max_seq_len, indices, budgets, cap, B, Tq, H_q, H_kv, D, *,
                     q_start=0, blk=64, sm_scale=None, out=None, lse=None, workspace=None, page_table=None,
                     page_tokens=0):
    ap = AttnParams()
    ap.q, ap.k, ap.v = q.data_ptr(), k.data_ptr(), v.data_ptr()
    ap.kv_stride_batch, ap.kv_stride_token, ap.kv_stride_head = kv_strides
    ap.seq_len = seq_len.data_ptr() if seq_len is not None else None
    ap.max_seq_len = max_seq_len
    ap.indices = indices.data_ptr() if indices is not None else None
    ap.budgets = budgets.data_ptr() if budgets is not None else None
    ap.cap = cap
    ap.B, ap.Tq, ap.H_q, ap.H_kv, ap.D = B, Tq, H_q, H_kv, D
    ap.q_start, ap.blk = q_start, blk
    ap.sm_scale = float(D ** -0.5 if sm_scale is None else sm_scale)
    ap.out = out.data_ptr() if out is not None else None
    ap.lse = lse.data_ptr() if lse is not None else None
    if workspace is not None:
        ap.workspace, ap.workspace_bytes = workspace.data_ptr(), workspace.numel() * workspace.element_size()
    if page_table is not None:
        ap.page_table, ap.page_table_stride, ap.page_tokens = page_table.data_ptr(), page_table.shape[1], page_tokens
    return ap


def spot_sparse_attn_decode_workspace_bytes(ap):
    return int(L.load().spot_sparse_attn_decode_workspace_bytes(C.byref(ap)))


def spot_sparse_attn_decode(ap, stream=None):
    _check(L.load().spot_sparse_attn_decode(C.byref(ap), _stream(stream)), "spot_sparse_attn_decode")


def spot_sparse_attn_decode_static(ap, stream=None):
    _check(L.load().spot_sparse_attn_decode_static(C.byref(ap), _stream(stream)), "spot_sparse_attn_decode_static")


def spot_dense_attn_decode_workspace_bytes(ap):
    return int(L.load().spot_dense_attn_decode_workspace_bytes(C.byref(ap)))


def spot_dense_attn_decode(ap, stream=None):
    _check(L.load().spot_dense_attn_decode(C.byref(ap), _stream(stream)), "spot_dense_attn_decode")


def spot_sparse_attn_prefill_workspace_bytes(ap):
    return int(L.load().spot_sparse_attn_prefill_workspace_bytes(C.byref(ap)))


def spot_sparse_attn_prefill(ap, stream=None):
    _check(L.load().spot_sparse_attn_prefill(C.byref(ap), _stream(stream)), "spot_sparse_attn_prefill")


def make_decode_step_params(sp, ap, workspace=None):
    dp = DecodeStepParams()
    dp.select, dp.attn = sp, ap
    if workspace is not None:
        dp.workspace, dp.workspace_bytes = workspace.data_ptr(), workspace.numel() * workspace.element_size()
    return dp


def spot_decode_step_workspace_bytes(dp):
    return int(L.load().spot_decode_step_workspace_bytes(C.byref(dp)))


def spot_decode_step(dp, stream=None):
    _check(L.load().spot_decode_step(C.byref(dp), _stream(stream)), "spot_decode_step")


def spot_decode_step_host(hp, stream=None):
    _check(L.load().spot_decode_step_host(C.byref(hp), _stream(stream)), "spot_decode_step_host")


def make_project_params(hidden, w_q, w_k, w_w, pos, B, d_model, H_idx, d_idx, *, rope_dims=64, rope_base=1.0e6,
                        sel_q=None, w=None, sel_k=None, fmt="bf16", cache_stride_tokens=0, workspace=None):
    pp = ProjectParams()
    pp.hidden, pp.w_q, pp.w_k, pp.w_w, pp.pos = (t.data_ptr() for t in (hidden, w_q, w_k, w_w, pos))
    pp.B, pp.d_model, pp.H_idx, pp.d_idx, pp.rope_dims = B, d_model, H_idx, d_idx, rope_dims
    pp.rope_base = float(rope_base)
    pp.sel_q, pp.w, pp.sel_k = sel_q.data_ptr(), w.data_ptr(), sel_k.data_ptr()
    pp.fmt = _fmt(fmt)
    pp.cache_stride_tokens = cache_stride_tokens
    if workspace is not None:
        pp.workspace, pp.workspace_bytes = workspace.data_ptr(), workspace.numel() * workspace.element_size()
    return pp


def spot_selector_project_append_workspace_bytes(pp):
    return int(L.load().spot_selector_project_append_workspace_bytes(C.byref(pp)))


def spot_selector_project_append(pp, stream=None):
    _check(L.load().spot_selector_project_append(C.byref(pp), _stream(stream)), "spot_selector_project_append")


def make_train_params(q, k, k_strides, sel_q, w, sel_k, L, H_q, H_kv, D, H_idx, d_idx, *, blk=16, top_k=512, sink_blocks=0,
                      recency_blocks=0, sm_scale=None, dense_kl=None, sparse_kl=None, teacher_lse=None, indices=None,
                      budgets=None, cap=0, workspace=None):
    tp = TrainParams()
    tp.q, tp.k = q.data_ptr(), k.data_ptr()
    tp.k_stride_token, tp.k_stride_head = k_strides
    tp.sel_q, tp.w, tp.sel_k = sel_q.data_ptr(), w.data_ptr(), sel_k.data_ptr()
    tp.L, tp.H_q, tp.H_kv, tp.D, tp.H_idx, tp.d_idx = L, H_q, H_kv, D, H_idx, d_idx
    tp.blk, tp.top_k, tp.sink_blocks, tp.recency_blocks = blk, top_k, sink_blocks, recency_blocks
    tp.sm_scale = float(D ** -0.5 if sm_scale is None else sm_scale)
    tp.dense_kl, tp.sparse_kl = dense_kl.data_ptr(), sparse_kl.data_ptr()
    tp.teacher_lse = teacher_lse.data_ptr() if teacher_lse is not None else None
    tp.indices = indices.data_ptr() if indices is not None else None
    tp.budgets = budgets.data_ptr() if budgets is not None else None
    tp.cap = cap
    if workspace is not None:
        tp.workspace, tp.workspace_bytes = workspace.data_ptr(), workspace.numel() * workspace.element_size()
    return tp


def spot_train_kl_workspace_bytes(tp):
    return int(L.load().spot_train_kl_workspace_bytes(C.byref(tp)))


def spot_train_kl(tp, stream=None):
    _check(L.load().spot_train_kl(C.byref(tp), _stream(stream)), "spot_train_kl")
