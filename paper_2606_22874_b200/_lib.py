"""ctypes view of libspot.so: structs and prototypes exactly as include/spot.h declares them.

No arithmetic of the method lives here (or anywhere in Python): every step runs in the CUDA kernels behind the
C ABI.  Importing this module builds nothing; loading fails loudly if the library is missing."""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libspot.so")

SPOT_OK, SPOT_ERR_INVALID_ARG, SPOT_ERR_UNSUPPORTED, SPOT_ERR_WORKSPACE_TOO_SMALL, SPOT_ERR_CUDA = range(5)
SPOT_SELK_BF16, SPOT_SELK_INT4_E4M3, SPOT_SELK_MXFP4, SPOT_SELK_FP8_E4M3, SPOT_SELK_MXINT8, SPOT_SELK_INT4_BF16S = range(6)
SPOT_MODE_TOPK, SPOT_MODE_DUAL_TOPP = range(2)
SPOT_STATIC_SCRATCH_BYTES = 8 << 20

FORMATS = {"bf16": SPOT_SELK_BF16, "int4_e4m3": SPOT_SELK_INT4_E4M3, "mxfp4": SPOT_SELK_MXFP4,
           "fp8_e4m3": SPOT_SELK_FP8_E4M3, "mxint8": SPOT_SELK_MXINT8, "int4_bf16s": SPOT_SELK_INT4_BF16S}
MODES = {"topk": SPOT_MODE_TOPK, "dual_topp": SPOT_MODE_DUAL_TOPP}


class SelectParams(C.Structure):
    _fields_ = [
        ("sel_q", C.c_void_p), ("w", C.c_void_p), ("sel_k", C.c_void_p), ("fmt", C.c_int32),
        ("cache_stride_tokens", C.c_int64), ("seq_len", C.c_void_p), ("max_seq_len", C.c_int32),
        ("B", C.c_int32), ("Tq", C.c_int32), ("H_idx", C.c_int32), ("d_idx", C.c_int32),
        ("q_start", C.c_int32), ("blk", C.c_int32), ("q_block", C.c_int32),
        ("mode", C.c_int32), ("top_k", C.c_int32), ("p", C.c_double),
        ("sink_blocks", C.c_int32), ("recency_blocks", C.c_int32), ("kmin_blocks", C.c_int32),
        ("temperature", C.c_double),
        ("indices", C.c_void_p), ("cap", C.c_int32), ("budgets", C.c_void_p),
        ("block_scores", C.c_void_p), ("block_probs", C.c_void_p), ("nb_stride", C.c_int32),
        ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
        ("q_fmt", C.c_int32),
    ]


class AttnParams(C.Structure):
    _fields_ = [
        ("q", C.c_void_p), ("k", C.c_void_p), ("v", C.c_void_p),
        ("kv_stride_batch", C.c_int64), ("kv_stride_token", C.c_int64), ("kv_stride_head", C.c_int64),
        ("seq_len", C.c_void_p), ("max_seq_len", C.c_int32),
        ("indices", C.c_void_p), ("budgets", C.c_void_p), ("cap", C.c_int32),
        ("B", C.c_int32), ("Tq", C.c_int32), ("H_q", C.c_int32), ("H_kv", C.c_int32), ("D", C.c_int32),
        ("q_start", C.c_int32), ("blk", C.c_int32), ("sm_scale", C.c_float),
        ("out", C.c_void_p), ("lse", C.c_void_p),
        ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
        ("page_table", C.c_void_p), ("page_table_stride", C.c_int32), ("page_tokens", C.c_int32),
    ]


class DecodeStepHostParams(C.Structure):
    _fields_ = [
        ("sel_q_host", C.c_void_p), ("w_host", C.c_void_p), ("q_host", C.c_void_p),
        ("out_host", C.c_void_p), ("budgets_host", C.c_void_p),
        ("select", SelectParams), ("attn", AttnParams),
        ("step_workspace", C.c_void_p), ("step_workspace_bytes", C.c_size_t),
    ]


class DecodeStepParams(C.Structure):
    _fields_ = [
        ("select", SelectParams), ("attn", AttnParams),
        ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
    ]


class ProjectParams(C.Structure):
    _fields_ = [
        ("hidden", C.c_void_p), ("w_q", C.c_void_p), ("w_k", C.c_void_p), ("w_w", C.c_void_p), ("pos", C.c_void_p),
        ("B", C.c_int32), ("d_model", C.c_int32), ("H_idx", C.c_int32), ("d_idx", C.c_int32), ("rope_dims", C.c_int32),
        ("rope_base", C.c_float),
        ("sel_q", C.c_void_p), ("w", C.c_void_p), ("sel_k", C.c_void_p), ("fmt", C.c_int32),
        ("cache_stride_tokens", C.c_int64),
        ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
    ]


class TrainParams(C.Structure):
    _fields_ = [
        ("q", C.c_void_p), ("k", C.c_void_p), ("k_stride_token", C.c_int64), ("k_stride_head", C.c_int64),
        ("sel_q", C.c_void_p), ("w", C.c_void_p), ("sel_k", C.c_void_p),
        ("L", C.c_int32), ("H_q", C.c_int32), ("H_kv", C.c_int32), ("D", C.c_int32), ("H_idx", C.c_int32), ("d_idx", C.c_int32),
        ("blk", C.c_int32), ("top_k", C.c_int32), ("sink_blocks", C.c_int32), ("recency_blocks", C.c_int32),
        ("sm_scale", C.c_float),
        ("dense_kl", C.c_void_p), ("sparse_kl", C.c_void_p), ("teacher_lse", C.c_void_p),
        ("indices", C.c_void_p), ("budgets", C.c_void_p), ("cap", C.c_int32),
        ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
    ]


# every symbol include/spot.h declares: name -> (restype, argtypes)
PROTOTYPES = {
    "spot_status_string": (C.c_char_p, [C.c_int]),
    "spot_last_cuda_error": (C.c_int, []),
    "spot_version": (C.c_char_p, []),
    "spot_struct_size": (C.c_size_t, [C.c_int]),
    "spot_selector_k_bytes": (C.c_size_t, [C.c_int, C.c_int64, C.c_int64, C.c_int, C.c_int]),
    "spot_quantize_selector_k": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int64, C.c_int64, C.c_int64,
                                           C.c_int64, C.c_int, C.c_int, C.c_void_p]),
    "spot_dequantize_selector_k": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int64, C.c_int64, C.c_int64,
                                             C.c_int64, C.c_int, C.c_int, C.c_void_p]),
    "spot_select_workspace_bytes": (C.c_size_t, [C.POINTER(SelectParams)]),
    "spot_select": (C.c_int, [C.POINTER(SelectParams), C.c_void_p]),
    "spot_score_blocks": (C.c_int, [C.POINTER(SelectParams), C.c_void_p]),
    "spot_sparse_attn_decode_workspace_bytes": (C.c_size_t, [C.POINTER(AttnParams)]),
    "spot_sparse_attn_decode": (C.c_int, [C.POINTER(AttnParams), C.c_void_p]),
    "spot_sparse_attn_prefill_workspace_bytes": (C.c_size_t, [C.POINTER(AttnParams)]),
    "spot_sparse_attn_prefill": (C.c_int, [C.POINTER(AttnParams), C.c_void_p]),
    "spot_sparse_attn_decode_static": (C.c_int, [C.POINTER(AttnParams), C.c_void_p]),
    "spot_dense_attn_decode_workspace_bytes": (C.c_size_t, [C.POINTER(AttnParams)]),
    "spot_dense_attn_decode": (C.c_int, [C.POINTER(AttnParams), C.c_void_p]),
    "spot_decode_step_host": (C.c_int, [C.POINTER(DecodeStepHostParams), C.c_void_p]),
    "spot_decode_step_workspace_bytes": (C.c_size_t, [C.POINTER(DecodeStepParams)]),
    "spot_decode_step": (C.c_int, [C.POINTER(DecodeStepParams), C.c_void_p]),
    "spot_selector_project_append_workspace_bytes": (C.c_size_t, [C.POINTER(ProjectParams)]),
    "spot_selector_project_append": (C.c_int, [C.POINTER(ProjectParams), C.c_void_p]),
    "spot_train_kl_workspace_bytes": (C.c_size_t, [C.POINTER(TrainParams)]),
    "spot_train_kl": (C.c_int, [C.POINTER(TrainParams), C.c_void_p]),
}

_lib = None


def load():
    """dlopen libspot.so (built in-tree by paper_2606_22874_b200.build).  Raises if it is missing: there is no
    fallback path."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libspot.so is not built: run `python -m paper_2606_22874_b200.build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        lib = C.CDLL(LIB_PATH)
        for name, (res, args) in PROTOTYPES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        for which, st in enumerate((SelectParams, AttnParams, DecodeStepHostParams, ProjectParams, DecodeStepParams, TrainParams)):
            if lib.spot_struct_size(which) != C.sizeof(st):
                raise RuntimeError("ABI mismatch: %s is %d bytes in libspot.so, %d in the binding"
                                   % (st.__name__, lib.spot_struct_size(which), C.sizeof(st)))
        _lib = lib
    return _lib
