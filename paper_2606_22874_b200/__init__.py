"""paper_2606_22874_b200 -- SpotAttention's per-step hot path (selector scoring, dual top-p selection, block-sparse
GQA attention, 4-bit selector K-cache) as hand-written CUDA for B200 (sm_100a) behind the C ABI of include/spot.h.

`api` mirrors the C entry points one to one; `build` compiles libspot.so in-tree.  There is no CPU fallback: the
binding raises if the library is missing."""
from . import _lib  # noqa: F401

__all__ = ["api", "build", "_lib"]
