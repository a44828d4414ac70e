"""-m gpu: guard bands around every buffer the decode step writes, and run-to-run bit equality of the decode step and the
prefill pass (tests/sanitize_smoke.py; what stands in for compute-sanitizer, which is closed on this GPU pool --
profiles/r2_sanitizers.md)."""
import pytest

pytestmark = pytest.mark.gpu


def test_guard_bands_and_determinism():
    import torch
    assert torch.cuda.is_available()
    from paper_2606_22874_b200 import _lib
    _lib.load()
    from tests import sanitize_smoke
    sanitize_smoke.guarded_cases()


def test_every_kernel_family_runs_on_tiny_inputs():
    from tests import sanitize_smoke
    sanitize_smoke.decode_cases()
    sanitize_smoke.prefill_cases()
