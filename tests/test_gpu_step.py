"""GPU parity, the one-call decode step (-m gpu): spot_decode_step = a1 + a2 + a3 launched as overlapping kernels (the
selection of sequence b beside the scoring of b + 1.., attention over the first B - 1 sequences before the last list is
needed; include/spot.h).  Same arithmetic as spot_select + spot_sparse_attn_decode: the index
lists and budgets must equal the oracle's, the attention output must be within the north_star tolerance of the oracle on
that list.  The hand-off words live in an uninitialised workspace, re-armed by every call: repeated calls, a workspace
full of garbage, and the replay of a captured graph are covered."""
import numpy as np
import pytest

from tests import _harness as H
from workloads import make_config, make_decode_workload

pytestmark = pytest.mark.gpu

MAX_ABS, MEAN_ABS = 2e-2, 2e-3
F3 = dict(blk=16, sink_blocks=8, recency_blocks=16, kmin_blocks=32)


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_22874_b200 import _lib
    _lib.load()
    return torch


def _check_step(dd, fmt, idx, bud, out, lse, every=1, **over):
    wl = dd.wl
    for b in range(0, wl.B, every):
        s_bar, sel = H.oracle_select(wl, fmt, b, **over)
        cls = H.classify_selection(s_bar, sel, idx[b], int(bud[b]), over.get("p", wl.p) if wl.mode == "dual_topp" else None)
        assert cls == "exact", (wl.name, fmt, b, cls)
        assert np.all(idx[b, int(bud[b]):] == -1)
        want, want_lse = H.oracle_attend(wl, b, sel.indices)
        err = np.abs(out[b] - want)
        assert err.max() <= MAX_ABS and err.mean() <= MEAN_ABS, (wl.name, b, err.max(), err.mean())
        assert np.abs(lse[b] - want_lse).max() <= 1e-3


@pytest.mark.parametrize("cfg,fmt,over", [("cfg1", "bf16", {}), ("mini2", "bf16", {}), ("mini2", "mxfp4", {}),
                                          ("mini4", "int4_e4m3", {}), ("mini4", "fp8_e4m3", {}), ("mini3", "bf16", {}),
                                          ("mini2", "bf16", F3), ("mini4", "mxfp4", F3),
                                          ("mini2", "mxint8", {}), ("mini4", "int4_bf16s", F3)])
def test_step_matches_oracle(torch_cuda, cfg, fmt, over):
    from paper_2606_22874_b200 import api
    wl = make_config(cfg, **over)
    dd = H.DeviceDecode(wl, fmt)
    dp = dd.step_params(garbage=0xAB)                  # the workspaces need not be initialised
    api.spot_decode_step(dp)
    idx, bud, out, lse = dd.step_results()
    _check_step(dd, fmt, idx, bud, out, lse)
    # the same block again (fresh token, re-armed words), then with other rule parameters on the same workspaces
    first = (idx.copy(), bud.copy(), out.copy())
    for _ in range(3):
        api.spot_decode_step(dp)
    idx2, bud2, out2, _ = dd.step_results()
    assert np.array_equal(idx2, first[0]) and np.array_equal(bud2, first[1]) and np.array_equal(out2, first[2])
    if wl.mode == "dual_topp":
        dp.select.p = 0.7
        api.spot_decode_step(dp)
        idx, bud, out, lse = dd.step_results()
        _check_step(dd, fmt, idx, bud, out, lse, p=0.7)


def test_step_equals_the_separate_calls(torch_cuda):
    """spot_select + spot_sparse_attn_decode on the same inputs: identical lists and budgets; outputs agree to the
    rounding of a different split of the same sums (the stream-K cut differs)."""
    from paper_2606_22874_b200 import api
    wl = make_config("mini4")
    dd = H.DeviceDecode(wl, "mxfp4")
    dp = dd.step_params()
    api.spot_decode_step(dp)
    idx, bud, out, lse = dd.step_results()
    idx_s, bud_s, _, _ = dd.select(want_probs=False)
    out_s, lse_s = dd.attend(idx_s, bud_s)
    assert np.array_equal(idx, idx_s) and np.array_equal(bud, bud_s)
    assert np.abs(out - out_s).max() <= 2e-2 and np.abs(lse - lse_s).max() <= 1e-4


def test_step_many_short_sequences(torch_cuda):
    """B = 40 ragged sequences (1 .. 36 blocks): more selection rows than SMs left to them, sequences shorter than the
    scoring grid, sequences shorter than the reserved tier."""
    from paper_2606_22874_b200 import api
    rng = np.random.default_rng(17)
    seqs = rng.integers(1, 2304, size=40).tolist()
    seqs[0], seqs[1], seqs[2], seqs[39] = 1, 64, 2304, 3
    wl = make_decode_workload("many", 23, B=40, L=2304, kind="zipf", seq_lens=seqs)
    for fmt in ("bf16", "mxfp4"):
        dd = H.DeviceDecode(wl, fmt)
        dp = dd.step_params(garbage=0x5C)
        api.spot_decode_step(dp)
        idx, bud, out, lse = dd.step_results()
        _check_step(dd, fmt, idx, bud, out, lse, every=3)


def test_step_is_capturable_in_a_cuda_graph(torch_cuda):
    """A replay carries the same token as the capture: it relies on every call leaving the hand-off words re-armed."""
    torch = torch_cuda
    from paper_2606_22874_b200 import api
    wl = make_config("mini2")
    dd = H.DeviceDecode(wl, "mxfp4")
    dp = dd.step_params(garbage=0xEE)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        api.spot_decode_step(dp, s)
    s.synchronize()
    ref = [t.clone() for t in (dd.indices, dd.budgets, dd.out)]
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        api.spot_decode_step(dp, torch.cuda.current_stream())
    for _ in range(4):
        dd.indices.zero_(); dd.budgets.zero_(); dd.out.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(dd.indices, ref[0]) and torch.equal(dd.budgets, ref[1]) and torch.equal(dd.out, ref[2])
    api.spot_decode_step(dp)                           # an eager call after the replays (new token) still works
    idx, bud, out, lse = dd.step_results()
    _check_step(dd, "mxfp4", idx, bud, out, lse)


def test_step_argument_errors(torch_cuda):
    from paper_2606_22874_b200 import api
    wl = make_config("mini2")
    dd = H.DeviceDecode(wl, "bf16")
    dp = dd.step_params()
    assert api.spot_decode_step_workspace_bytes(dp) > 0
    dp.attn.cap = dp.select.cap - 1                    # the two blocks must describe one step
    assert api.spot_decode_step_workspace_bytes(dp) == 0
    with pytest.raises(api.SpotError, match="INVALID_ARG"):
        api.spot_decode_step(dp)
    dp.attn.cap = dp.select.cap
    dp.workspace_bytes = 8
    with pytest.raises(api.SpotError, match="WORKSPACE"):
        api.spot_decode_step(dp)
