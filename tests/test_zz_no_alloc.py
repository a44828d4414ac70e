"""spot_sparse_attn_decode_static (include/spot.h): decode attention whose split-KV scratch is a `static __device__` array
inside the library, for callers that cannot allocate.  Checked against the existing workspace path (same kernels: bit for
bit, and so within the decode tests' tolerance) on calls in a row that share the array, and against the oracle.

Collected last on purpose (file name): the run is `pytest -x`, a failure here must not hide another test."""
import numpy as np
import pytest

from tests import _harness as H
from workloads import make_config

pytestmark = pytest.mark.gpu

MAX_ABS, MEAN_ABS = 2e-2, 2e-3            # the tolerance of tests/test_gpu_decode.py


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_22874_b200 import _lib
    _lib.load()          # fails loudly if libspot.so is missing: no fallback
    return torch


def _lists_and_params(torch, dd, lists, out, lse):
    wl, api = dd.wl, dd.api
    cap = max(len(x) for x in lists)
    idx = np.full((wl.B, cap), -1, dtype=np.int32)
    for b, x in enumerate(lists):
        idx[b, :len(x)] = x
    bud = np.array([len(x) for x in lists], dtype=np.int32)
    d_idx, d_bud = torch.from_numpy(idx).cuda(), torch.from_numpy(bud).cuda()
    ap = api.make_attn_params(dd.q, dd.K, dd.V, dd.kv_strides, dd.seq_len, dd.max_seq_len, d_idx, d_bud, cap, wl.B, 1,
                              wl.H_q, wl.H_kv, wl.D, blk=wl.blk, sm_scale=wl.sm_scale, out=out, lse=lse)
    return idx, bud, ap, (d_idx, d_bud)


def test_static_scratch_decode_matches_the_workspace_path(torch_cuda):
    torch = torch_cuda
    from paper_2606_22874_b200 import _lib, api
    cases = []
    for cfg in ("mini4", "cfg1", "mini4"):                 # two shapes alternating: the array always holds another call's partials
        wl = make_config(cfg)
        dd = H.DeviceDecode(wl, "bf16")
        lists = [H.oracle_select(wl, "bf16", b)[1].indices.tolist() for b in range(wl.B)]
        cases.append((wl, dd, lists))
    # the existing path first (caller-owned workspace)
    want = []
    for wl, dd, lists in cases:
        cap = max(len(x) for x in lists)
        idx = np.full((wl.B, cap), -1, dtype=np.int32)
        for b, x in enumerate(lists):
            idx[b, :len(x)] = x
        want.append(dd.attend(idx, np.array([len(x) for x in lists], dtype=np.int32)))
    # the static-scratch entry point: all calls in a row on one stream, no synchronisation and no allocation between the
    # launches of consecutive calls (outputs and parameter blocks are made up front)
    runs = []
    for wl, dd, lists in cases:
        out = torch.zeros((wl.B, wl.H_q, wl.D), dtype=torch.int16, device="cuda")
        lse = torch.zeros((wl.B, wl.H_q), device="cuda")
        idx, bud, ap, keep = _lists_and_params(torch, dd, lists, out, lse)
        assert 0 < api.spot_sparse_attn_decode_workspace_bytes(ap) <= _lib.SPOT_STATIC_SCRATCH_BYTES
        assert not ap.workspace and ap.workspace_bytes == 0          # nothing of the caller's is used as scratch
        runs.append((out, lse, ap, keep))
    torch.cuda.synchronize()
    mem_before = torch.cuda.memory_allocated()
    for _, _, ap, _ in runs:
        api.spot_sparse_attn_decode_static(ap)
    for _, _, ap, _ in runs[:2]:                                      # and the first two once more, over each other's leftovers
        api.spot_sparse_attn_decode_static(ap)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == mem_before
    for (wl, dd, lists), (w_out, w_lse), (out, lse, _, _) in zip(cases, want, runs):
        got = H.bf16_bits_to_f64(H.to_np_u16(out))
        err = np.abs(got - w_out)
        assert err.max() <= MAX_ABS and err.mean() <= MEAN_ABS, (wl.name, err.max(), err.mean())
        assert np.array_equal(got, w_out), (wl.name, err.max())      # the same kernels on the same grid: the same bits
        assert np.array_equal(lse.cpu().numpy(), w_lse)
        for b in range(wl.B):                                         # and the oracle, as the decode tests check it
            o_want, o_lse = H.oracle_attend(wl, b, lists[b])
            e = np.abs(got[b] - o_want)
            assert e.max() <= MAX_ABS and e.mean() <= MEAN_ABS, (wl.name, b, e.max(), e.mean())


def test_static_scratch_decode_refuses_what_does_not_fit(torch_cuda):
    """Beyond SPOT_STATIC_SCRATCH_BYTES the call returns SPOT_ERR_WORKSPACE_TOO_SMALL and launches nothing (outputs untouched);
    argument errors are the workspace form's."""
    torch = torch_cuda
    from paper_2606_22874_b200 import _lib, api
    B, H_q, H_kv, D, L = 32, 128, 8, 128, 128                         # G = 16: 2 (296 + 256) 16 * 520 B = 9.2 MB > 8 MiB
    q = torch.zeros((B, H_q, D), dtype=torch.int16, device="cuda")
    K = torch.zeros((B, H_kv, L, D), dtype=torch.int16, device="cuda")
    V = torch.zeros_like(K)
    seq_len = torch.full((B,), L, dtype=torch.int32, device="cuda")
    idx = torch.zeros((B, 2), dtype=torch.int32, device="cuda")
    idx[:, 1] = 1
    bud = torch.full((B,), 2, dtype=torch.int32, device="cuda")
    out = torch.full((B, H_q, D), 0x1234, dtype=torch.int16, device="cuda")
    ap = api.make_attn_params(q, K, V, (H_kv * L * D, D, L * D), seq_len, L, idx, bud, 2, B, 1, H_q, H_kv, D, blk=64,
                              sm_scale=D ** -0.5, out=out)
    assert api.spot_sparse_attn_decode_workspace_bytes(ap) > _lib.SPOT_STATIC_SCRATCH_BYTES
    with pytest.raises(api.SpotError) as e:
        api.spot_sparse_attn_decode_static(ap)
    assert "WORKSPACE_TOO_SMALL" in str(e.value)
    torch.cuda.synchronize()
    assert bool((out == 0x1234).all())
    ap.D = 64
    with pytest.raises(api.SpotError) as e:
        api.spot_sparse_attn_decode_static(ap)
    assert "UNSUPPORTED" in str(e.value)
