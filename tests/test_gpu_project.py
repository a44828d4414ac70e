"""GPU parity of the upstream step f1 (-m gpu): selector projections + RoPE + mixing weights + append of the new
token's key to the cache, against oracle/projection.py (fp64) on the same seeded bits.

q^I, k^I: the GPU accumulates BF16 products in fp32 and rounds once to BF16 -> within one BF16 ulp of the fp64 value
(|err| <= 2^-8 |ref| + 1e-6), and at least 99 % of the elements equal to the correctly rounded one.  w: fp32,
rtol 1e-5.  Cache: the slot pos[b] holds exactly what a0's quantiser makes of the GPU's BF16 k^I (bit-exact against
the oracle quantiser), every other slot is untouched."""
import numpy as np
import pytest

from oracle import projection as OP
from oracle import quant as OQ
from oracle.bf16 import bf16_bits_to_f64
from tests import _harness as H
from workloads import f32_to_bf16_bits, make_project_workload

pytestmark = pytest.mark.gpu

FMTS = ("bf16", "mxfp4", "int4_e4m3", "fp8_e4m3", "mxint8", "int4_bf16s")


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available()
    from paper_2606_22874_b200 import _lib
    _lib.load()
    return torch


def _run(torch, wl, fmt, stride, rope_dims, base, cache_init):
    from paper_2606_22874_b200 import api
    B, dm, Hh, d = wl["B"], wl["d_model"], wl["H_idx"], wl["d_idx"]
    dev = {k: H.dev_u16(wl[k]) for k in ("hidden", "w_q", "w_k", "w_w")}
    pos = torch.from_numpy(wl["pos"]).cuda()
    sel_q = torch.zeros((B, Hh, d), dtype=torch.int16, device="cuda")
    w = torch.zeros((B, Hh), device="cuda")
    init = H.dev_u16(cache_init)                                  # [B][stride][H][d] BF16 pattern
    if fmt == "bf16":
        cache = init.clone()
    else:
        cache = torch.zeros(api.spot_selector_k_bytes(fmt, B, stride, Hh, d), dtype=torch.uint8, device="cuda")
        api.spot_quantize_selector_k(init, cache, fmt, B, stride, 0, stride, Hh, d)
    pp = api.make_project_params(dev["hidden"], dev["w_q"], dev["w_k"], dev["w_w"], pos, B, dm, Hh, d,
                                 rope_dims=rope_dims, rope_base=base, sel_q=sel_q, w=w, sel_k=cache, fmt=fmt,
                                 cache_stride_tokens=stride)
    ws = torch.empty(api.spot_selector_project_append_workspace_bytes(pp), dtype=torch.uint8, device="cuda")
    pp.workspace, pp.workspace_bytes = ws.data_ptr(), ws.numel()
    api.spot_selector_project_append(pp)
    back = torch.zeros((B, stride, Hh, d), dtype=torch.int16, device="cuda")
    api.spot_dequantize_selector_k(cache, back, fmt, B, stride, 0, stride, Hh, d)
    torch.cuda.synchronize()
    return H.to_np_u16(sel_q), w.cpu().numpy(), H.to_np_u16(back)


@pytest.mark.parametrize("B,d_model,d_idx,rope_dims", [(4, 4096, 64, 64), (1, 4096, 128, 64), (11, 1024, 64, 32),
                                                        (3, 5120, 64, 0)])
def test_project_rope_append(torch_cuda, B, d_model, d_idx, rope_dims):
    torch = torch_cuda
    stride, base = 256, 1.0e6
    wl = make_project_workload(seed=6006 + B, B=B, d_model=d_model, d_idx=d_idx, L=131072)
    Hh = wl["H_idx"]
    slot = wl["pos"] % stride                                     # cache slots (positions are large, the test cache small)
    rng = np.random.default_rng(9)
    cache_init = f32_to_bf16_bits(rng.standard_normal((B, stride, Hh, d_idx), dtype=np.float32))
    # the kernel takes ONE position per sequence (rotation angle and cache slot); run it per role
    res = {}
    for fmt in FMTS:
        wl_f = dict(wl)
        wl_f["pos"] = slot.astype(np.int32)
        res[fmt] = _run(torch, wl_f, fmt, stride, rope_dims, base, cache_init)
    hid, Wq, Wk, Ww = (bf16_bits_to_f64(wl[k]) for k in ("hidden", "w_q", "w_k", "w_w"))
    q_gpu, w_gpu, back_bf16 = res["bf16"]
    exact = total = 0
    for b in range(B):
        q_ref, k_ref, w_ref = OP.project(hid[b], Wq, Wk, Ww, int(slot[b]), Hh, d_idx, rope_dims, base)
        k_gpu_bits = back_bf16[b, slot[b]]                        # BF16 cache: the slot IS the GPU's k^I
        for got_bits, ref in ((q_gpu[b], q_ref), (k_gpu_bits, k_ref)):
            got = bf16_bits_to_f64(got_bits)
            assert np.all(np.abs(got - ref) <= 2.0 ** -8 * np.abs(ref) + 1e-6), np.abs(got - ref).max()
            exact += int(np.sum(got == bf16_bits_to_f64(f32_to_bf16_bits(ref.astype(np.float32)))))
            total += ref.size
        assert np.allclose(w_gpu[b], w_ref, rtol=1e-5, atol=1e-6)
        for fmt in FMTS:
            q_f, w_f, back = res[fmt]
            assert np.array_equal(q_f, q_gpu) and np.array_equal(w_f, w_gpu)          # format-independent outputs
            want_slot = H.oracle_dequantised_view(fmt, k_gpu_bits)
            assert np.array_equal(bf16_bits_to_f64(back[b, slot[b]]), want_slot), (fmt, b)
            others = np.ones(stride, dtype=bool)
            others[slot[b]] = False
            assert np.array_equal(bf16_bits_to_f64(back[b, others]), H.oracle_dequantised_view(fmt, cache_init[b, others]))
    assert exact >= 0.99 * total, (exact, total)


def test_project_rotation_uses_the_large_position_and_skips_out_of_range_slots(torch_cuda):
    """positions up to 2^17 (fp64 angle), and a sequence whose slot lies outside the cache gets q and w but no write."""
    torch = torch_cuda
    B, stride = 3, 131072
    wl = make_project_workload(seed=6106, B=B, d_model=1024, d_idx=64, L=stride)
    wl["pos"] = np.array([131071, 65537, stride + 5], dtype=np.int32)
    Hh, d = wl["H_idx"], wl["d_idx"]
    cache_init = np.zeros((B, stride, Hh, d), dtype=np.uint16)
    q_gpu, w_gpu, back = _run(torch, wl, "bf16", stride, 64, 1.0e6, cache_init)
    hid, Wq, Wk, Ww = (bf16_bits_to_f64(wl[k]) for k in ("hidden", "w_q", "w_k", "w_w"))
    for b in range(B):
        q_ref, k_ref, _ = OP.project(hid[b], Wq, Wk, Ww, int(wl["pos"][b]), Hh, d, 64, 1.0e6)
        assert np.all(np.abs(bf16_bits_to_f64(q_gpu[b]) - q_ref) <= 2.0 ** -8 * np.abs(q_ref) + 1e-6)
        if wl["pos"][b] < stride:
            assert np.all(np.abs(bf16_bits_to_f64(back[b, wl["pos"][b]]) - k_ref) <= 2.0 ** -8 * np.abs(k_ref) + 1e-6)
            assert np.count_nonzero(back[b]) <= Hh * d
        else:
            assert np.count_nonzero(back[b]) == 0
