"""Pins for oracle/quant.py (step a0) -- none of them re-types the oracle's own formula.

* footprints the paper prints;
* the golden group and E4M3 spot values (tests/golden);
* "nearest representable value, ties to even" by brute force over the whole code book with
  exact rationals -- an independent definition of RNE, against the oracle's threshold chains;
* exact round trips on grid-valued groups; error bounds; BF16-exactness of dequantised keys.
"""
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import quant
from oracle.bf16 import bf16_bits_to_f64, f64_to_bf16_bits_exact
from workloads.bf16 import f32_to_bf16_bits


def _bits(vals):
    return f32_to_bf16_bits(np.asarray(vals, dtype=np.float32))


def test_footprints_printed_by_the_paper(golden):
    g = golden("footprint.txt")
    n = int(g["tokens"][0][0]) * int(g["layers"][0][0]) * int(g["h_idx"][0][0]) * int(g["d_idx"][0][0])
    GiB = 2.0 ** 30
    assert quant.selector_k_bytes("bf16", n) / GiB == pytest.approx(float(g["bf16_gib"][0][0]), abs=0.005)
    assert quant.selector_k_bytes("bf16", n) == 131072 * 36 * 4 * 128 * 2
    # 1.27 GiB <=> 4.5 bit/elt (16-bit group metadata); 1.20 GiB <=> 4.25 bit/elt (8-bit scale)
    assert quant.selector_k_bytes("int4_scale16", n) / GiB == pytest.approx(float(g["int4_gib"][0][0]), abs=0.005)
    assert quant.selector_k_bytes("mxfp4", n) / GiB == pytest.approx(float(g["fp4_gib"][0][0]), abs=0.005)
    assert quant.selector_k_bytes("int4_scale16", n) / quant.selector_k_bytes("bf16", n) == \
        pytest.approx(float(g["ratio_4p5bit"][0][0]), abs=0.0005)
    assert quant.selector_k_bytes("int4_e4m3", n) * 32 == n * 17           # 4.25 bit/elt
    # BASELINE.json geometry: 4 heads x 64 -> 512 B/token BF16, 136 B/token 4-bit
    assert quant.selector_k_bytes("bf16", 256) == 512
    assert quant.selector_k_bytes("mxfp4", 256) == 136


def _golden_group():
    v = [(i - 15.5) * 0.17 * (1.3 if i % 5 == 0 else 1.0) for i in range(32)]
    return _bits(v)


def test_golden_group_mxfp4(golden):
    g = golden("quant_group.txt")
    bits = _golden_group()
    vals = bf16_bits_to_f64(bits)
    assert np.abs(vals).max() == float(g["amax"][0][0])
    codes, scale = quant.quantize_mxfp4(bits)
    assert scale.tolist() == [int(g["mxfp4_scale"][0][0])]
    assert "".join("%x" % c for c in codes) == g["mxfp4_codes"][0][0]
    dq = quant.dequantize_mxfp4(codes, scale)
    assert np.abs(dq - vals).max() == float(g["mxfp4_max_abs_err"][0][0])


def test_golden_group_int4(golden):
    g = golden("quant_group.txt")
    bits = _golden_group()
    vals = bf16_bits_to_f64(bits)
    q, code = quant.quantize_int4_e4m3(bits)
    assert code.tolist() == [int(g["int4_scale_code"][0][0], 16)]
    assert q.tolist() == [int(x) for x in g["int4_q"][0]]
    dq = quant.dequantize_int4_e4m3(q, code)
    assert np.abs(dq - vals).max() == pytest.approx(float(g["int4_max_abs_err"][0][0]), abs=5e-6)


def test_e4m3_spot_values(golden):
    here = os.path.dirname(os.path.abspath(__file__))
    with open(os.path.join(here, "golden", "e4m3_spot.txt")) as f:
        rows = [l.split() for l in f if l.strip() and not l.startswith("#")]
    for val, code in rows:
        got = int(quant.encode_e4m3_rne_satfinite(np.float32(float(val))))
        assert got == int(code, 16), (val, hex(got), code)


# ---- brute-force "nearest representable, ties to even" with exact rationals -----------------

def _e4m3_table():
    tab = []
    for code in range(0x7F):
        E, m = code >> 3, code & 7
        v = Fraction(m, 512) if E == 0 else Fraction(8 + m, 8) * Fraction(2) ** (E - 7)
        tab.append((v, code))
    return tab


def _nearest_even(x, table):
    """table: ascending [(value, code)]; ties -> even code (even mantissa lsb)."""
    best = None
    for v, c in table:
        d = abs(x - v)
        if best is None or d < best[0] or (d == best[0] and c % 2 == 0 and best[1] % 2 == 1):
            best = (d, c)
    return best[1]


def test_e4m3_value_table_is_the_ocp_format():
    v = quant.e4m3_value(np.arange(0x7F))
    assert v[0] == 0 and v[1] == 2.0 ** -9 and v[7] == 7 * 2.0 ** -9
    assert v[8] == 2.0 ** -6 and v[0x38] == 1.0 and v[0x30] == 0.5 and v[0x7E] == 448.0
    assert np.all(np.diff(v) > 0)
    tab = _e4m3_table()
    assert [float(t[0]) for t in tab] == v.tolist()


def test_e4m3_encode_matches_bruteforce_rne():
    tab = _e4m3_table()
    rng = np.random.default_rng(7)
    xs = list(np.exp(rng.uniform(np.log(2.0 ** -12), np.log(600.0), 3000)).astype(np.float32))
    vals = [float(t[0]) for t in tab]
    # every exact value, every midpoint (ties), and neighbours of midpoints
    xs += [np.float32(v) for v in vals]
    for a, b in zip(vals[:-1], vals[1:]):
        mid = np.float32((a + b) / 2)
        xs += [mid, np.nextafter(mid, np.float32(0)), np.nextafter(mid, np.float32(1e9))]
    xs += [np.float32(0), np.float32(448), np.float32(464), np.float32(463.9), np.float32(1e6)]
    got = quant.encode_e4m3_rne_satfinite(np.asarray(xs, dtype=np.float32))
    for x, c in zip(xs, got):
        fx = Fraction(float(x))
        want = 0x7E if fx >= 448 else _nearest_even(fx, tab)
        # above 448 the format saturates (satfinite); the tie 464 also saturates
        assert int(c) == want, (float(x), hex(int(c)), hex(want))


def _e2m1_table():
    return [(Fraction(v).limit_denominator(2), c) for c, v in enumerate([0, .5, 1, 1.5, 2, 3, 4, 6])]


def test_mxfp4_codes_match_bruteforce_rne():
    rng = np.random.default_rng(11)
    tab = _e2m1_table()
    vals = rng.standard_normal((200, 32)).astype(np.float32) * np.exp(rng.uniform(-6, 6, (200, 1))).astype(np.float32)
    # inject exact ties relative to the group scale: multiples of 0.25 * 2^k
    vals[0] = np.array([0.25, 0.75, 1.25, 1.75, 2.5, 3.5, 5.0, 6.0, 7.0, 7.9, -0.25, -0.75, -1.25, -1.75,
                        -2.5, -3.5, -5.0, 4.0, 0.0, -0.0, 0.1, 0.3, 0.6, 0.9, 1.1, 1.4, 1.6, 2.2, 2.9, 3.2, 4.4, 5.5],
                       dtype=np.float32)
    bits = _bits(vals)
    v = bf16_bits_to_f64(bits)
    codes, scale = quant.quantize_mxfp4(bits)
    for r in range(v.shape[0]):
        amax = max(abs(Fraction(x)) for x in v[r])
        e = 0
        if amax > 0:                                  # floor(log2 amax) by exact comparison
            while Fraction(2) ** (e + 1) <= amax:
                e += 1
            while Fraction(2) ** e > amax:
                e -= 1
            e = max(-127, min(127, e - 2))
        assert int(scale[r, 0]) == e + 127
        X = Fraction(2) ** e
        for i in range(32):
            a = abs(Fraction(float(v[r, i]))) / X
            want = 7 if a >= 6 else _nearest_even(a, tab)
            assert int(codes[r, i]) & 7 == want, (r, i, float(a))
            assert (int(codes[r, i]) >> 3) == int(np.signbit(v[r, i]))


def test_mxfp4_tie_rule_spelled_out():
    # ties go to the even mantissa bit: 0.25->0, 0.75->1, 1.25->1, 1.75->2, 2.5->2, 3.5->4, 5->4
    grp = np.zeros(32, dtype=np.float32)
    grp[:8] = [4.0, 0.25, 0.75, 1.25, 1.75, 2.5, 3.5, 5.0]     # amax 5 -> e = 0, X = 1
    codes, scale = quant.quantize_mxfp4(_bits(grp))
    assert scale.tolist() == [127]
    assert quant.dequantize_mxfp4(codes, scale)[:8].tolist() == [4.0, 0.0, 1.0, 1.0, 2.0, 2.0, 4.0, 4.0]


def test_mxfp4_roundtrip_on_grid_and_zero_group():
    rng = np.random.default_rng(3)
    grid = np.array([0, .5, 1, 1.5, 2, 3, 4, 6])
    for k in (-20, -3, 0, 5, 40):
        g = rng.choice(grid, 32) * rng.choice([-1.0, 1.0], 32) * 2.0 ** k
        g[0] = 6 * 2.0 ** k                                  # pins the scale
        bits = _bits(g)
        dq = quant.dequantize_mxfp4(*quant.quantize_mxfp4(bits))
        assert np.array_equal(dq, bf16_bits_to_f64(bits))
    z = np.zeros(32, dtype=np.float32)
    z[3] = -0.0
    codes, scale = quant.quantize_mxfp4(_bits(z))
    assert scale.tolist() == [127] and (codes & 7).max() == 0 and codes[3] == 8


def test_int4_roundtrip_on_grid_zero_group_and_tiny_group():
    rng = np.random.default_rng(5)
    for code in (0x01, 0x08, 0x30, 0x38, 0x45, 0x7E):
        s = float(quant.e4m3_value(code))
        q = rng.integers(-7, 8, 32)
        q[0] = 7                                             # amax = 7 s -> sf = s exactly
        bits = _bits(q * s)
        qq, cc = quant.quantize_int4_e4m3(bits)
        assert cc.tolist() == [code] and qq.tolist() == q.tolist()
        assert np.array_equal(quant.dequantize_int4_e4m3(qq, cc), bf16_bits_to_f64(bits))
    qq, cc = quant.quantize_int4_e4m3(_bits(np.zeros(32)))
    assert cc.tolist() == [0] and not qq.any()
    tiny = np.zeros(32, dtype=np.float32)
    tiny[5] = 1e-5                                           # amax/7 rounds to E4M3 zero -> bumped to 0x01
    qq, cc = quant.quantize_int4_e4m3(_bits(tiny))
    assert cc.tolist() == [1] and qq[5] == 0                 # 1e-5 / 2^-9 = 0.005 -> 0
    tiny[5] = 0.0015                                         # 0.0015 / 2^-9 = 0.768 -> 1
    qq, cc = quant.quantize_int4_e4m3(_bits(tiny))
    assert cc.tolist() == [1] and qq[5] == 1


def test_int4_q_is_nearest_integer_of_binary32_quotient_and_error_bound():
    rng = np.random.default_rng(13)
    vals = rng.standard_normal((300, 64)).astype(np.float32) * np.exp(rng.uniform(-4, 4, (300, 1))).astype(np.float32)
    bits = _bits(vals)
    v = bf16_bits_to_f64(bits)
    q, code = quant.quantize_int4_e4m3(bits)
    s = quant.e4m3_value(code)                                # [300, 2]
    vg = v.reshape(300, 2, 32)
    qg = q.reshape(300, 2, 32)
    amax = np.abs(vg).max(-1)
    # the scale is the E4M3 value nearest amax/7: within half an E4M3 step
    # (<= 1/16 relative for normals, <= 2^-10 absolute in the subnormal range)
    assert np.all(np.abs(s - amax / 7) <= np.maximum(amax / 7 / 16, 2.0 ** -10) + 1e-9)
    # q is within 1/2 (+ one binary32 ulp of the quotient) of v/s, clamped to [-7, 7]
    t = vg / s[..., None]
    tc = np.clip(t, -7, 7)
    assert np.all(np.abs(qg - tc) <= 0.5 + 1e-6)
    assert qg.min() >= -7 and qg.max() <= 7
    # reconstruction error: half a step, plus the clipped excess when amax/s > 7
    dq = quant.dequantize_int4_e4m3(q, code).reshape(300, 2, 32)
    bound = s[..., None] * (0.5 + 1e-6) + np.maximum(0, np.abs(vg) - 7 * s[..., None])
    assert np.all(np.abs(dq - vg) <= bound)


def test_dequantised_keys_are_bf16_exact_and_sign_of_zero():
    rng = np.random.default_rng(17)
    bits = _bits(rng.standard_normal((64, 4, 64)).astype(np.float32) * 3)
    for fmt in ("mxfp4", "int4_e4m3"):
        dq = quant.quantize_dequantize(fmt, bits)
        f64_to_bf16_bits_exact(dq)                            # raises if not exact
        v = bf16_bits_to_f64(bits)
        assert np.all(np.sign(dq) * np.sign(v) >= 0)          # never flips a sign
    q, code = quant.quantize_int4_e4m3(bits)
    dq = quant.dequantize_int4_e4m3(q, code)
    assert not np.any(np.signbit(dq[dq == 0]))                # INT4 zero is +0.0
    # MXFP4 error bound: X/2 below 2X... worst spacing 2X (between 4X and 6X) -> X; saturation < 2X
    codes, scale = quant.quantize_mxfp4(bits)
    X = np.ldexp(1.0, scale.astype(int) - 127)
    err = np.abs(quant.dequantize_mxfp4(codes, scale) - bf16_bits_to_f64(bits)).reshape(64, 4, 2, 32)
    assert np.all(err < 2 * X[..., None])


def test_fp8_cache_is_nearest_e4m3_value_per_element():
    """f2 (R30): every element goes to the nearest of the 253 finite E4M3 values (ties to the even code),
    saturating at +-448 -- brute force over the value table; every finite code round-trips; half the BF16 footprint."""
    table = quant.e4m3_value(np.arange(0x7F))                            # 0 .. 448, increasing
    assert table[0] == 0.0 and table[-1] == 448.0 and np.all(np.diff(table) > 0)
    rng = np.random.default_rng(8)
    x = np.concatenate([rng.standard_normal(4000) * 3, rng.standard_normal(500) * 300, rng.standard_normal(500) * 1e-3,
                        [0.0, -0.0, 448.0, -448.0, 460.0, 1e9, -1e9, 2.0 ** -9, 2.0 ** -10, 3 * 2.0 ** -10]]).astype(np.float32)
    bits = f32_to_bf16_bits(x)
    v = bf16_bits_to_f64(bits)
    codes = quant.quantize_fp8_e4m3(bits)
    got = quant.dequantize_fp8_e4m3(codes)
    for vi, ci, gi in zip(v, codes, got):
        a = min(abs(vi), 448.0)
        d = np.abs(table - a)
        best = np.flatnonzero(d == d.min())
        want_code = best[0] if len(best) == 1 else [c for c in best if c % 2 == 0][0]
        assert int(ci & 0x7F) == want_code, (vi, ci, want_code)
        assert (ci >> 7) == (1 if np.signbit(vi) else 0)
        assert gi == (-table[want_code] if np.signbit(vi) else table[want_code])
    all_codes = np.concatenate([np.arange(0x7F), 0x80 + np.arange(0x7F)]).astype(np.uint8)
    vals = quant.dequantize_fp8_e4m3(all_codes)
    assert np.array_equal(quant.quantize_fp8_e4m3(f32_to_bf16_bits(vals.astype(np.float32))) & 0x7F, all_codes & 0x7F)
    assert quant.selector_k_bytes("fp8_e4m3", 131072 * 36 * 512) * 2 == quant.selector_k_bytes("bf16", 131072 * 36 * 512)


def test_quantised_query_times_quantised_key_scores_are_scores_of_the_two_images():
    """f2 / R33: "quantised queries x quantised keys" is, by definition, the score of the two dequantised images.  Pins of
    that composition: (a) inputs that already sit on the E4M3 grid pass through the quantiser unchanged, so the quantised
    score equals the plain one; (b) scalar loops over the E4M3 value table on a tiny case; (c) every product of two E4M3
    values has <= 8 significant bits (what makes the FP8 x FP8 tensor-core products exact)."""
    from fractions import Fraction
    from oracle import quant as OQ
    from oracle import selection as OS
    from oracle.bf16 import f64_to_bf16_bits_exact
    rng = np.random.default_rng(9)
    grid = OQ.e4m3_value(np.arange(0x7F))
    q = rng.choice(grid, size=(2, 32)) * rng.choice([-1.0, 1.0], size=(2, 32))
    k = rng.choice(grid, size=(5, 2, 32)) * rng.choice([-1.0, 1.0], size=(5, 2, 32))
    w = np.array([0.7, -0.3])
    qd = OQ.quantize_dequantize("fp8_e4m3", f64_to_bf16_bits_exact(q))
    kd = OQ.quantize_dequantize("fp8_e4m3", f64_to_bf16_bits_exact(k))
    assert np.array_equal(qd, q) and np.array_equal(kd, k)                                 # (a)
    got = OS.token_scores(qd, w, kd)
    for t in range(5):                                                                     # (b)
        want = sum(w[h] * max(0.0, sum(float(q[h, i]) * float(k[t, h, i]) for i in range(32))) for h in range(2))
        assert abs(got[t] - want) < 1e-12
    for a_ in grid[::7]:                                                                   # (c)
        for b_ in grid[::5]:
            pr = Fraction(float(a_)) * Fraction(float(b_))
            if pr:
                num = pr.numerator
                while num % 2 == 0:
                    num //= 2
                assert num < 256
    # off-grid inputs: the quantised score is NOT the plain one (the quantiser does something)
    q2 = rng.standard_normal((2, 32))
    from workloads import f32_to_bf16_bits
    qb = f32_to_bf16_bits(q2.astype(np.float32))
    assert not np.array_equal(OQ.quantize_dequantize("fp8_e4m3", qb), OQ.quantize_dequantize("bf16", qb))


# ---- f2: MXINT8 and INT4 with a BF16 group scale (R38 / R39) ----------------------------------------------

def _floor_log2(x):
    """floor(log2 x) of a positive Fraction by exact comparisons."""
    e = 0
    while Fraction(2) ** (e + 1) <= x:
        e += 1
    while Fraction(2) ** e > x:
        e -= 1
    return e


def test_mxint8_codes_match_bruteforce_rne():
    """Every element goes to the nearest of the 255 values code * 2^(e-6), code in [-127, 127] (ties to the even code,
    saturating), with e = floor(log2 amax) found by exact comparisons -- an independent statement of the format."""
    rng = np.random.default_rng(21)
    vals = rng.standard_normal((120, 32)).astype(np.float32) * np.exp(rng.uniform(-6, 6, (120, 1))).astype(np.float32)
    # ties: with amax = 1.5 (e = 0) the grid step is 1/64; odd multiples of 1/128 are exact ties
    vals[0] = np.array([1.5] + [(2 * i + 1) / 128.0 * (-1) ** i for i in range(31)], dtype=np.float32)
    # clamp: amax = 1.9921875 = 255/128 -> 127.5 -> 128 by RNE -> clamped to 127; -amax likewise to -127
    vals[1] = np.array([255 / 128.0, -255 / 128.0, 1.984375, -1.984375] + [0.0] * 28, dtype=np.float32)
    bits = _bits(vals)
    v = bf16_bits_to_f64(bits)
    codes, scale = quant.quantize_mxint8(bits)
    assert codes.dtype == np.int8 and codes.min() >= -127
    for r in range(v.shape[0]):
        amax = max(abs(Fraction(x)) for x in v[r])
        e = max(-127, min(127, _floor_log2(amax))) if amax > 0 else 0
        assert int(scale[r, 0]) == e + 127
        step = Fraction(2) ** (e - 6)
        for i in range(32):
            x = Fraction(float(v[r, i])) / step
            lo = x.numerator // x.denominator            # floor
            frac = x - lo
            want = lo + (1 if frac > Fraction(1, 2) or (frac == Fraction(1, 2) and lo % 2 == 1) else 0)
            want = max(-127, min(127, want))
            assert int(codes[r, i]) == want, (r, i, float(x))
    assert codes[1, :4].tolist() == [127, -127, 127, -127]
    assert codes[0, 1:5].tolist() == [0, -2, 2, -4]       # 1/128 -> 0.5 -> 0; -3/128 -> -1.5 -> -2; 5/128 -> 2; -7/128 -> -4


def test_mxint8_roundtrip_zero_group_error_bound_and_bf16_exactness():
    rng = np.random.default_rng(22)
    for k in (-30, -3, 0, 7, 60):
        c = rng.integers(-127, 128, 32)
        c[0] = 64 + int(rng.integers(0, 64))                 # largest-magnitude class [1, 2) X: pins the scale
        c = np.clip(c, -c[0], c[0])
        g = c * 2.0 ** (k - 6)
        bits = _bits(g)                                      # <= 7 significant bits: BF16-exact inputs
        cc, ss = quant.quantize_mxint8(bits)
        assert ss.tolist() == [k + 127] and cc.tolist() == c.tolist()
        assert np.array_equal(quant.dequantize_mxint8(cc, ss), bf16_bits_to_f64(bits))
    cc, ss = quant.quantize_mxint8(_bits(np.zeros(32)))
    assert ss.tolist() == [127] and not cc.any()
    bits = _bits(rng.standard_normal((64, 4, 64)).astype(np.float32) * 3)
    v = bf16_bits_to_f64(bits)
    cc, ss = quant.quantize_mxint8(bits)
    dq = quant.dequantize_mxint8(cc, ss)
    f64_to_bf16_bits_exact(dq)                               # raises if a dequantised key is not a BF16 number
    X = np.ldexp(1.0, ss.astype(int) - 127)                  # [64, 4, 2]
    err = np.abs(dq - v).reshape(64, 4, 2, 32)
    assert np.all(err <= X[..., None] / 64)                  # half a step (X / 128), or the clamp's X / 128 .. X / 64
    assert np.all(err[np.abs(cc).reshape(64, 4, 2, 32) < 127] <= np.broadcast_to(X[..., None] / 128, err.shape)[
        np.abs(cc).reshape(64, 4, 2, 32) < 127])
    assert not np.any(np.signbit(dq[dq == 0]))
    # against the (pinned) MXFP4 quantiser: same floor(log2 amax), so the E8M0 bytes differ by E2M1's emax = 2
    _, s4 = quant.quantize_mxfp4(bits)
    assert np.array_equal(ss.astype(int), s4.astype(int) + 2)
    assert quant.selector_k_bytes("mxint8", 256) == 256 + 8


def _bf16_value(bits):
    return Fraction(float(bf16_bits_to_f64(np.array([bits], dtype=np.uint16))[0]))


def test_int4_bf16s_scale_is_the_nearest_bf16_to_amax_over_7_and_q_the_nearest_integer():
    rng = np.random.default_rng(23)
    vals = rng.standard_normal((300, 64)).astype(np.float32) * np.exp(rng.uniform(-5, 5, (300, 1))).astype(np.float32)
    bits = _bits(vals)
    v = bf16_bits_to_f64(bits)
    q, sb = quant.quantize_int4_bf16s(bits)
    assert sb.dtype == np.uint16 and q.min() >= -7 and q.max() <= 7
    vg = v.reshape(300, 2, 32)
    qg = q.reshape(300, 2, 32)
    for r in range(0, 300, 3):
        for gi in range(2):
            amax = max(abs(Fraction(float(x))) for x in vg[r, gi])
            want = amax / 7
            b = int(sb[r, gi])
            s, below, above = _bf16_value(b), _bf16_value(b - 1), _bf16_value(b + 1)
            assert abs(s - want) <= abs(below - want) and abs(s - want) <= abs(above - want), (r, gi)
    s = bf16_bits_to_f64(sb)
    t = vg / s[..., None]
    assert np.all(np.abs(qg - np.clip(t, -7, 7)) <= 0.5 + 1e-6)
    dq = quant.dequantize_int4_bf16s(q, sb).reshape(300, 2, 32)
    bound = s[..., None] * (0.5 + 1e-6) + np.maximum(0, np.abs(vg) - 7 * s[..., None])
    assert np.all(np.abs(dq - vg) <= bound)
    # the 16-bit scale is what the format buys: it sits within 2^-9 relative of amax / 7 (E4M3: 2^-4)
    assert np.all(np.abs(s - np.abs(vg).max(-1) / 7) <= np.abs(vg).max(-1) / 7 * 2.0 ** -8)
    # dequantised values carry up to 11 significant bits: not BF16 numbers in general
    with pytest.raises(ValueError):
        f64_to_bf16_bits_exact(dq)


def test_int4_bf16s_roundtrip_special_groups_and_agreement_with_int4_e4m3_on_e4m3_scales(golden):
    rng = np.random.default_rng(24)
    # scales with <= 5 significant bits keep q * s inside BF16, so the inputs are exact and must round-trip
    for sbits in (0x3F80, 0x3FC0, 0x3E10, 0x4288, 0x0080, 0x7000):
        s = float(bf16_bits_to_f64(np.array([sbits], dtype=np.uint16))[0])
        q = rng.integers(-7, 8, 32)
        q[0] = 7                                             # amax = 7 s -> amax / 7 = s exactly
        bits = _bits(q * s)
        qq, ss = quant.quantize_int4_bf16s(bits)
        assert ss.tolist() == [sbits] and qq.tolist() == q.tolist()
        assert np.array_equal(quant.dequantize_int4_bf16s(qq, ss), bf16_bits_to_f64(bits))
    qq, ss = quant.quantize_int4_bf16s(_bits(np.zeros(32)))
    assert ss.tolist() == [0] and not qq.any()
    tiny = np.zeros(32, dtype=np.float32)
    tiny[5] = 2.0 ** -133                                    # smallest BF16 subnormal: amax / 7 rounds to zero -> bumped
    qq, ss = quant.quantize_int4_bf16s(_bits(tiny))
    assert ss.tolist() == [1] and qq[5] == 1
    # where amax / 7 is itself an E4M3 value, both INT4 formats hold the same scale value, hence the same codes and keys
    # (int4_e4m3 is pinned above by the survey's golden group and the E4M3 brute force)
    for code in (0x08, 0x21, 0x38, 0x45, 0x6B):
        s = float(quant.e4m3_value(code))
        g = rng.standard_normal(32) * 3 * s
        g[0] = 7 * s
        g = np.clip(g, -7 * s, 7 * s)
        bits = _bits(g.astype(np.float32))
        q1, c1 = quant.quantize_int4_e4m3(bits)
        q2, s2 = quant.quantize_int4_bf16s(bits)
        assert c1.tolist() == [code] and float(bf16_bits_to_f64(s2)[0]) == s
        assert np.array_equal(q1, q2)
        assert np.array_equal(quant.dequantize_int4_e4m3(q1, c1), quant.dequantize_int4_bf16s(q2, s2))
    # the paper's own INT4 accounting: 4.5 bit/elt, 1.27 GiB at Qwen3-8B / 128K
    g = golden("footprint.txt")
    n = int(g["tokens"][0][0]) * int(g["layers"][0][0]) * int(g["h_idx"][0][0]) * int(g["d_idx"][0][0])
    assert quant.selector_k_bytes("int4_bf16s", n) / 2.0 ** 30 == pytest.approx(float(g["int4_gib"][0][0]), abs=0.005)
    assert quant.selector_k_bytes("int4_bf16s", n) * 32 == n * 18
