"""Step a0 -- group-32 "microscale" quantisers for the selector K-cache (oracle).

TEST INFRASTRUCTURE (see oracle/__init__.py).

PAPER.md:184 "We quantize the selector's queries and key cache to INT8, INT4,
FP8, and FP4 (group-32 microscale)"; "INT4 / FP4 microscale at
group 32 stores 4.5 bits per element"; PAPER.md:539 (Table 9 caption).  The
paper fixes only "4-bit codes, groups of 32, one shared scale"; the scale
format, rounding and clipping below are DESIGN.md readings R16/R17 (SURVEY.md
section 8(c) step 0').  A group is 32 consecutive elements along d_idx of one
token's one selector head.

All scale arithmetic is defined in IEEE binary32, round-to-nearest-even; numpy
float32 ops implement exactly that.  Codes are returned one per uint8 (values
0..15) -- the oracle has no packed layout; the GPU library's packed layout is
opaque and is compared through its own dequantiser.
"""
import numpy as np

from .bf16 import bf16_bits_to_f32

GROUP = 32

# E2M1 magnitudes by 3-bit code (OCP MX v1.0 FP4): s e e m
E2M1_VALUES = np.array([0.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0], dtype=np.float64)


def selector_k_bytes(fmt, n_elements):
    """Closed-form footprint of n_elements selector-key elements.

    PAPER.md:188: BF16 16 bit/elt; "4.5 bits per element, 0.281x" is the
    16-bit-group-metadata variant; 4 + 8/32 = 4.25 bit/elt is the 8-bit-scale
    variant (E8M0 for MXFP4, E4M3 for BASELINE.json's INT4 format).
    """
    if n_elements % GROUP:
        raise ValueError("n_elements must be a multiple of 32")
    if fmt == "bf16":
        return 2 * n_elements
    if fmt in ("mxfp4", "int4_e4m3"):
        return n_elements // 2 + n_elements // GROUP
    if fmt == "fp8_e4m3":                # f2: one E4M3 byte per element, no scale (the paper's "0.5x" variants)
        return n_elements
    if fmt in ("int4_scale16", "int4_bf16s"):   # the paper's 4.5 bit/elt accounting: 4-bit codes + a 16-bit group scale
        return n_elements // 2 + 2 * (n_elements // GROUP)
    if fmt == "mxint8":                  # f2: INT8 codes + one E8M0 byte per group (8.25 bit/elt; R38)
        return n_elements + n_elements // GROUP
    raise ValueError(fmt)


def _groups(k_bits):
    k_bits = np.asarray(k_bits, dtype=np.uint16)
    if k_bits.shape[-1] % GROUP:
        raise ValueError("last axis must be a multiple of 32")
    v = bf16_bits_to_f32(k_bits)
    return v.reshape(k_bits.shape[:-1] + (k_bits.shape[-1] // GROUP, GROUP))


# --------------------------------------------------------------------------
# MXFP4: E2M1 elements, E8M0 shared scale (R16)
# --------------------------------------------------------------------------

def _round_to_e2m1(a):
    """|value| (float64, exact) -> 3-bit magnitude code, RNE on the E2M1 grid,
    saturating at 6.  Ties go to the code with an even mantissa bit:
    0.25->0, 0.75->1.0, 1.25->1.0, 1.75->2.0, 2.5->2.0, 3.5->4.0, 5.0->4.0."""
    code = np.zeros(a.shape, dtype=np.uint8)
    code += (a > 0.25)       # -> 0.5   (tie 0.25 stays at 0:   code 0 even)
    code += (a >= 0.75)      # -> 1.0   (tie 0.75 goes up:      code 2 even)
    code += (a > 1.25)       # -> 1.5   (tie 1.25 stays at 1.0: code 2 even)
    code += (a >= 1.75)      # -> 2.0   (tie 1.75 goes up:      code 4 even)
    code += (a > 2.5)        # -> 3.0   (tie 2.5 stays at 2.0:  code 4 even)
    code += (a >= 3.5)       # -> 4.0   (tie 3.5 goes up:       code 6 even)
    code += (a > 5.0)        # -> 6.0   (tie 5.0 stays at 4.0:  code 6 even)
    return code


def quantize_mxfp4(k_bits):
    """BF16 bits [..., d] -> (codes uint8 [..., d] in 0..15, scale bytes uint8 [..., d/32]).

    amax = max|v| over the group.  amax == 0: scale byte 127, every code keeps
    the input's sign bit with magnitude 0.  Else e = floor(log2 amax) - 2
    (2 = emax of E2M1), clamped to [-127, 127]; scale byte = e + 127; X = 2^e;
    code = sign | RNE_E2M1(|v| / X), saturating at 6.
    """
    g = _groups(k_bits)
    amax = np.max(np.abs(g), axis=-1).astype(np.float64)
    _, ex = np.frexp(amax)                    # amax = m * 2^ex, m in [0.5, 1)
    e = np.where(amax > 0, ex.astype(np.int64) - 1 - 2, 0)
    e = np.clip(e, -127, 127)
    X = np.ldexp(1.0, e)                      # exact in float64
    r = np.abs(g.astype(np.float64)) / X[..., None]   # exact (power-of-two divide)
    mag = _round_to_e2m1(r)
    sign = np.signbit(g).astype(np.uint8)
    codes = (sign << 3) | mag
    scale = (e + 127).astype(np.uint8)
    return codes.reshape(g.shape[:-2] + (-1,)), scale


def dequantize_mxfp4(codes, scale):
    """-> float64 [..., d]; value = (+-)E2M1(code) * 2^(scale-127), exact in BF16."""
    codes = np.asarray(codes, dtype=np.uint8)
    scale = np.asarray(scale, dtype=np.uint8)
    c = codes.reshape(codes.shape[:-1] + (codes.shape[-1] // GROUP, GROUP))
    mag = E2M1_VALUES[c & 7]
    sgn = np.where((c >> 3) & 1, -1.0, 1.0)
    X = np.ldexp(1.0, scale.astype(np.int64) - 127)
    out = sgn * mag * X[..., None]
    return out.reshape(codes.shape)


# --------------------------------------------------------------------------
# INT4 with one FP8-E4M3 scale per group (BASELINE.json config 3; R16)
# --------------------------------------------------------------------------

def e4m3_value(code):
    """E4M3 (OCP FP8, bias 7, no infinities) code 0..0x7E -> float64."""
    code = np.asarray(code, dtype=np.int64)
    E = (code >> 3) & 0xF
    m = code & 7
    sub = m * 2.0 ** -9
    nrm = np.ldexp(1.0 + m / 8.0, E - 7)
    return np.where(E == 0, sub, nrm)


def encode_e4m3_rne_satfinite(x):
    """non-negative float32 -> E4M3 code, round-to-nearest-even, saturating at
    448 (0x7E), subnormals down to 2^-9, never NaN."""
    x = np.asarray(x, dtype=np.float32).astype(np.float64)
    if np.any(x < 0) or np.any(~np.isfinite(x)):
        raise ValueError("encode_e4m3 takes finite non-negative inputs")
    code = np.zeros(x.shape, dtype=np.int64)
    # subnormal range: multiples of 2^-9 below 2^-6
    sub = x < 2.0 ** -6
    rs = np.rint(np.where(sub, x, 0.0) / 2.0 ** -9).astype(np.int64)   # 0..8, half-to-even; 8 == min normal 0x08
    code = np.where(sub, rs, code)
    # normal range
    _, ex = np.frexp(np.where(sub, 1.0, x))
    ex = ex.astype(np.int64) - 1                      # floor(log2 x)
    q = np.where(sub, 8.0, x) / np.ldexp(1.0, ex - 3)  # in [8, 16), exact
    r = np.rint(q).astype(np.int64)                   # half-to-even
    carry = r == 16
    ex = np.where(carry, ex + 1, ex)
    r = np.where(carry, 8, r)
    ncode = ((ex + 7) << 3) | (r - 8)
    ncode = np.where(ncode > 0x7E, 0x7E, ncode)       # satfinite (covers 0x7F and above)
    code = np.where(sub, code, ncode)
    return code.astype(np.uint8)


def quantize_int4_e4m3(k_bits):
    """BF16 bits [..., d] -> (q int8 [..., d] in -7..7, scale codes uint8 [..., d/32]).

    sf = amax / 7 (binary32); scale code = RNE-satfinite E4M3(sf); a zero code
    with amax > 0 is bumped to 0x01 (smallest subnormal) so the group is never
    silently zeroed; amax == 0 -> code 0, all q = 0.  s = value(code);
    q = clamp(rint(v / s), -7, 7) with the division in binary32 and rint
    half-to-even.
    """
    g = _groups(k_bits)
    amax = np.max(np.abs(g), axis=-1)                         # float32
    sf = amax / np.float32(7.0)                               # binary32 RNE
    code = encode_e4m3_rne_satfinite(sf)
    code = np.where((code == 0) & (amax > 0), np.uint8(1), code).astype(np.uint8)
    s = e4m3_value(code).astype(np.float32)                   # exact
    with np.errstate(divide="ignore", invalid="ignore"):
        t = g / s[..., None]                                  # binary32 RNE
    t = np.where(s[..., None] > 0, t, np.float32(0))
    q = np.clip(np.rint(t), -7, 7).astype(np.int8)
    return q.reshape(g.shape[:-2] + (-1,)), code


def dequantize_int4_e4m3(q, scale_code):
    """-> float64 [..., d]; value = q * E4M3(scale), <= 8 significant bits so exact in BF16."""
    q = np.asarray(q, dtype=np.int8)
    qq = q.reshape(q.shape[:-1] + (q.shape[-1] // GROUP, GROUP)).astype(np.float64)
    s = e4m3_value(np.asarray(scale_code, dtype=np.uint8))
    out = qq * s[..., None]
    out = out + 0.0                                           # q == 0 -> +0.0
    return out.reshape(q.shape)


# --------------------------------------------------------------------------
# FP8-E4M3 per element (R30): the paper lists FP8 among the selector-cache precisions
# (Table 9) at half the BF16 footprint and says nothing else.
# --------------------------------------------------------------------------

def quantize_fp8_e4m3(k_bits):
    """BF16 bits [..., d] -> uint8 codes [..., d]: sign bit | RNE-satfinite E4M3 of |v| (no scale, saturating at 448,
    subnormals down to 2^-9, a zero keeps its sign)."""
    k_bits = np.asarray(k_bits, dtype=np.uint16)
    v = bf16_bits_to_f32(k_bits)
    sign = (k_bits >> np.uint16(15)).astype(np.uint8)
    return (sign << np.uint8(7)) | encode_e4m3_rne_satfinite(np.abs(v))


def dequantize_fp8_e4m3(codes):
    """-> float64 [..., d]; 4 significant bits, so exact in BF16."""
    codes = np.asarray(codes, dtype=np.uint8)
    mag = e4m3_value(codes & np.uint8(0x7F))
    return np.where(codes >> np.uint8(7), -mag, mag)


# --------------------------------------------------------------------------
# MXINT8 (R38): PAPER.md:184 lists INT8 among the "group-32 microscale" precisions and fixes
# nothing else.  Reading: the OCP MX v1.0 INT8 element -- a two's-complement byte read as code * 2^-6, so that the
# group's largest element lands in [1, 2) -- under one E8M0 shared scale per group of 32.
# --------------------------------------------------------------------------

def quantize_mxint8(k_bits):
    """BF16 bits [..., d] -> (codes int8 [..., d] in -127..127, scale bytes uint8 [..., d/32]).

    amax = max|v| over the group.  amax == 0: scale byte 127, codes 0.  Else e = floor(log2 amax) (0 = emax of the
    element format), clamped to [-127, 127]; scale byte = e + 127; X = 2^e; code = clamp(RNE(v / X * 64), -127, 127)
    (symmetric clamp: -128 is never produced).
    """
    g = _groups(k_bits)
    amax = np.max(np.abs(g), axis=-1).astype(np.float64)
    _, ex = np.frexp(amax)                    # amax = m * 2^ex, m in [0.5, 1)
    e = np.where(amax > 0, ex.astype(np.int64) - 1, 0)
    e = np.clip(e, -127, 127)
    X = np.ldexp(1.0, e)                      # exact in float64
    r = g.astype(np.float64) / X[..., None] * 64.0        # exact (power-of-two scalings)
    codes = np.clip(np.rint(r), -127, 127).astype(np.int8)   # rint: half-to-even
    scale = (e + 127).astype(np.uint8)
    return codes.reshape(g.shape[:-2] + (-1,)), scale


def dequantize_mxint8(codes, scale):
    """-> float64 [..., d]; value = code * 2^(scale - 127 - 6): <= 7 significant bits, exact in BF16; code 0 -> +0.0."""
    codes = np.asarray(codes, dtype=np.int8)
    scale = np.asarray(scale, dtype=np.uint8)
    c = codes.reshape(codes.shape[:-1] + (codes.shape[-1] // GROUP, GROUP)).astype(np.float64)
    X = np.ldexp(1.0, scale.astype(np.int64) - 127 - 6)
    out = c * X[..., None] + 0.0
    return out.reshape(codes.shape)


# --------------------------------------------------------------------------
# INT4 with a 16-bit group scale (R39): the paper's own INT4 accounting, "4.5 bits per element",
# 1.27 GiB against MXFP4's 1.20 GiB at Qwen3-8B / 128K.  The paper does not say which 16-bit number the
# scale is.  Reading: a BF16 scale (the cache's own number format); everything else as in int4_e4m3.
# --------------------------------------------------------------------------

def _f32_to_bf16_bits_rne(x):
    """finite binary32 -> BF16 bits, round-to-nearest-even on the 16 dropped bits (integer arithmetic on the pattern)."""
    u = np.asarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    lsb = (u >> np.uint64(16)) & np.uint64(1)
    return ((u + np.uint64(0x7FFF) + lsb) >> np.uint64(16)).astype(np.uint16)


def quantize_int4_bf16s(k_bits):
    """BF16 bits [..., d] -> (q int8 [..., d] in -7..7, scale BF16 bits uint16 [..., d/32]).

    sf = amax / 7 (binary32); scale = RNE-to-BF16(sf); a zero scale with amax > 0 is bumped to the smallest BF16
    subnormal (bits 0x0001); amax == 0 -> scale bits 0, all q = 0.  s = value(scale);
    q = clamp(rint(v / s), -7, 7) with the division in binary32 and rint half-to-even.
    """
    g = _groups(k_bits)
    amax = np.max(np.abs(g), axis=-1)                         # float32
    sf = amax / np.float32(7.0)                               # binary32 RNE
    sb = _f32_to_bf16_bits_rne(sf)
    sb = np.where((sb == 0) & (amax > 0), np.uint16(1), sb).astype(np.uint16)
    s = bf16_bits_to_f32(sb)                                  # exact
    with np.errstate(divide="ignore", invalid="ignore"):
        t = g / s[..., None]                                  # binary32 RNE
    t = np.where(s[..., None] > 0, t, np.float32(0))
    q = np.clip(np.rint(t), -7, 7).astype(np.int8)
    return q.reshape(g.shape[:-2] + (-1,)), sb


def dequantize_int4_bf16s(q, scale_bits):
    """-> float64 [..., d]; value = q * BF16(scale), exact here.  Up to 11 significant bits: NOT a BF16 number in general
    (the scoring kernels use the exact product; a BF16 view of it is a rounding)."""
    q = np.asarray(q, dtype=np.int8)
    qq = q.reshape(q.shape[:-1] + (q.shape[-1] // GROUP, GROUP)).astype(np.float64)
    s = bf16_bits_to_f32(np.asarray(scale_bits, dtype=np.uint16)).astype(np.float64)
    out = qq * s[..., None] + 0.0
    return out.reshape(q.shape)


def quantize_dequantize(fmt, k_bits):
    """Convenience: BF16 bits -> float64 dequantised keys for a format name."""
    if fmt == "bf16":
        from .bf16 import bf16_bits_to_f64
        return bf16_bits_to_f64(k_bits)
    if fmt == "mxfp4":
        return dequantize_mxfp4(*quantize_mxfp4(k_bits))
    if fmt == "int4_e4m3":
        return dequantize_int4_e4m3(*quantize_int4_e4m3(k_bits))
    if fmt == "fp8_e4m3":
        return dequantize_fp8_e4m3(quantize_fp8_e4m3(k_bits))
    if fmt == "mxint8":
        return dequantize_mxint8(*quantize_mxint8(k_bits))
    if fmt == "int4_bf16s":
        return dequantize_int4_bf16s(*quantize_int4_bf16s(k_bits))
    raise ValueError(fmt)
