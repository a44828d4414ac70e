"""BF16 bit patterns -> exact float64 values (oracle side; test infrastructure).

BF16 is the upper 16 bits of an IEEE binary32, so every BF16 value is exactly
representable in float64.  The oracle receives inputs as uint16 bit patterns
(the same bits the GPU path reads) and decodes them with no rounding.
"""
import numpy as np


def bf16_bits_to_f64(bits):
    """uint16 array of BF16 bit patterns -> float64 array of the exact values."""
    b = np.ascontiguousarray(bits, dtype=np.uint16)
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def bf16_bits_to_f32(bits):
    """uint16 array of BF16 bit patterns -> float32 array (exact)."""
    b = np.ascontiguousarray(bits, dtype=np.uint16)
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32)


def f64_to_bf16_bits_exact(x):
    """float64 values that are exactly BF16-representable -> uint16 bits.

    Raises if any value would need rounding: the oracle never rounds to BF16
    on its own (dequantised selector keys are exact in BF16 by construction,
    DESIGN.md R16), so a failure here is a bug in the caller.
    """
    x = np.asarray(x, dtype=np.float64)
    f = x.astype(np.float32)
    if not np.array_equal(f.astype(np.float64), x):
        raise ValueError("value not representable in binary32")
    u = f.view(np.uint32)
    if np.any(u & np.uint32(0xFFFF)):
        raise ValueError("value not representable in BF16")
    return (u >> np.uint32(16)).astype(np.uint16)
