"""float32 <-> BF16 bit patterns for the input generators (data format only)."""
import numpy as np


def f32_to_bf16_bits(x):
    """float32 array -> uint16 BF16 bit patterns, round-to-nearest-even
    (finite inputs; the generators never produce NaN/Inf)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = (u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)
    return r.astype(np.uint16)


def bf16_bits_to_f32(b):
    """uint16 BF16 bit patterns -> float32 array (exact)."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)
