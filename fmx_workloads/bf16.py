"""bf16 bit-pattern helpers (storage format only; round-to-nearest-even, done once)."""
import numpy as np


def f32_to_bf16_bits(x):
    """fp32 array -> uint16 bf16 bit patterns, round-to-nearest-even (NaN not expected)."""
    a = np.ascontiguousarray(x, dtype=np.float32)
    u = a.view(np.uint32)
    rounding = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + rounding) >> np.uint32(16)).astype(np.uint16).reshape(a.shape)


def bf16_bits_to_f32(b):
    b = np.ascontiguousarray(b, dtype=np.uint16)
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32).reshape(b.shape)


def bf16_bits_to_f64(b):
    return bf16_bits_to_f32(b).astype(np.float64)
