"""Seeded feature tensors and storage-dtype rounding (no method arithmetic here).

bf16 tensors are carried through numpy as uint16 bit patterns (numpy has no bfloat16);
``bf16_bits_to_f32`` up-casts them exactly, which is what the fp64 oracle reads
("inputs are the stored fp32/bf16 values up-cast exactly").
"""
from __future__ import annotations

import numpy as np


def rng_for(cfg: int, stream: int, seed: int = 0) -> np.random.Generator:
    """numpy PCG64 keyed by (seed, cfg, stream).  Streams: 0 graph, 1 relabel,
    2 hub planting, 3 long-range edges, 10..13 Q/K/V/dO, 20..24 X/W_s/W_t/a/dO."""
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([seed, cfg, stream])))


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16, returned as uint16 bit patterns."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    bias = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + bias) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    """Exact bf16 (uint16 bits) -> fp32."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def normal_tensor(rng: np.random.Generator, shape, std: float = 1.0, chunk: int = 1 << 24) -> np.ndarray:
    """N(0, std^2) fp32 tensor, drawn in fixed-size chunks so the stream does not depend
    on available memory."""
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.float32)
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        out[s:e] = rng.standard_normal(e - s, dtype=np.float32)
    if std != 1.0:
        out *= np.float32(std)
    return out.reshape(shape)


def store(x32: np.ndarray, dtype: str, keep_f32: bool = True):
    """Round an fp32 tensor to the storage dtype.

    Returns (stored, as_f32): ``stored`` is what is handed to the GPU (fp32 array, or
    uint16 bf16 bit patterns); ``as_f32`` is the same values up-cast exactly to fp32 (what
    the oracle reads).  For fp32 both are the same array.
    """
    if dtype == "f32":
        x32 = np.ascontiguousarray(x32, dtype=np.float32)
        return x32, x32
    if dtype == "bf16":
        bits = f32_to_bf16_bits(x32)
        return bits, (bf16_bits_to_f32(bits) if keep_f32 else None)
    raise ValueError(f"unknown dtype {dtype!r}")
