"""CPU oracle for the group-wise INT4 KV codec, the same-box comparison codec of SURVEY §8(f) NEXT-3.

TEST INFRASTRUCTURE ONLY (same rules as scd_oracle.py: imported by tests/, smoke() and bench.py's CPU legs,
shares nothing with the CUDA path).

The paper names the codec only as a baseline: "Quantized KV: transmits 4-bit quantized KV caches (group-wise
INT4) and dequantizes on the consumer" (Table 2 / Table 4 rows `:308`, `:352-359`).  Group size,
symmetric vs asymmetric range and the metadata precision are not stated.  Reading taken here (DESIGN.md §2,
U19): asymmetric min/max quantisation of G consecutive channels of one token row (G in {32, 64, 128}; a group
never straddles a head because G divides head_dim), 16 levels, metadata = one bf16 scale and one bf16 zero
point (the group minimum, which is a stored bf16 value already) per group.

This is an ENCODING: floating point decides an integer.  Both sides therefore take the decision in the
kernel's precision, IEEE fp32 with round-to-nearest-even, operation by operation as written below (numpy
float32 scalars/arrays are IEEE; no fused operations are needed because q * s is exact in fp32: 4 x 8
significant bits).  Codes, metadata and dequantised bf16 values are compared BIT-EXACTLY with the CUDA path.

  lo = min_i x_i ; hi = max_i x_i                        (exact: inputs are bf16)
  s  = bf16_rne( (hi - lo) / 15 )        fp32 subtract, fp32 divide ; s = 1 if that is 0 (constant group)
  q_i = clamp( rint( (x_i - lo) * (1 / s) ), 0, 15 )     fp32 subtract; 1 / s one fp32 divide; fp32 multiply; RNE to integer
  byte j of a row = q_{2j} | q_{2j+1} << 4
  dequantise:  x^_i = bf16_rne( q_i * s + lo )           fp32

Parity pins: tests/test_oracle_int4.py (scalar `Fraction` walk of the same steps, all 16 codes, constant and
two-point groups, hand bytes, error bound |x - x^| <= s/2 + rounding, payload count).
"""
from __future__ import annotations

from typing import Tuple

import numpy as np

LEVELS = 15          # codes 0..15


def bf16_rne_f32(x: np.ndarray) -> np.ndarray:
    """fp32 -> nearest bf16 (ties to even), returned as fp32.  Finite inputs only."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).reshape(x.shape)


def quantize(x: np.ndarray, group: int) -> Tuple[np.ndarray, np.ndarray, np.ndarray, np.ndarray]:
    """x [T, W] (bf16 values held in any float type) -> (q [T, W] uint8 codes 0..15, packed [T, W/2] uint8,
    scale [T, W/G] fp32 holding bf16 values, zero [T, W/G] fp32 holding bf16 values)."""
    x = np.asarray(x, dtype=np.float32)
    T, W = x.shape
    assert W % group == 0 and group % 2 == 0
    xg = x.reshape(T, W // group, group)
    lo = xg.min(axis=2)
    hi = xg.max(axis=2)
    s = bf16_rne_f32((hi - lo).astype(np.float32) / np.float32(LEVELS))
    s = np.where(s == 0, np.float32(1.0), s).astype(np.float32)
    inv = (np.float32(1.0) / s).astype(np.float32)
    t = ((xg - lo[:, :, None]).astype(np.float32) * inv[:, :, None]).astype(np.float32)
    q = np.clip(np.rint(t), 0, LEVELS).astype(np.uint8).reshape(T, W)
    packed = (q[:, 0::2] | (q[:, 1::2] << 4)).astype(np.uint8)
    return q, packed, s, lo.astype(np.float32)


def unpack(packed: np.ndarray) -> np.ndarray:
    """[T, W/2] bytes -> [T, W] codes (low nibble = even channel)."""
    T, Wh = packed.shape
    q = np.empty((T, Wh * 2), dtype=np.uint8)
    q[:, 0::2] = packed & 0xF
    q[:, 1::2] = packed >> 4
    return q


def dequantize(q: np.ndarray, scale: np.ndarray, zero: np.ndarray, group: int) -> np.ndarray:
    """codes [T, W], scale / zero [T, W/G] -> bf16 values [T, W] as fp32."""
    T, W = q.shape
    qg = q.reshape(T, W // group, group).astype(np.float32)
    y = (qg * scale[:, :, None].astype(np.float32)).astype(np.float32) + zero[:, :, None].astype(np.float32)
    return bf16_rne_f32(y.astype(np.float32).reshape(T, W))


def payload_bytes(total_tokens: int, width: int, group: int, n_tensors: int) -> int:
    """|Z| of Eq. 3 for this codec: 4 bits per element + two bf16 per group, per tensor."""
    return n_tensors * total_tokens * (width // 2 + 2 * 2 * (width // group))
