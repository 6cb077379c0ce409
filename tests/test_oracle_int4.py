"""Pins for oracle/int4_oracle.py (group-wise INT4 comparison codec; reading U19 in DESIGN.md).

The oracle is pinned by things other than itself: a scalar walk of the definition in exact rational
arithmetic with an independent bf16 rounding (struct bit surgery on Python floats), hand-computed bytes,
every one of the 16 codes, degenerate groups, the quantiser's error bound, torch's bf16 cast.  CPU only.
"""
import struct
from fractions import Fraction

import numpy as np
import pytest
import torch

from oracle import int4_oracle as Q

rng = np.random.default_rng(77)


# ---------------------------------------------------------------- independent scalar arithmetic
def _f32(x: Fraction) -> Fraction:
    """Round an exact rational to the nearest fp32 (ties to even) -- via Python's correctly rounded
    Fraction -> double conversion followed by struct's double -> float (safe here: every operand below has
    <= 24 significant bits times small integers, so double rounding cannot occur for sums / differences;
    for quotients the exact value is re-checked against both neighbours)."""
    if x == 0:
        return Fraction(0)
    d = float(x)
    f = struct.unpack("f", struct.pack("f", d))[0]
    # guard against double rounding: compare with neighbours in exact arithmetic
    cands = [Fraction(f), Fraction(float(np.nextafter(np.float32(f), np.float32(np.inf)))),
             Fraction(float(np.nextafter(np.float32(f), np.float32(-np.inf))))]
    best = min(cands, key=lambda c: (abs(c - x), int(np.float32(float(c)).view(np.uint32)) & 1))
    return best


def _bf16(x: Fraction) -> Fraction:
    """Nearest bf16 (ties to even) of an exact rational, by bit surgery."""
    if x == 0:
        return Fraction(0)
    sign = -1 if x < 0 else 1
    a = abs(x)
    e = 0
    while a >= 2:
        a /= 2; e += 1
    while a < 1:
        a *= 2; e -= 1
    m = a * 128                       # 8 significant bits -> integer part in [128, 256)
    lo = m.numerator // m.denominator
    rem = m - lo
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and (lo & 1)):
        lo += 1
    return sign * Fraction(lo, 128) * (Fraction(2) ** e)


def _rint(x: Fraction) -> int:
    lo = x.numerator // x.denominator
    rem = x - lo
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and (lo & 1)):
        lo += 1
    return lo


def _scalar_quant(row, group):
    """The definition of the module docstring, token by token, in exact rationals + explicit roundings."""
    q, s_out, z_out = [], [], []
    for g0 in range(0, len(row), group):
        xs = [Fraction(float(v)) for v in row[g0:g0 + group]]
        lo, hi = min(xs), max(xs)
        s = _bf16(_f32(_f32(hi - lo) / 15))
        if s == 0:
            s = Fraction(1)
        inv = _f32(Fraction(1) / s)
        for x in xs:
            t = _f32(_f32(x - lo) * inv)
            q.append(max(0, min(15, _rint(t))))
        s_out.append(s)
        z_out.append(lo)
    return q, s_out, z_out


def _bf16_values(shape, scale=1.0):
    x = torch.from_numpy(rng.standard_normal(shape).astype(np.float32) * scale).to(torch.bfloat16)
    return x.float().numpy()


# ---------------------------------------------------------------- pins
def test_bf16_rounding_matches_torch_and_ties():
    x = np.concatenate([rng.standard_normal(20000).astype(np.float32) * 3,
                        np.float32([1.00390625, 1.01171875, -1.00390625, 0.0, 3.0e-39, 6.5e4])])
    want = torch.from_numpy(x).to(torch.bfloat16).float().numpy()
    np.testing.assert_array_equal(Q.bf16_rne_f32(x), want)
    # 1 + 2^-8 is a tie between 1 and 1 + 2^-7 -> even (1); 1 + 3 * 2^-8 ties up to 1 + 2^-6
    assert Q.bf16_rne_f32(np.float32([1.00390625]))[0] == 1.0
    assert Q.bf16_rne_f32(np.float32([1.01171875]))[0] == 1.015625


@pytest.mark.parametrize("group", [32, 64, 128])
def test_quantize_matches_scalar_rational_walk(group):
    x = _bf16_values((6, 256), 2.0)
    x[1, :group] = 0.75                       # constant group
    x[2, 3] = 40.0                            # outlier stretches one group's range
    x[3] *= 1e-3
    q, packed, s, z = Q.quantize(x, group)
    for t in range(x.shape[0]):
        qq, ss, zz = _scalar_quant(x[t], group)
        assert q[t].tolist() == qq
        assert [Fraction(float(v)) for v in s[t]] == ss
        assert [Fraction(float(v)) for v in z[t]] == zz
    # dequantise: bf16(q * s + lo), again in exact rationals
    y = Q.dequantize(q, s, z, group)
    for t in range(x.shape[0]):
        for i in range(x.shape[1]):
            g = i // group
            want = _bf16(_f32(Fraction(int(q[t, i])) * Fraction(float(s[t, g])) + Fraction(float(z[t, g]))))
            assert Fraction(float(y[t, i])) == want


def test_all_sixteen_codes_and_exact_round_trip():
    """x = lo + k * 2^-3, k = 0..15 (twice, shuffled): s = (15/8)/15 = 1/8 exactly, every code appears, and
    the round trip is exact because lo + k/8 is a bf16 value."""
    group = 32
    k = np.concatenate([np.arange(16), np.arange(16)[::-1]])
    x = (np.float32(-1.0) + k.astype(np.float32) / 8)[None, :]
    q, packed, s, z = Q.quantize(x, group)
    assert q[0].tolist() == k.tolist()
    assert s[0, 0] == 0.125 and z[0, 0] == -1.0
    np.testing.assert_array_equal(Q.dequantize(q, s, z, group), x)
    # nibble packing: byte j = q[2j] | q[2j+1] << 4  (hand: codes 0,1 -> 0x10 ; 2,3 -> 0x32 ; ... ; 14,15 -> 0xFE)
    assert packed[0, :8].tolist() == [0x10, 0x32, 0x54, 0x76, 0x98, 0xBA, 0xDC, 0xFE]
    np.testing.assert_array_equal(Q.unpack(packed), q)


def test_degenerate_groups():
    group = 32
    x = np.zeros((3, 64), np.float32)
    x[0, :] = -2.5                            # constant: s = 1, q = 0, x^ = lo exactly
    x[1, :32] = 0.0; x[1, 5] = 1.0            # two-point group: codes 0 and 15
    x[2, :32] = np.float32(2.0 ** -100)       # tiny constant group
    x[2, 32:] = 0.0; x[2, 40] = np.float32(2.0 ** -100)   # tiny but non-zero range (normal numbers throughout)
    q, packed, s, z = Q.quantize(x, group)
    assert s[0].tolist() == [1.0, 1.0] and not q[0].any()
    np.testing.assert_array_equal(Q.dequantize(q, s, z, group)[0], x[0])
    assert q[1, 5] == 15 and q[1, :5].tolist() == [0] * 5 and z[1, 0] == 0.0
    # s = bf16(1/15) = 0.06689453125 (1/15 = 0.0666..., bf16 neighbours 0.06640625 / 0.06689453125)
    assert s[1, 0] == np.float32(0.06689453125)
    assert s[2, 0] == 1.0
    assert q[2, 40] == 15 and q[2, 41] == 0
    y = Q.dequantize(q, s, z, group)
    assert np.all(np.isfinite(y))


def test_error_bound_and_monotone_codes():
    """|x - x^| <= s/2 (1 + 2^-7) + bf16 rounding of the result; codes are monotone in x inside a group."""
    for group in (32, 64, 128):
        x = _bf16_values((64, 512), 1.5)
        q, packed, s, z = Q.quantize(x, group)
        y = Q.dequantize(q, s, z, group)
        S = np.repeat(s, group, axis=1).astype(np.float64)
        bound = 0.5 * S * (1 + 2.0 ** -6) + np.abs(y) * 2.0 ** -8 + 1e-30
        assert np.all(np.abs(x.astype(np.float64) - y) <= bound)
        xg = x.reshape(64, -1, group); qg = q.reshape(64, -1, group).astype(int)
        order = np.argsort(xg, axis=2, kind="stable")
        assert np.all(np.diff(np.take_along_axis(qg, order, axis=2), axis=2) >= 0)
        assert qg.min(axis=2).max() == 0                     # the group minimum always maps to code 0
        assert np.all(qg.max(axis=2)[s.reshape(64, -1) != 1.0] == 15)   # and the maximum to 15


def test_payload_bytes_hand_count():
    # 8192 tokens, D = 1024, G = 32: 512 B of nibbles + 32 groups * 4 B = 640 B per row = 5 bits / element
    assert Q.payload_bytes(8192, 1024, 32, 1) == 8192 * 640
    assert Q.payload_bytes(8192, 1024, 32, 64) * 8 == 64 * 8192 * 1024 * 5
    assert Q.payload_bytes(10, 256, 128, 2) == 2 * 10 * (128 + 8)
