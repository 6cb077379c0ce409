"""Property tests of the oracles (tier 4): hypothesis draws shapes, positions, page tables and values;
each property is something the mathematics fixes independently of the implementation (an inverse, an invariant, a bound,
a bijection).  CPU only, a few seconds."""
import numpy as np
from hypothesis import given, settings, strategies as st

from oracle import fit_oracle as F
from oracle import int4_oracle as Q
from oracle import scd_oracle as O

SET = dict(max_examples=30, deadline=None)


@settings(**SET)
@given(st.integers(1, 4), st.sampled_from([4, 8, 32]), st.integers(1, 12), st.integers(0, 100000),
       st.sampled_from([1e4, 5e5, 1e6]), st.sampled_from([O.ROPE_HALF, O.ROPE_INTERLEAVED]), st.integers(0, 2 ** 31 - 1))
def test_rope_is_an_isometry_with_an_inverse(H, d_h, T, p0, theta, style, seed):
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((T, H * d_h))
    pos = p0 + rng.integers(0, 50, T)
    y = O.rope(x, pos, theta, +1, H, d_h, style)
    np.testing.assert_allclose(O.rope(y, pos, theta, -1, H, d_h, style), x, atol=1e-9)
    np.testing.assert_allclose(np.linalg.norm(y.reshape(T, H, d_h), axis=2), np.linalg.norm(x.reshape(T, H, d_h), axis=2), rtol=1e-12)
    # composition: rotating by p then by q is rotating by p + q
    z = O.rope(y, pos + 7, theta, +1, H, d_h, style)
    np.testing.assert_allclose(z, O.rope(x, 2 * pos + 7, theta, +1, H, d_h, style), atol=1e-8)


@settings(**SET)
@given(st.lists(st.integers(1, 70), min_size=1, max_size=6), st.sampled_from([4, 16]), st.integers(0, 2 ** 31 - 1))
def test_slot_mapping_is_injective_and_paging_round_trips(lens, bs, seed):
    rng = np.random.default_rng(seed)
    pages = [(l + bs - 1) // bs for l in lens]
    perm = rng.permutation(sum(pages) + 2)
    table = -np.ones((len(lens), max(pages) + 1), int)
    at = 0
    for i, p in enumerate(pages):
        table[i, :p] = perm[at:at + p]
        at += p
    batch = O.Batch(np.concatenate([[0], np.cumsum(lens)]), table)
    slots = O.slot_mapping(batch, bs)
    assert len(set(slots.tolist())) == sum(lens) and slots.min() >= 0 and slots.max() < perm.size * bs
    assert np.all(slots % bs == np.concatenate([np.arange(l) % bs for l in lens]))
    rows = rng.standard_normal((sum(lens), 6))
    pool = np.full((perm.size, bs, 2, 3), np.nan)
    O.write_paged(pool, slots, rows)
    np.testing.assert_array_equal(O.read_paged(pool, slots), rows)
    assert np.isnan(pool).sum() == (perm.size * bs - sum(lens)) * 6


@settings(**SET)
@given(st.integers(0, 2 ** 31 - 1), st.floats(1e-3, 1e3))
def test_e4m3_quantiser_is_monotone_and_within_half_a_step(seed, scale):
    rng = np.random.default_rng(seed)
    x = np.sort(rng.standard_normal(400) * scale)
    q = O.e4m3_quantize(x)
    v = O.E4M3_VALUES[q]
    assert np.all(np.diff(v) >= 0) and np.all(np.abs(v) <= 448)
    inside = np.abs(x) <= 448
    step = np.maximum(2.0 ** -3 * np.abs(v), 2.0 ** -9)          # spacing of the grid at v (normal / subnormal range)
    assert np.all(np.abs(v - x)[inside] <= step[inside] / 2 * (1 + 1e-12))
    assert np.all(np.abs(v[~inside]) == 448)


@settings(**SET)
@given(st.sampled_from([32, 64, 128]), st.integers(1, 5), st.integers(0, 2 ** 31 - 1), st.floats(1e-2, 1e2), st.floats(-50, 50))
def test_int4_codes_bounds_and_round_trip(group, T, seed, scale, offset):
    rng = np.random.default_rng(seed)
    x = Q.bf16_rne_f32((rng.standard_normal((T, 2 * group)) * scale + offset).astype(np.float32))
    q, packed, s, z = Q.quantize(x, group)
    assert q.max() <= 15 and np.array_equal(Q.unpack(packed), q)
    xg, qg = x.reshape(T, 2, group), q.reshape(T, 2, group).astype(int)
    assert np.all(np.take_along_axis(qg, xg.argmin(axis=2)[..., None], axis=2) == 0)        # the minimum is code 0
    np.testing.assert_array_equal(z, xg.min(axis=2))
    y = Q.dequantize(q, s, z, group)
    bound = 0.5 * np.repeat(s, group, axis=1) * (1 + 2.0 ** -6) + np.abs(y) * 2.0 ** -8
    assert np.all(np.abs(y - x) <= bound + 1e-30)
    # dequantised values lie on the group's 16-level grid (up to the bf16 rounding of the result)
    grid = z[:, :, None] + np.arange(16)[None, None, :] * s[:, :, None]
    d = np.abs(y.reshape(T, 2, group)[..., None] - grid[:, :, None, :]).min(axis=3)
    assert np.all(d <= np.abs(y.reshape(T, 2, group)) * 2.0 ** -8 + 1e-30)


@settings(max_examples=15, deadline=None)
@given(st.integers(8, 40), st.integers(2, 5), st.integers(1, 4), st.integers(0, 2 ** 31 - 1))
def test_fit_truncation_and_sign_freedom(n, w, r, seed):
    rng = np.random.default_rng(seed)
    a, b = rng.standard_normal((n, w)), rng.standard_normal((n, w))
    r = min(r, 2 * w - 1)
    fit = F.fit_reuse(a, b, r, lam_rel=1e-3)
    x = np.concatenate([a, b], axis=1)
    vt = np.concatenate([fit.w_dec_a, fit.w_dec_b], axis=1)
    s_all = np.linalg.svd(x, compute_uv=False)
    np.testing.assert_allclose(np.sum((x - x @ vt.T @ vt) ** 2), np.sum(s_all[r:] ** 2), rtol=1e-9, atol=1e-12)   # Eckart-Young
    flip = rng.choice([-1.0, 1.0], r)
    g = F.ReuseFit(fit.w_enc * flip, fit.w_dec_a * flip[:, None], fit.w_dec_b * flip[:, None], fit.sigma, None, None, fit.lam)
    for u, v in zip(F.invariants(fit), F.invariants(g)):
        np.testing.assert_allclose(u, v, atol=1e-12)
    # ridge shrinks: ||A W_enc|| <= ||Z|| column by column
    z = x @ vt.T
    assert np.all(np.linalg.norm(a @ fit.w_enc, axis=0) <= np.linalg.norm(z, axis=0) * (1 + 1e-12))
