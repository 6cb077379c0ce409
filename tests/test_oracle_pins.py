"""Pins for oracle/scd_oracle.py: every function is checked against something other than
itself -- closed forms, invariants, independent library routines (numpy SVD, torch
bf16 / float8 casts, cmath), exact rational arithmetic, brute force.  CPU only.

Each pin is chosen so that a plausible mistake (dropped term, wrong sign or index,
transposed operand) fails at least one test; see DESIGN.md "Oracle pins".
"""
import cmath
import json
import math
import os
from fractions import Fraction

import numpy as np
import pytest
import torch

from oracle import scd_oracle as O

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "hand_examples.json")))
rng = np.random.default_rng(1234)


# ------------------------------------------------------------------ RoPE (Eq. 5, :152)
def _rope_complex(x, p, theta, d_h, style):
    """Independent formulation: each pair is a complex number multiplied by e^{i phi}."""
    out = [0.0] * d_h
    for j in range(d_h // 2):
        a, b = (j, j + d_h // 2) if style == O.ROPE_HALF else (2 * j, 2 * j + 1)
        z = complex(x[a], x[b]) * cmath.exp(1j * p * theta ** (-2.0 * j / d_h))
        out[a], out[b] = z.real, z.imag
    return out


@pytest.mark.parametrize("style,key", [(O.ROPE_HALF, "half"), (O.ROPE_INTERLEAVED, "interleaved")])
def test_rope_worked_example(style, key):
    g = GOLD["rope"]
    x = np.array([g["x"]], dtype=np.float64)
    y = O.rope(x, np.array([g["pos"]]), g["theta"], +1, 1, g["head_dim"], style)
    ref = _rope_complex(g["x"], g["pos"], g["theta"], g["head_dim"], style)
    np.testing.assert_allclose(y[0], ref, atol=1e-14)
    np.testing.assert_allclose(y[0], g[key], atol=5e-7)          # SURVEY 8(c) printed digits
    back = O.rope(y, np.array([g["pos"]]), g["theta"], -1, 1, g["head_dim"], style)
    np.testing.assert_allclose(back[0], g["x"], atol=1e-14)


@pytest.mark.parametrize("style", [O.ROPE_HALF, O.ROPE_INTERLEAVED])
def test_rope_invariants(style):
    H, d_h, T = 3, 16, 40
    x = rng.standard_normal((T, H * d_h))
    pos = rng.integers(0, 5000, T)
    y = O.rope(x, pos, 5e5, +1, H, d_h, style)
    # inverse
    np.testing.assert_allclose(O.rope(y, pos, 5e5, -1, H, d_h, style), x, atol=1e-12)
    # per-head norms preserved
    np.testing.assert_allclose(np.linalg.norm(y.reshape(T, H, d_h), axis=2),
                               np.linalg.norm(x.reshape(T, H, d_h), axis=2), rtol=1e-13)
    # position 0 is the identity
    np.testing.assert_array_equal(O.rope(x, np.zeros(T, int), 5e5, +1, H, d_h, style), x)
    # <RoPE(q, m), RoPE(k, n)> depends only on m - n
    q, k = x[:1], x[1:2]
    def dot(m, n):
        return float((O.rope(q, [m], 1e4, +1, H, d_h, style) @ O.rope(k, [n], 1e4, +1, H, d_h, style).T)[0, 0])
    assert abs(dot(17, 5) - dot(112, 100)) < 1e-10
    assert abs(dot(17, 5) - dot(5, 17)) > 1e-6            # and really does depend on it
    # every (row, head, pair) against the complex formulation (catches index slips)
    for t in (0, 7, T - 1):
        for h in range(H):
            ref = _rope_complex(list(x[t, h * d_h:(h + 1) * d_h]), int(pos[t]), 5e5, d_h, style)
            np.testing.assert_allclose(y[t, h * d_h:(h + 1) * d_h], ref, atol=1e-9)


def test_rope_interleaved_is_half_after_permutation():
    H, d_h, T = 2, 8, 5
    x = rng.standard_normal((T, H * d_h))
    pos = np.arange(T) + 3
    perm = np.concatenate([np.arange(0, d_h, 2), np.arange(1, d_h, 2)])   # even then odd
    xh = x.reshape(T, H, d_h)[:, :, perm].reshape(T, H * d_h)
    yh = O.rope(xh, pos, 1e4, +1, H, d_h, O.ROPE_HALF).reshape(T, H, d_h)
    yi = O.rope(x, pos, 1e4, +1, H, d_h, O.ROPE_INTERLEAVED).reshape(T, H, d_h)
    np.testing.assert_allclose(yi[:, :, perm], yh, atol=1e-14)


# ------------------------------------------------------------------ packing (U11, U15)
def test_bf16_rounding_matches_torch():
    x = np.concatenate([rng.standard_normal(20000) * 10.0 ** rng.integers(-6, 6, 20000),
                        [0.0, 1.0, -1.0, 1.00390625, 1.01171875, 3.0e-5, 65280.0]])
    ref = torch.from_numpy(x).to(torch.float32)
    # only values exactly representable in fp32 make the two-step torch cast a fair referee
    x32 = ref.double().numpy()
    got = O.round_to_bf16(x32)
    want = ref.to(torch.bfloat16).double().numpy()
    np.testing.assert_array_equal(got, want)
    # explicit ties: 1 + 2^-8 is halfway between 1 and 1 + 2^-7 -> even (1.0); 1 + 3*2^-8 -> 1 + 2^-6
    assert O.round_to_bf16(np.array([1 + 2.0 ** -8]))[0] == 1.0
    assert O.round_to_bf16(np.array([1 + 3 * 2.0 ** -8]))[0] == 1 + 2.0 ** -6


def test_e4m3_table_matches_torch_float8():
    b = torch.arange(256, dtype=torch.uint8)
    ref = b.view(torch.float8_e4m3fn).to(torch.float64).numpy()
    np.testing.assert_array_equal(np.isnan(ref), np.isnan(O.E4M3_VALUES))
    ok = ~np.isnan(ref)
    np.testing.assert_array_equal(ref[ok], O.E4M3_VALUES[ok])
    assert np.nanmax(O.E4M3_VALUES) == 448.0


def test_e4m3_quantizer_exhaustive():
    vals = O.E4M3_VALUES
    finite = [b for b in range(256) if not np.isnan(vals[b])]
    assert len(finite) == 254
    # every finite code decodes -> encodes to itself (0x80 = -0 keeps its sign bit)
    q = O.e4m3_quantize(vals[finite])
    np.testing.assert_array_equal(q, np.array(finite, dtype=np.uint8))
    # every midpoint between adjacent magnitudes rounds to the even code; just off rounds to nearest
    for c in range(0x7E):
        lo, hi = vals[c], vals[c + 1]
        mid = (lo + hi) / 2
        even = c if c % 2 == 0 else c + 1
        assert O.e4m3_quantize(np.array([mid]))[0] == even
        assert O.e4m3_quantize(np.array([-mid]))[0] == even | 0x80
        eps = (hi - lo) * 1e-6
        assert O.e4m3_quantize(np.array([mid - eps]))[0] == c
        assert O.e4m3_quantize(np.array([mid + eps]))[0] == c + 1
    # saturation
    np.testing.assert_array_equal(O.e4m3_quantize(np.array([448.0, 449.0, 480.0, 1e9, -1e9])),
                                  [0x7E, 0x7E, 0x7E, 0x7E, 0xFE])
    for x, want in GOLD["e4m3_ties"]:
        assert vals[O.e4m3_quantize(np.array([float(x)]))[0]] == want


def test_e4m3_rowscale_worked_example_and_bounds():
    g = GOLD["e4m3_rowscale"]
    z = np.array([g["z"]])
    q, s = O.pack_codes(z, O.E4M3_ROWSCALE)
    assert s.dtype == np.float32 and abs(float(s[0]) - g["scale"]) < 1e-9
    np.testing.assert_array_equal(q[0], g["bytes"])
    np.testing.assert_array_equal(O.E4M3_VALUES[q[0]], g["q"])
    np.testing.assert_allclose(O.unpack_codes(q, s, O.E4M3_ROWSCALE)[0], g["dequant"], atol=5e-7)
    # random rows: amax element maps to +-448, relative error <= 2^-4 in the normal range,
    # all-zero row gets scale 1 and zero codes
    z = rng.standard_normal((64, 96)) * 10.0 ** rng.uniform(-3, 3, (64, 1))
    z[5] = 0.0
    q, s = O.pack_codes(z, O.E4M3_ROWSCALE)
    assert s[5] == 1.0 and not q[5].any()
    dq = O.unpack_codes(q, s, O.E4M3_ROWSCALE)
    for i in range(64):
        if i == 5:
            continue
        j = np.argmax(np.abs(z[i]))
        assert abs(O.E4M3_VALUES[q[i, j]]) == 448.0
        normal = np.abs(z[i] / s[i]) >= 2.0 ** -6
        assert np.all(np.abs(dq[i] - z[i])[normal] <= 2.0 ** -4 * np.abs(z[i])[normal] * (1 + 1e-6))


def test_pack_f32_and_bf16():
    z = rng.standard_normal((7, 5))
    q, s = O.pack_codes(z, O.F32)
    assert s is None and q.dtype == np.float32
    np.testing.assert_array_equal(q, z.astype(np.float32))
    q, s = O.pack_codes(z, O.BF16)
    z32 = z.astype(np.float32).astype(np.float64)               # fp32-representable -> torch is a fair referee
    np.testing.assert_array_equal(O.pack_codes(z32, O.BF16)[0],
                                  torch.from_numpy(z32).float().to(torch.bfloat16).double().numpy())
    assert np.max(np.abs(q - z) / np.abs(z)) <= 2.0 ** -8


# ------------------------------------------------------------------ encode / decode (Eq. 8-9)
def _model(**kw):
    base = dict(n_layers=1, d_model=8, n_kv_heads=1, head_dim=4, code_dtype=O.F32,
                k_is_roped=False, rope_on_reuse_k=False)
    base.update(kw)
    return O.Model(**base)


def test_encode_decode_worked_example_exact():
    g = GOLD["encode_decode"]
    B = np.array(g["B"]); mu = np.array(g["mu"]); X = np.array(g["X"], dtype=float)
    # exact rational re-derivation, independent of numpy matmul
    Bf = [[Fraction(v).limit_denominator() for v in row] for row in g["B"]]
    muf = [Fraction(v).limit_denominator() for v in g["mu"]]
    Zf = [[sum((Fraction(x) - m) * b for x, m, b in zip(row, muf, brow)) for brow in Bf] for row in g["X"]]
    Xf = [[sum(z * Bf[i][c] for i, z in enumerate(zr)) + muf[c] for c in range(4)] for zr in Zf]
    assert [[float(v) for v in r] for r in Zf] == g["Z"]
    assert [[float(v) for v in r] for r in Xf] == g["Xhat"]
    m = _model()
    lay = O.Layer(O.REUSE, enc_k=B.T, enc_v=B.T, dec_k=B, dec_v=B, mean_src_k=mu, mean_src_v=mu,
                  mean_dst_k=mu, mean_dst_v=mu)
    zk = O.encode_k(m, lay, X, np.zeros(2, int))
    zv = O.encode_v(m, lay, X)
    np.testing.assert_array_equal(zk, g["Z"]); np.testing.assert_array_equal(zv, g["Z"])
    k, v = O.reuse_decode_layer(m, lay, zk, zv, np.zeros(2, int))
    np.testing.assert_array_equal(k, g["Xhat"]); np.testing.assert_array_equal(v, g["Xhat"])
    np.testing.assert_array_equal(((X - k) ** 2).sum(1), g["sq_residual"])


def _orthobasis(width, r):
    q, _ = np.linalg.qr(rng.standard_normal((width, width)))
    return q[:, :r].T.copy()                                 # [r, width], orthonormal rows


def test_full_rank_round_trip_with_rope_returns_roped_k():
    H, d_h, T = 2, 8, 33
    D = H * d_h
    m = O.Model(n_layers=1, d_model=32, n_kv_heads=H, head_dim=d_h, rope_theta_producer=5e5,
                rope_theta_consumer=5e5, k_is_roped=True, rope_on_reuse_k=True)
    B = _orthobasis(D, D)
    mu_k, mu_v = rng.standard_normal(D), rng.standard_normal(D)
    lay = O.Layer(O.REUSE, enc_k=B.T, enc_v=B.T, dec_k=B, dec_v=B, mean_src_k=mu_k, mean_dst_k=mu_k,
                  mean_src_v=mu_v, mean_dst_v=mu_v)
    K, V = rng.standard_normal((T, D)), rng.standard_normal((T, D))
    pos = rng.integers(0, 9000, T)
    k, v = O.reuse_decode_layer(m, lay, O.encode_k(m, lay, K, pos), O.encode_v(m, lay, V), pos)
    np.testing.assert_allclose(k, K, atol=1e-11)
    np.testing.assert_allclose(v, V, atol=1e-12)
    # different producer / consumer theta: result is RoPE_cons(deRoPE_prod(K)), not K
    m2 = O.Model(**{**m.__dict__, "rope_theta_consumer": 1e4})
    k2, _ = O.reuse_decode_layer(m2, lay, O.encode_k(m2, lay, K, pos), O.encode_v(m2, lay, V), pos)
    want = O.rope(O.rope(K, pos, 5e5, -1, H, d_h), pos, 1e4, +1, H, d_h)
    np.testing.assert_allclose(k2, want, atol=1e-11)
    assert np.abs(k2 - K).max() > 1e-2


def test_projection_properties_and_eckart_young():
    T, D, r = 200, 24, 6
    X = rng.standard_normal((T, 9)) @ rng.standard_normal((9, D)) + 0.05 * rng.standard_normal((T, D))
    mu = X.mean(0)
    # basis from an independent library routine: numpy SVD of the centred matrix
    U, S, Vt = np.linalg.svd(X - mu, full_matrices=False)
    B = Vt[:r]
    m = _model(n_kv_heads=1, head_dim=D)
    lay = O.Layer(O.REUSE, enc_k=B.T, enc_v=B.T, dec_k=B, dec_v=B, mean_src_k=mu, mean_dst_k=mu,
                  mean_src_v=mu, mean_dst_v=mu)
    z = O.encode_v(m, lay, X)
    _, xhat = O.reuse_decode_layer(m, lay, z, z, np.zeros(T, int))
    # Eckart-Young: squared residual = sum of the discarded sigma^2
    np.testing.assert_allclose(((X - xhat) ** 2).sum(), (S[r:] ** 2).sum(), rtol=1e-10)
    # codes are the top-r principal components U S
    np.testing.assert_allclose(np.abs(z), np.abs(U[:, :r] * S[:r]), atol=1e-10)
    # idempotence: encode(decode(encode(X))) = encode(X); decode∘encode is an orthogonal projector
    np.testing.assert_allclose(O.encode_v(m, lay, xhat), z, atol=1e-12)
    P = B.T @ B
    np.testing.assert_allclose(xhat - mu, (X - mu) @ P, atol=1e-12)
    np.testing.assert_allclose(P @ P, P, atol=1e-12); np.testing.assert_allclose(P, P.T, atol=1e-15)
    # W_enc and W_dec are separate operands (U3): a non-transpose pair must be honoured
    Wenc = rng.standard_normal((D, r)); Wdec = rng.standard_normal((r, D))
    lay2 = O.Layer(O.REUSE, enc_k=Wenc, enc_v=Wenc, dec_k=Wdec, dec_v=Wdec)
    z2 = O.encode_v(m, lay2, X)
    np.testing.assert_allclose(z2, np.einsum("td,dr->tr", X, Wenc), atol=1e-12)
    _, v2 = O.reuse_decode_layer(m, lay2, z2, z2, np.zeros(T, int))
    np.testing.assert_allclose(v2, np.einsum("tr,rd->td", z2, Wdec), atol=1e-12)


def test_k_and_v_use_their_own_artifacts():
    T, D, r = 11, 8, 3
    m = _model(n_kv_heads=2, head_dim=4)
    lay = O.Layer(O.REUSE, enc_k=rng.standard_normal((D, r)), enc_v=rng.standard_normal((D, r + 1)),
                  dec_k=rng.standard_normal((r, D)), dec_v=rng.standard_normal((r + 1, D)),
                  mean_src_k=rng.standard_normal(D), mean_src_v=rng.standard_normal(D),
                  mean_dst_k=rng.standard_normal(D), mean_dst_v=rng.standard_normal(D))
    K, V = rng.standard_normal((T, D)), rng.standard_normal((T, D))
    zk, zv = O.encode_k(m, lay, K, np.zeros(T, int)), O.encode_v(m, lay, V)
    for t in range(T):                                         # element-wise brute force
        for c in range(r):
            assert abs(zk[t, c] - sum((K[t, i] - lay.mean_src_k[i]) * lay.enc_k[i, c] for i in range(D))) < 1e-12
        for c in range(r + 1):
            assert abs(zv[t, c] - sum((V[t, i] - lay.mean_src_v[i]) * lay.enc_v[i, c] for i in range(D))) < 1e-12
    k, v = O.reuse_decode_layer(m, lay, zk, zv, np.zeros(T, int))
    for t in (0, T - 1):
        for c in range(D):
            assert abs(k[t, c] - (sum(zk[t, i] * lay.dec_k[i, c] for i in range(r)) + lay.mean_dst_k[c])) < 1e-12
            assert abs(v[t, c] - (sum(zv[t, i] * lay.dec_v[i, c] for i in range(r + 1)) + lay.mean_dst_v[c])) < 1e-12


def test_per_head_reading_equals_block_diagonal_per_layer():
    """the paper-literal per-head translator W (d_h x r) shared by all heads equals
    the per-layer map with I_H (x) W."""
    H, d_h, r, T = 3, 4, 2, 9
    W_enc, W_dec = rng.standard_normal((d_h, r)), rng.standard_normal((r, d_h))
    X = rng.standard_normal((T, H * d_h))
    per_head = np.stack([X.reshape(T, H, d_h)[:, h] @ W_enc @ W_dec for h in range(H)], 1).reshape(T, -1)
    m = _model(n_kv_heads=H, head_dim=d_h)
    lay = O.Layer(O.REUSE, enc_v=np.kron(np.eye(H), W_enc), dec_v=np.kron(np.eye(H), W_dec),
                  enc_k=np.kron(np.eye(H), W_enc), dec_k=np.kron(np.eye(H), W_dec))
    z = O.encode_v(m, lay, X)
    _, v = O.reuse_decode_layer(m, lay, z, z, np.zeros(T, int))
    np.testing.assert_allclose(v, per_head, atol=1e-13)


# ------------------------------------------------------------------ PATCH (Eq. 11-12)
def test_silu_and_rms_worked_examples():
    for x, y in GOLD["silu"]:
        assert abs(O.silu(np.array([float(x)]))[0] - y) < 5e-7
        assert abs(O.silu(np.array([float(x)]))[0] - x / (1 + math.exp(-x))) < 1e-15
    g = GOLD["norm_rms"]
    m = _model(patch_norm=O.NORM_RMS, rms_eps=0.0)
    lay = O.Layer(O.PATCH, norm_gamma=np.array(g["gamma"]))
    u = np.array([g["u"]], dtype=float)
    assert abs(math.sqrt(sum(v * v for v in g["u"]) / 4) - g["rms"]) < 5e-7
    np.testing.assert_allclose(O.rms_consistent(m, lay, u)[0], g["h"], atol=5e-7)
    assert O.rms_consistent(_model(patch_norm=O.NORM_NONE), lay, u) is u


def _patch_problem(T=13, d=16, H=2, d_h=4, r=6, d_a=10, biases=True):
    D = H * d_h
    lay = O.Layer(O.PATCH, enc_h=rng.standard_normal((d, r)), w1=rng.standard_normal((r, d_a)),
                  b1=rng.standard_normal(d_a) if biases else None, w2=rng.standard_normal((d_a, d)),
                  b2=rng.standard_normal(d) if biases else None, norm_gamma=1 + 0.1 * rng.standard_normal(d),
                  w_k=rng.standard_normal((D, d)), w_v=rng.standard_normal((D, d)),
                  b_k=rng.standard_normal(D) if biases else None, b_v=rng.standard_normal(D) if biases else None)
    return lay, rng.standard_normal((T, r)), rng.integers(0, 4000, T), (T, d, H, d_h, r, d_a)


def test_patch_true_input_invariant():
    """r_h = d, W_enc,H = Q^T orthogonal, act = identity, W1 = Q, W2 = I, no biases => u = x, so
    K, V are the consumer's own RoPE(x_norm W_k), x_norm W_v (computed here with einsum +
    the complex RoPE, independent of patch_layer)."""
    T, d, H, d_h = 7, 8, 2, 4
    D = H * d_h
    Q = _orthobasis(d, d)
    x_raw = rng.standard_normal((T, d))
    gamma = 1 + 0.1 * rng.standard_normal(d)
    w_k, w_v = rng.standard_normal((D, d)), rng.standard_normal((D, d))
    pos = rng.integers(0, 999, T)
    lay = O.Layer(O.PATCH, enc_h=Q.T, w1=Q, w2=np.eye(d), norm_gamma=gamma, w_k=w_k, w_v=w_v)

    def consumer_kv(x_norm):
        k = np.einsum("td,nd->tn", x_norm, w_k); v = np.einsum("td,nd->tn", x_norm, w_v)
        kr = np.array([sum((_rope_complex(list(k[t, h * d_h:(h + 1) * d_h]), int(pos[t]), 5e5, d_h, O.ROPE_HALF)
                            for h in range(H)), []) for t in range(T)])
        return kr, v

    # NORM_NONE, x = consumer's x_norm
    m = O.Model(n_layers=1, d_model=d, n_kv_heads=H, head_dim=d_h, rope_theta_consumer=5e5,
                patch_act=O.ACT_IDENTITY, patch_norm=O.NORM_NONE)
    x_norm = gamma * x_raw / np.sqrt((x_raw ** 2).mean(1, keepdims=True))
    k, v = O.patch_layer(m, lay, O.encode_h(m, lay, x_norm), pos)
    kr, vr = consumer_kv(x_norm)
    np.testing.assert_allclose(k, kr, atol=1e-11); np.testing.assert_allclose(v, vr, atol=1e-11)
    # NORM_RMS, eps = 0, x = x_raw / rms(x_raw) (or any positive multiple: scale invariance)
    m = O.Model(**{**m.__dict__, "patch_norm": O.NORM_RMS, "rms_eps": 0.0})
    for c in (1.0, 37.5):
        k, v = O.patch_layer(m, lay, O.encode_h(m, lay, c * x_raw), pos)
        np.testing.assert_allclose(k, kr, atol=1e-10); np.testing.assert_allclose(v, vr, atol=1e-10)


def test_patch_linear_collapse_and_bruteforce():
    lay, z, pos, (T, d, H, d_h, r, d_a) = _patch_problem(biases=False)
    m = O.Model(n_layers=1, d_model=d, n_kv_heads=H, head_dim=d_h, rope_theta_consumer=1e4,
                patch_act=O.ACT_IDENTITY, patch_norm=O.NORM_NONE)
    # identity activation, no norm: the chain is one matrix W1 W2 [W_k^T W_v^T]
    M = np.linalg.multi_dot([lay.w1, lay.w2, np.concatenate([lay.w_k.T, lay.w_v.T], 1)])
    k, v = O.patch_layer(m, lay, z, pos)
    kv = z @ M
    np.testing.assert_allclose(O.rope(k, pos, 1e4, -1, H, d_h), kv[:, :H * d_h], atol=1e-10)
    np.testing.assert_allclose(v, kv[:, H * d_h:], atol=1e-10)
    # full chain with SiLU, RMS, all biases: scalar loops for one row
    lay, z, pos, _ = _patch_problem(biases=True)
    m = O.Model(n_layers=1, d_model=d, n_kv_heads=H, head_dim=d_h, rope_theta_consumer=1e4,
                patch_act=O.ACT_SILU, patch_norm=O.NORM_RMS, rms_eps=1e-5)
    k, v = O.patch_layer(m, lay, z, pos)
    t = 4
    a = [sum(z[t, i] * lay.w1[i, j] for i in range(r)) + lay.b1[j] for j in range(d_a)]
    a = [x / (1 + math.exp(-x)) for x in a]
    u = [sum(a[j] * lay.w2[j, c] for j in range(d_a)) + lay.b2[c] for c in range(d)]
    ms = sum(x * x for x in u) / d
    h = [lay.norm_gamma[c] * u[c] / math.sqrt(ms + 1e-5) for c in range(d)]
    kk = [sum(h[c] * lay.w_k[n, c] for c in range(d)) + lay.b_k[n] for n in range(H * d_h)]
    vv = [sum(h[c] * lay.w_v[n, c] for c in range(d)) + lay.b_v[n] for n in range(H * d_h)]
    kk = sum((_rope_complex(kk[hh * d_h:(hh + 1) * d_h], int(pos[t]), 1e4, d_h, O.ROPE_HALF) for hh in range(H)), [])
    np.testing.assert_allclose(k[t], kk, atol=1e-10); np.testing.assert_allclose(v[t], vv, atol=1e-10)


# ------------------------------------------------------------------ paging / routing / payload
def test_slot_mapping_bruteforce_and_identity():
    g = GOLD["slot"]
    b = O.Batch(np.array([0, 40]), np.array([g["page_table"]]))
    assert O.slot_mapping(b, g["block_size"])[g["t"]] == g["slot"]
    lens = [5, 16, 33, 1, 48]
    bs = 16
    pages = [(l + bs - 1) // bs for l in lens]
    perm = rng.permutation(sum(pages) + 3)
    table = -np.ones((len(lens), max(pages)), int)
    at = 0
    for i, p in enumerate(pages):
        table[i, :p] = perm[at:at + p]; at += p
    cu = np.concatenate([[0], np.cumsum(lens)])
    batch = O.Batch(cu, table, np.array([0, 100, 7, 0, 3]))
    slots, pos = O.slot_mapping(batch, bs), O.positions(batch)
    n = 0
    for i, l in enumerate(lens):                       # walk every request token by token
        for t in range(l):
            assert slots[n] == table[i][t // bs] * bs + t % bs
            assert pos[n] == [0, 100, 7, 0, 3][i] + t
            n += 1
    assert len(set(slots.tolist())) == len(slots)      # no two tokens share a slot
    # identity page table, one request = contiguous layout
    one = O.Batch(np.array([0, 37]), np.arange(3)[None, :])
    np.testing.assert_array_equal(O.slot_mapping(one, bs), np.arange(37))
    # write_paged touches exactly those rows
    pool = np.full((perm.size, bs, 2, 3), -7.0)
    rows = rng.standard_normal((len(slots), 6))
    O.write_paged(pool, slots, rows)
    flat = pool.reshape(-1, 6)
    np.testing.assert_array_equal(flat[slots], rows)
    untouched = np.setdiff1d(np.arange(flat.shape[0]), slots)
    assert np.all(flat[untouched] == -7.0)
    # read_paged (paged producer cache) is the inverse walk: token by token through the table
    got = O.read_paged(pool, slots)
    n = 0
    for i, l in enumerate(lens):
        for t in range(l):
            np.testing.assert_array_equal(got[n], pool[table[i][t // bs], t % bs].reshape(-1))
            n += 1
    np.testing.assert_array_equal(got, rows)


def test_route_and_payload():
    r_k, r_v, r_h, D, d = 4, 6, 5, 8, 16
    reuse = O.Layer(O.REUSE, enc_k=np.zeros((D, r_k)), enc_v=np.zeros((D, r_v)))
    patch = O.Layer(O.PATCH, enc_h=np.zeros((d, r_h)))
    layers = [reuse, patch, reuse, reuse, patch]
    assert O.route(layers) == ([0, 2, 3], [1, 4])
    T = 100
    for dt, cb, sb in ((O.F32, 4, 0), (O.BF16, 2, 0), (O.E4M3_ROWSCALE, 1, 4)):
        m = _model(code_dtype=dt)
        want = T * (3 * ((r_k + r_v) * cb + 2 * sb) + 2 * (r_h * cb + sb))
        assert O.payload_bytes(m, layers, T) == want
    # config-2 figure quoted in SURVEY 8(a): 29 reuse x 2 x 128 + 3 x 128 codes, bf16, 8192 tokens = 128 MB
    big = [O.Layer(O.REUSE, enc_k=np.zeros((1, 128)), enc_v=np.zeros((1, 128)))] * 29 + \
          [O.Layer(O.PATCH, enc_h=np.zeros((1, 128)))] * 3
    assert O.payload_bytes(_model(code_dtype=O.BF16), big, 8192) == 8192 * 61 * 128 * 2


# ------------------------------------------------------------------ whole-call forms + third opinion
def test_whole_call_tiny_against_torch_fp64():
    """Tiny-shaped end to end (encode -> pack -> reuse_decode + patch -> paged pools) against
    an independent torch fp64 evaluation; also checks that PATCH layers get only Z_H
     and REUSE layers only Z_K, Z_V."""
    H, d_h, d, r, T1, T2 = 2, 8, 24, 5, 21, 10
    D = H * d_h
    m = O.Model(n_layers=3, d_model=d, n_kv_heads=H, head_dim=d_h, rope_theta_producer=1e4,
                rope_theta_consumer=5e5, code_dtype=O.F32)
    layers = []
    for i in range(3):
        if i == 1:
            lay, _, _, _ = _patch_problem(d=d, H=H, d_h=d_h, r=r, d_a=12)
            lay.mean_src_h = rng.standard_normal(d)
        else:
            lay = O.Layer(O.REUSE, enc_k=rng.standard_normal((D, r)), enc_v=rng.standard_normal((D, r)),
                          dec_k=rng.standard_normal((r, D)), dec_v=rng.standard_normal((r, D)),
                          mean_src_k=rng.standard_normal(D), mean_dst_v=rng.standard_normal(D))
        layers.append(lay)
    table = np.array([[4, 0, -1], [2, -1, -1]]) if T1 <= 32 else None
    batch = O.Batch(np.array([0, T1, T1 + T2]), table, np.array([3, 50]))
    T = T1 + T2
    K = {i: rng.standard_normal((T, D)) for i in (0, 2)}
    V = {i: rng.standard_normal((T, D)) for i in (0, 2)}
    Hs = {1: rng.standard_normal((T, d))}
    codes = O.scd_encode(m, layers, batch, K, V, Hs)
    assert sorted(codes) == [(0, 0), (0, 1), (1, 2), (2, 0), (2, 1)]
    kp = {i: np.full((5, 16, H, d_h), np.nan) for i in range(3)}
    vp = {i: np.full((5, 16, H, d_h), np.nan) for i in range(3)}
    O.scd_reuse_decode(m, layers, batch, codes, kp, vp)
    assert np.isnan(kp[1]).all() and not np.isnan(kp[0]).all()
    O.scd_patch(m, layers, batch, codes, kp, vp)

    # --- torch fp64 third opinion ---
    tt = lambda a: torch.from_numpy(np.asarray(a, dtype=np.float64))
    pos = torch.cat([3 + torch.arange(T1), 50 + torch.arange(T2)]).double()
    slots = torch.cat([torch.tensor([4, 0])[torch.arange(T1) // 16] * 16 + torch.arange(T1) % 16,
                       torch.tensor([2])[torch.arange(T2) // 16] * 16 + torch.arange(T2) % 16])

    def trope(x, theta, sign):
        xh = x.view(T, H, d_h)
        inv = theta ** (-torch.arange(0, d_h, 2).double() / d_h)
        ang = sign * pos[:, None] * inv[None, :]
        cos, sin = torch.cat([ang.cos()] * 2, -1)[:, None], torch.cat([ang.sin()] * 2, -1)[:, None]
        rot = torch.cat([-xh[..., d_h // 2:], xh[..., :d_h // 2]], -1)       # HF rotate_half
        return (xh * cos + rot * sin).reshape(T, D)

    for i in (0, 2):
        l = layers[i]
        zk = ((trope(tt(K[i]), 1e4, -1) - tt(l.mean_src_k)) @ tt(l.enc_k)).float().double()
        zv = (tt(V[i]) @ tt(l.enc_v)).float().double()
        k = trope(zk @ tt(l.dec_k), 5e5, +1)
        v = zv @ tt(l.dec_v) + tt(l.mean_dst_v)
        np.testing.assert_allclose(kp[i].reshape(-1, D)[slots], k.numpy(), atol=1e-9)
        np.testing.assert_allclose(vp[i].reshape(-1, D)[slots], v.numpy(), atol=1e-9)
    l = layers[1]
    zh = ((tt(Hs[1]) - tt(l.mean_src_h)) @ tt(l.enc_h)).float().double()
    u = torch.nn.functional.silu(zh @ tt(l.w1) + tt(l.b1)) @ tt(l.w2) + tt(l.b2)
    hh = tt(l.norm_gamma) * u * torch.rsqrt((u * u).mean(-1, keepdim=True) + 1e-5)
    k = trope(hh @ tt(l.w_k).T + tt(l.b_k), 5e5, +1)
    v = hh @ tt(l.w_v).T + tt(l.b_v)
    np.testing.assert_allclose(kp[1].reshape(-1, D)[slots], k.numpy(), atol=1e-9)
    np.testing.assert_allclose(vp[1].reshape(-1, D)[slots], v.numpy(), atol=1e-9)
    # nothing but the addressed slots was written
    mask = np.ones(5 * 16, bool); mask[slots.numpy()] = False
    for i in range(3):
        assert np.isnan(kp[i].reshape(-1, D)[mask]).all() and np.isnan(vp[i].reshape(-1, D)[mask]).all()
    # row-subset form writes the same values for those rows
    kp2 = {i: np.full((5, 16, H, d_h), np.nan) for i in range(3)}
    vp2 = {i: np.full((5, 16, H, d_h), np.nan) for i in range(3)}
    sel = np.array([0, 5, 20, 21, 30])
    O.scd_reuse_decode(m, layers, batch, codes, kp2, vp2, rows=sel)
    O.scd_patch(m, layers, batch, codes, kp2, vp2, rows=sel)
    s_np = slots.numpy()
    for i in range(3):
        np.testing.assert_array_equal(kp2[i].reshape(-1, D)[s_np[sel]], kp[i].reshape(-1, D)[s_np[sel]])
        assert np.isnan(kp2[i].reshape(-1, D)[np.setdiff1d(np.arange(80), s_np[sel])]).all()


def test_per_head_mode_against_block_diagonal_and_scalar_loops():
    """Paper-literal REUSE (heads flattened into the sample axis, one d_h x r map for
    all heads) as Model(reuse_per_head=True): pinned (i) against the per-layer functions with I_H (x) W and the
    mean tiled over heads -- the reading pinned above, now the other way round -- and (ii) against plain scalar
    loops over (token, head, code) with RoPE from the complex-multiplication form."""
    rng = np.random.default_rng(11)
    T, H, d_h, r_k, r_v = 5, 3, 8, 4, 2
    D = H * d_h
    K, V = rng.standard_normal((T, D)), rng.standard_normal((T, D))
    ek, dk = rng.standard_normal((d_h, r_k)), rng.standard_normal((r_k, d_h))
    ev, dv = rng.standard_normal((d_h, r_v)), rng.standard_normal((r_v, d_h))
    mk, mv, nk, nv = (rng.standard_normal(d_h) for _ in range(4))
    pos = np.array([0, 3, 7, 8, 100])
    ph = O.Model(1, 16, H, d_h, rope_theta_producer=1e4, rope_theta_consumer=5e5, reuse_per_head=True)
    pl = O.Model(1, 16, H, d_h, rope_theta_producer=1e4, rope_theta_consumer=5e5)
    lay_h = O.Layer(O.REUSE, enc_k=ek, dec_k=dk, enc_v=ev, dec_v=dv, mean_src_k=mk, mean_src_v=mv, mean_dst_k=nk, mean_dst_v=nv)
    eye = np.eye(H)
    lay_l = O.Layer(O.REUSE, enc_k=np.kron(eye, ek), dec_k=np.kron(eye, dk), enc_v=np.kron(eye, ev), dec_v=np.kron(eye, dv),
                    mean_src_k=np.tile(mk, H), mean_src_v=np.tile(mv, H), mean_dst_k=np.tile(nk, H), mean_dst_v=np.tile(nv, H))
    zk, zv = O.encode_k(ph, lay_h, K, pos), O.encode_v(ph, lay_h, V)
    assert zk.shape == (T, H * r_k) and zv.shape == (T, H * r_v)
    np.testing.assert_allclose(zk, O.encode_k(pl, lay_l, K, pos), atol=1e-12)
    np.testing.assert_allclose(zv, O.encode_v(pl, lay_l, V), atol=1e-12)
    k1, v1 = O.reuse_decode_layer(ph, lay_h, zk, zv, pos)
    k2, v2 = O.reuse_decode_layer(pl, lay_l, zk, zv, pos)
    np.testing.assert_allclose(k1, k2, atol=1e-12)
    np.testing.assert_allclose(v1, v2, atol=1e-12)
    # (ii) scalar loops
    def rot(x, p, theta, sign):          # one head, HALF pairing, complex multiplication
        out = np.empty(d_h)
        for j in range(d_h // 2):
            z = complex(x[j], x[j + d_h // 2]) * cmath.exp(1j * sign * p * theta ** (-2.0 * j / d_h))
            out[j], out[j + d_h // 2] = z.real, z.imag
        return out
    for t in range(T):
        for h in range(H):
            kc = rot(K[t, h * d_h:(h + 1) * d_h], pos[t], 1e4, -1)
            for i in range(r_k):
                assert abs(zk[t, h * r_k + i] - sum((kc[j] - mk[j]) * ek[j, i] for j in range(d_h))) < 1e-12
            for i in range(r_v):
                assert abs(zv[t, h * r_v + i] - sum((V[t, h * d_h + j] - mv[j]) * ev[j, i] for j in range(d_h))) < 1e-12
            kd = np.array([sum(zk[t, h * r_k + i] * dk[i, j] for i in range(r_k)) + nk[j] for j in range(d_h)])
            np.testing.assert_allclose(k1[t, h * d_h:(h + 1) * d_h], rot(kd, pos[t], 5e5, +1), atol=1e-12)
            for j in range(d_h):
                assert abs(v1[t, h * d_h + j] - (sum(zv[t, h * r_v + i] * dv[i, j] for i in range(r_v)) + nv[j])) < 1e-12
    # payload: H * r codes per token and branch
    assert O.payload_bytes(ph, [lay_h], 10) == 10 * H * (r_k + r_v) * 4


# ------------------------------------------------------------------ fp8 pools (build extension U20)
def test_quantize_pool_scalar_walk_and_properties():
    """Per (token, head) walk with torch's fp32 / bf16 / float8 arithmetic as the independent side; the amax element of
    every head maps to +-448; |deq - x| <= 2^-4 |x| in the normal range; an all-zero head has scale 1 and bytes 0."""
    H, d_h, T = 3, 16, 9
    y = rng.standard_normal((T, H * d_h)) * np.array([0.01, 1.0, 30.0]).repeat(d_h)[None, :]
    y[4, d_h:2 * d_h] = 0.0
    q, s = O.quantize_pool(y, H)
    assert q.dtype == np.uint8 and s.dtype == np.float32 and q.shape == y.shape and s.shape == (T, H)
    xb = torch.from_numpy(y).to(torch.bfloat16).float()
    for t in range(T):
        for h in range(H):
            xs = xb[t, h * d_h:(h + 1) * d_h]
            amax = xs.abs().max()
            sc = (amax / torch.tensor(448.0)) if amax > 0 else torch.tensor(1.0)
            assert float(sc) == float(s[t, h])
            inv = torch.tensor(1.0) / sc
            for i in range(d_h):
                v = float(xs[i] * inv)                       # fp32 product
                want = torch.tensor(max(-448.0, min(448.0, v))).to(torch.float8_e4m3fn).view(torch.uint8).item()
                got = int(q[t, h * d_h + i])
                assert got == want or (O.E4M3_VALUES[got] == 0 and O.E4M3_VALUES[want] == 0), (t, h, i, v, got, want)
            if amax > 0:
                assert 448.0 in np.abs(O.E4M3_VALUES[q[t, h * d_h:(h + 1) * d_h]])
    assert s[4, 1] == 1.0 and not (q[4, d_h:2 * d_h] & 0x7F).any()
    deq = O.dequantize_pool(q, s)
    x64 = xb.double().numpy()
    big = np.abs(x64) >= np.repeat(s, d_h, axis=1) * 2.0 ** -6       # normal range of the head's scale
    assert np.all(np.abs(deq - x64)[big] <= 2.0 ** -4 * np.abs(x64)[big] * (1 + 1e-6))
