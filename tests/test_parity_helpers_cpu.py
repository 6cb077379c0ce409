"""The block / element bounds of tests/_parity.py (fine_check) must pass what the CUDA path legitimately produces and
must fail the faults a layer-wide Frobenius norm hides: one wrong head of one token, one wrong 16-column chunk, two
swapped rows.  The "GPU result" here is the oracle's fp64 value rounded to bf16 -- the best a correct kernel can do."""
import numpy as np
import pytest

from oracle import scd_oracle as O
from tests import _parity as P
from paper_2606_07684_b200 import workloads as W

T, H, DH, R = 1000, 8, 128, 128


def _decode_case(seed=0):
    rng = np.random.default_rng(seed)
    om = O.Model(n_layers=1, d_model=1024, n_kv_heads=H, head_dim=DH, rope_theta_consumer=5e5, code_dtype=O.BF16)
    s = 0.97 ** np.arange(R)
    z = rng.standard_normal((T, R)) * s[None, :]
    q, _ = np.linalg.qr(rng.standard_normal((H * DH, R)))
    lay = O.Layer(O.REUSE, dec_k=q.T, dec_v=q.T, mean_dst_k=0.1 * rng.standard_normal(H * DH),
                  mean_dst_v=0.1 * rng.standard_normal(H * DH))
    k, v = O.reuse_decode_layer(om, lay, z, z, np.arange(T))
    return k, v


def _check(got, want):
    return P.fine_check(got, want, H, P.FINE_TOL[W.BF16], P.REL_OUT[W.BF16], P.K_ABS["reuse"][W.BF16], "case")


def test_correctly_rounded_output_passes_with_margin():
    for want in _decode_case():
        used = _check(O.round_to_bf16(want), want)
        assert used["block"] < 0.25 and used["element"] <= 1.0      # half-ulp rounding sits exactly on `rel`


@pytest.mark.parametrize("fault", ["wrong_head", "wrong_chunk", "swapped_rows", "zeroed_chunk", "off_by_one_position"])
def test_local_faults_fail_although_the_layer_norm_passes(fault):
    want, _ = _decode_case(1)
    got = O.round_to_bf16(want)
    rng = np.random.default_rng(2)
    if fault == "wrong_head":                      # one head of one token replaced by another token's
        got[500, 3 * DH:4 * DH] = got[17, 3 * DH:4 * DH]
    elif fault == "wrong_chunk":                   # one 16-column chunk (a 32-byte store) from a neighbouring row
        got[123, 640:656] = got[124, 640:656]
    elif fault == "swapped_rows":
        got[[10, 11]] = got[[11, 10]]
    elif fault == "zeroed_chunk":
        got[777, 256:272] = 0.0
    else:                                          # RoPE applied with position p + 1 to one row
        om = O.Model(n_layers=1, d_model=1024, n_kv_heads=H, head_dim=DH, rope_theta_consumer=5e5)
        raw = O.rope(want[300:301], np.array([300]), 5e5, -1, H, DH)
        got[300] = O.round_to_bf16(O.rope(raw, np.array([301]), 5e5, +1, H, DH))[0]
    if fault != "swapped_rows":                    # (two whole rows of 1000 move the layer norm by 4.6e-2; of 8192 by 1.6e-2)
        assert P.rel_fro(got, want) <= P.TOL[W.BF16]               # the north_star criterion alone does not see it
    with pytest.raises(AssertionError):
        _check(got, want)


def test_rerounded_operand_noise_term_is_a_bound_not_a_blank_cheque():
    """The K-encode noise term (U15) must cover the real effect of re-rounding the rotated operand to
    bf16 and stay far below the Cauchy-Schwarz worst case it replaced."""
    rng = np.random.default_rng(3)
    om = O.Model(n_layers=1, d_model=1024, n_kv_heads=H, head_dim=DH, rope_theta_producer=5e5, code_dtype=O.BF16)
    kt = rng.standard_normal((256, H * DH)) * 0.2
    q, _ = np.linalg.qr(rng.standard_normal((H * DH, R)))
    lay = O.Layer(O.REUSE, enc_k=q)
    extra = P._rerounded_operand_noise(om, lay, kt)
    real = np.abs(O.round_to_bf16(kt) @ q - kt @ q)                 # the effect of the re-rounding alone
    assert (real <= extra).all() and real.max() >= 0.1 * extra.min()
    cauchy = 2.0 ** -8 * np.linalg.norm(kt, axis=1)[:, None] * np.linalg.norm(q, axis=0)[None, :]
    assert extra.max() < cauchy.min() / 8.0


def test_e4m3_cell_check_accepts_the_oracles_own_codes_and_rejects_a_neighbouring_code():
    rng = np.random.default_rng(4)
    z = rng.standard_normal((64, 96)) * (0.97 ** np.arange(96))[None, :]
    z[5] = 0.0                                                     # all-zero row: scale 1, codes 0
    q, s = O.pack_codes(z, O.E4M3_ROWSCALE)
    tiny = np.full(z.shape, 1e-12)
    assert P.e4m3_cell_check(z, q, s, tiny, "own codes") == 0.0
    bad = q.copy()
    bad[10, 3] = bad[10, 3] + 1 if (bad[10, 3] & 0x7F) < 0x7E else bad[10, 3] - 1      # the next code up (or down at the top)
    with pytest.raises(AssertionError):
        P.e4m3_cell_check(z, bad, s, tiny, "neighbouring code")
    flipped = q.copy()
    flipped[20, 7] ^= 0x80                                         # wrong sign
    if (q[20, 7] & 0x7F) != 0:
        with pytest.raises(AssertionError):
            P.e4m3_cell_check(z, flipped, s, tiny, "wrong sign")
    # a value just past a rounding boundary may legitimately take either neighbour when the noise allowance covers it
    z2 = np.array([[448.0, 17.0 + 1e-9]])                          # scale 1; 17 is the midpoint of codes 16 and 18
    q2 = np.array([[0x7E, O.e4m3_quantize(np.array([16.0]))[0]]], dtype=np.uint8)
    assert 0.0 < P.e4m3_cell_check(z2, q2, np.ones(1, np.float32), np.full((1, 2), 1e-6), "boundary") <= 1.0
