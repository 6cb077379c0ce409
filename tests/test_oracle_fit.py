"""Pins for oracle/fit_oracle.py (offline REUSE calibration: stack-SVD + ridge).

Pinned by things other than the oracle's own library calls: a plain one-sided Jacobi SVD written here (the
"brute-force SVD on tiny inputs" BASELINE.json's north_star asks for), the eigen-decomposition of X^T X, the
planted subspace of a noise-free input, Eckart-Young, exact rational normal equations, and the stationarity
condition of the ridge objective.  CPU only.
"""
from fractions import Fraction

import numpy as np
import pytest

from oracle import fit_oracle as F

rng = np.random.default_rng(2606)


def jacobi_svd(x, sweeps=60, tol=1e-15):
    """One-sided (Hestenes) Jacobi: rotate column pairs of U = X until they are mutually orthogonal; then
    sigma_j = ||u_j||, V accumulates the rotations.  Plain loops, no library decomposition."""
    u = np.array(x, dtype=np.float64)
    n = u.shape[1]
    v = np.eye(n)
    for _ in range(sweeps):
        off = 0.0
        for p in range(n - 1):
            for q in range(p + 1, n):
                a, b, c = u[:, p] @ u[:, p], u[:, q] @ u[:, q], u[:, p] @ u[:, q]
                if abs(c) <= tol * np.sqrt(a * b) or c == 0.0:
                    continue
                off = max(off, abs(c) / np.sqrt(a * b))
                zeta = (b - a) / (2.0 * c)
                t = np.sign(zeta) / (abs(zeta) + np.sqrt(1.0 + zeta * zeta)) if zeta != 0 else 1.0
                cs = 1.0 / np.sqrt(1.0 + t * t)
                sn = cs * t
                for m in (u, v):
                    mp, mq = m[:, p].copy(), m[:, q].copy()
                    m[:, p], m[:, q] = cs * mp - sn * mq, sn * mp + cs * mq
        if off <= tol:
            break
    s = np.linalg.norm(u, axis=0)
    order = np.argsort(-s)
    return s[order], v[:, order]


def _planted(n, w, k, decay=0.8, noise=0.0, seed=0):
    g = np.random.default_rng(seed)
    q, _ = np.linalg.qr(g.standard_normal((2 * w, k)))
    s = decay ** np.arange(k)
    x = (g.standard_normal((n, k)) * s) @ q.T + noise * g.standard_normal((n, 2 * w))
    return x[:, :w], x[:, w:], q


def test_joint_svd_against_brute_force_jacobi_eigh_and_planted_subspace():
    a, b, q = _planted(60, 5, 4, noise=0.0, seed=1)
    r = 4
    s, v = F.joint_svd(a, b, r)
    x = np.concatenate([a, b], axis=1)
    sj, vj = jacobi_svd(x)
    np.testing.assert_allclose(s, sj[:r], rtol=1e-12)
    np.testing.assert_allclose(v @ v.T, vj[:, :r] @ vj[:, :r].T, atol=1e-11)
    lam, e = np.linalg.eigh(x.T @ x)                               # third opinion: eigen-decomposition of the Gram matrix
    np.testing.assert_allclose(s ** 2, lam[::-1][:r], rtol=1e-11)
    np.testing.assert_allclose(v @ v.T, e[:, ::-1][:, :r] @ e[:, ::-1][:, :r].T, atol=1e-10)
    np.testing.assert_allclose(v @ v.T, q @ q.T, atol=1e-10)       # noise-free: the top-k subspace IS the planted one
    assert sj[r] < 1e-12 * sj[0]
    # with noise the three decompositions still agree with one another
    a, b, _ = _planted(80, 6, 5, noise=0.05, seed=2)
    s, v = F.joint_svd(a, b, 3)
    sj, vj = jacobi_svd(np.concatenate([a, b], axis=1))
    np.testing.assert_allclose(s, sj[:3], rtol=1e-12)
    np.testing.assert_allclose(v @ v.T, vj[:, :3] @ vj[:, :3].T, atol=1e-10)


def test_eq6_is_the_best_rank_r_approximation():
    """A ~ Z W_dec,A, B ~ Z W_dec,B (Eq. 6): the residual is exactly the discarded singular values (Eckart-Young, :585);
    decoder rows are orthonormal; Z = U S (U4)."""
    a, b, _ = _planted(200, 8, 10, noise=0.02, seed=3)
    r = 6
    fit = F.fit_reuse(a, b, r, lam_rel=0.0)
    x = np.concatenate([a, b], axis=1)
    vt = np.concatenate([fit.w_dec_a, fit.w_dec_b], axis=1)
    z = x @ vt.T
    s_all = jacobi_svd(x)[0]
    np.testing.assert_allclose(np.sum((x - z @ vt) ** 2), np.sum(s_all[r:] ** 2), rtol=1e-10)
    np.testing.assert_allclose(vt @ vt.T, np.eye(r), atol=1e-12)
    np.testing.assert_allclose(np.linalg.norm(z, axis=0), fit.sigma, rtol=1e-12)      # columns of U S
    np.testing.assert_allclose(fit.sigma, s_all[:r], rtol=1e-12)
    assert np.all(np.diff(fit.sigma) <= 0)


def test_ridge_exact_rational_normal_equations():
    """3 x 2 example: (A^T A + lam I) W = A^T Z solved by Cramer's rule in exact rationals."""
    A = [[1, 2], [0, 1], [3, -1]]
    Z = [[2], [1], [-1]]
    lam = Fraction(1, 2)
    ata = [[sum(Fraction(A[i][p]) * A[i][q] for i in range(3)) + (lam if p == q else 0) for q in range(2)] for p in range(2)]
    atz = [sum(Fraction(A[i][p]) * Z[i][0] for i in range(3)) for p in range(2)]
    det = ata[0][0] * ata[1][1] - ata[0][1] * ata[1][0]
    w0 = (atz[0] * ata[1][1] - ata[0][1] * atz[1]) / det
    w1 = (ata[0][0] * atz[1] - atz[0] * ata[1][0]) / det
    # by hand: A^T A = [[10, -1], [-1, 6]], + lam I = [[10.5, -1], [-1, 6.5]], A^T Z = [-1, 6]; det = 67.25
    assert (ata, atz, det) == ([[Fraction(21, 2), -1], [-1, Fraction(13, 2)]], [-1, 6], Fraction(269, 4))
    got = F.ridge(np.array(A, float), np.array(Z, float), float(lam))
    np.testing.assert_allclose(got[:, 0], [float(w0), float(w1)], rtol=1e-14)
    assert (w0, w1) == (Fraction(-2, 269), Fraction(248, 269))


def test_ridge_stationarity_limits_and_lambda_rule():
    a = rng.standard_normal((50, 7))
    z = rng.standard_normal((50, 3))
    lam = 0.37
    w = F.ridge(a, z, lam)
    np.testing.assert_allclose(a.T @ (a @ w - z) + lam * w, 0, atol=1e-12)          # gradient of Eq. 7 vanishes
    # objective is not improved by random perturbations
    obj = lambda w_: np.sum((a @ w_ - z) ** 2) + lam * np.sum(w_ ** 2)
    for _ in range(20):
        assert obj(w + 1e-3 * rng.standard_normal(w.shape)) > obj(w)
    np.testing.assert_allclose(F.ridge(a, z, 0.0), np.linalg.lstsq(a, z, rcond=None)[0], atol=1e-12)
    assert np.abs(F.ridge(a, z, 1e12)).max() < 1e-9
    # U4: lam = lam_rel * trace(A^T A) / W ; hand example: A = [[1, 2], [3, 4]] -> trace 30, W = 2
    assert F.ridge_lambda(np.array([[1.0, 2.0], [3.0, 4.0]]), 1e-3) == pytest.approx(0.015, rel=1e-15)


def test_fit_closed_forms():
    """(i) B = A M (consumer states linear in the producer's): Z lies in the column space of A, so with lam = 0
    A W_enc = Z exactly and encode -> decode reproduces the rank-r truncation of B.  (ii) A = B: decoders are equal,
    W_enc W_dec,B = V_A V_A^T (the PCA projector of A), sigma = sqrt(2) sigma(A)."""
    a = rng.standard_normal((120, 6)) @ np.diag(0.7 ** np.arange(6))
    m = rng.standard_normal((6, 6))
    b = a @ m
    fit = F.fit_reuse(a, b, 4, lam_rel=0.0)
    x = np.concatenate([a, b], axis=1)
    vt = np.concatenate([fit.w_dec_a, fit.w_dec_b], axis=1)
    np.testing.assert_allclose(a @ fit.w_enc, x @ vt.T, atol=1e-9)
    np.testing.assert_allclose(a @ fit.w_enc @ fit.w_dec_b, (x @ vt.T @ vt)[:, 6:], atol=1e-9)
    fit2 = F.fit_reuse(a, a, 3, lam_rel=0.0)
    np.testing.assert_allclose(fit2.w_dec_a, fit2.w_dec_b, atol=1e-12)
    sa, va = jacobi_svd(a)
    np.testing.assert_allclose(fit2.sigma, np.sqrt(2.0) * sa[:3], rtol=1e-12)
    np.testing.assert_allclose(fit2.w_enc @ fit2.w_dec_b, va[:, :3] @ va[:, :3].T, atol=1e-10)


def test_centring_and_invariants_are_sign_free():
    a, b, _ = _planted(150, 6, 5, noise=0.03, seed=9)
    a = a + 3.0
    b = b - 1.5
    fit = F.fit_reuse(a, b, 4, lam_rel=1e-3, center=True)
    np.testing.assert_allclose(fit.mu_a, a.mean(axis=0), rtol=1e-14)
    np.testing.assert_allclose(fit.mu_b, b.mean(axis=0), rtol=1e-14)
    ref = F.fit_reuse(a - a.mean(axis=0), b - b.mean(axis=0), 4, lam_rel=1e-3, center=False)
    p1, m1 = F.invariants(fit)
    p0, m0 = F.invariants(ref)
    np.testing.assert_allclose(p1, p0, atol=1e-12)
    np.testing.assert_allclose(m1, m0, atol=1e-12)
    # flipping the sign of a latent direction changes W_enc and W_dec but not the invariants (U14)
    flip = F.ReuseFit(fit.w_enc * [-1, 1, 1, -1], fit.w_dec_a * np.array([-1, 1, 1, -1])[:, None],
                      fit.w_dec_b * np.array([-1, 1, 1, -1])[:, None], fit.sigma, fit.mu_a, fit.mu_b, fit.lam)
    p2, m2 = F.invariants(flip)
    np.testing.assert_allclose(p2, p1, atol=1e-14)
    np.testing.assert_allclose(m2, m1, atol=1e-14)
    assert p1.shape == (12, 12) and m1.shape == (6, 12)
    np.testing.assert_allclose(p1 @ p1, p1, atol=1e-12)              # an orthogonal projector of rank r
    assert round(np.trace(p1)) == 4
