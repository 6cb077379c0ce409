"""CPU oracle for the offline REUSE calibration fit: stack-SVD + ridge encoder.

TEST INFRASTRUCTURE ONLY (same rules as scd_oracle.py: imported by tests/, smoke() and bench.py's CPU legs,
shares nothing with the CUDA path).  numpy fp64; the SVD and the linear solve are library primitives used as
single steps, in the paper's order.

What the paper defines (section 4.3.1, Eq. 6-7; App. F.1 :583-586), per layer and branch:

  1. paired samples A (producer), B (consumer) in R^{N x W}, flattened over prefixes (keys are deRoPE'd first,
     Eq. 5 :124 -- the caller hands content-space keys); joint matrix X = [A B] in R^{N x 2W}   (:129)
  2. rank-r truncated SVD of X ("Subspace Identification via Truncated SVD", :585):  X ~ U_r S_r V_r^T.
     Latents Z = U_r S_r = X V_r in R^{N x r}; decoders [W_dec,A  W_dec,B] = V_r^T in R^{r x 2W}, so that
     A ~ Z W_dec,A and B ~ Z W_dec,B                                                          (Eq. 6 :131)
  3. producer encoder by ridge regression (Eq. 7 :139, F.1 :586):
        W_enc = argmin_W ||A W - Z||_F^2 + lam ||W||_F^2 = (A^T A + lam I)^-1 A^T Z

Readings where the paper is silent:
  * the scale split of the SVD factors: Z = U S (all of the scale in the latents), W_dec = V_r^T (orthonormal rows);
  * lam = lam_rel * trace(A^T A) / W with lam_rel = 1e-3;
  * optional centring (build extension, U2): mu_A, mu_B = column means, the fit runs on A - mu_A, B - mu_B and the
    means become mu_src = mu_A (encode) and mu_dst = mu_B (decode); `center=False` is the paper-literal case.

Several results are correct (U14): V_r is defined up to the sign of each column (and a rotation inside equal
singular values), so tests compare the singular values, the projector V_r V_r^T and the sign-free products
W_enc W_dec, never basis entries.

Parity pins: tests/test_oracle_fit.py (a plain one-sided Jacobi SVD written in the test, eigen-decomposition of
X^T X, the planted subspace, Eckart-Young, exact rational normal equations, stationarity of the ridge objective).
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional, Tuple

import numpy as np


def ridge_lambda(a: np.ndarray, lam_rel: float) -> float:
    """lam = lam_rel * trace(A^T A) / W."""
    a = np.asarray(a, dtype=np.float64)
    return float(lam_rel) * float(np.sum(a * a)) / a.shape[1]


def ridge(a: np.ndarray, z: np.ndarray, lam: float) -> np.ndarray:
    """Eq. 7: (A^T A + lam I)^-1 A^T Z."""
    a = np.asarray(a, dtype=np.float64)
    z = np.asarray(z, dtype=np.float64)
    return np.linalg.solve(a.T @ a + lam * np.eye(a.shape[1]), a.T @ z)


def joint_svd(a: np.ndarray, b: np.ndarray, r: int) -> Tuple[np.ndarray, np.ndarray]:
    """Top-r singular values [r] and right singular vectors V_r [2W, r] of X = [A B]."""
    x = np.concatenate([np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)], axis=1)
    _, s, vt = np.linalg.svd(x, full_matrices=False)
    return s[:r].copy(), vt[:r].T.copy()


@dataclass
class ReuseFit:
    w_enc: np.ndarray            # [W, r]   producer encoder (Eq. 7)
    w_dec_a: np.ndarray          # [r, W]   producer-side decoder (Eq. 6; not used by the hot path)
    w_dec_b: np.ndarray          # [r, W]   consumer decoder W_dec,B (Eq. 6, Eq. 9)
    sigma: np.ndarray            # [r]      singular values of the (centred) joint matrix
    mu_a: Optional[np.ndarray]   # [W] or None
    mu_b: Optional[np.ndarray]
    lam: float


def fit_reuse(a: np.ndarray, b: np.ndarray, r: int, lam_rel: float = 1e-3, center: bool = False) -> ReuseFit:
    """Steps 1-3 of the module docstring for one (layer, branch)."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    w = a.shape[1]
    mu_a = mu_b = None
    if center:
        mu_a, mu_b = a.mean(axis=0), b.mean(axis=0)
        a, b = a - mu_a, b - mu_b
    sigma, v = joint_svd(a, b, r)
    z = np.concatenate([a, b], axis=1) @ v                      # Z = X V_r = U_r S_r
    lam = ridge_lambda(a, lam_rel)
    w_enc = ridge(a, z, lam)
    return ReuseFit(w_enc, v[:w].T.copy(), v[w:].T.copy(), sigma, mu_a, mu_b, lam)


def invariants(fit: ReuseFit) -> Tuple[np.ndarray, np.ndarray]:
    """What is unique about a fit (U14): the projector V_r V_r^T [2W, 2W] and W_enc [W_dec,A W_dec,B] [W, 2W]."""
    vt = np.concatenate([fit.w_dec_a, fit.w_dec_b], axis=1)     # [r, 2W]
    return vt.T @ vt, fit.w_enc @ vt
