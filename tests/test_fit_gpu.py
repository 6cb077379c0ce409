"""GPU parity of scd_fit_reuse (stack-SVD + ridge on the GPU) against oracle/fit_oracle.py.

Several results are correct (a singular direction's sign is arbitrary), so what is compared is what is
unique: the singular values, the projector V_r V_r^T and the sign-free product W_enc [W_dec,A W_dec,B].

Tolerances: the GPU forms G = X^T X from exact bf16 x bf16 products accumulated in
fp32 by the tensor core over chunks of n_c = 4096 samples (then fp64).  Each of the n_c additions rounds by at most
2^-24 of the running sum; the roundings are modelled as independent (random walk), with a factor 4 for safety:
|E_ij| <= eps_G sum_n |x_ni| |x_nj|, eps_G = 4 sqrt(n_c) 2^-24 = 1.5e-5 (the worst case, every rounding in the same
direction, would be n_c 2^-24 = 2.4e-4 and makes the bounds below vacuous).  Then (Weyl) |d lambda_k| <= ||E||_2 and
(Davis-Kahan) ||d P||_F <= 2 sqrt(2) ||E||_F / gap_r.  The test evaluates both bounds from the inputs and prints
how much of them was used.
"""
import numpy as np
import pytest
import torch

from oracle import fit_oracle as F
from oracle import scd_oracle as O
from paper_2606_07684_b200 import workloads as W
from tests import _parity as P

pytestmark = pytest.mark.gpu

EPS_G = 4 * 4096 ** 0.5 * 2.0 ** -24


def _pair(n, w, k, decay, noise, seed, offset=0.0):
    """Paired producer / consumer samples with a planted joint subspace of rank k: X = (G diag(s)) Q^T + noise."""
    g = torch.Generator().manual_seed(seed)
    q, _ = torch.linalg.qr(torch.randn(2 * w, k, generator=g, dtype=torch.float64))
    s = decay ** torch.arange(k, dtype=torch.float64)
    x = (torch.randn(n, k, generator=g, dtype=torch.float64) * s) @ q.t() * (2 * w) ** 0.5
    x = x + noise * torch.randn(n, 2 * w, generator=g, dtype=torch.float64) + offset
    a, b = x[:, :w].to(torch.bfloat16).contiguous(), x[:, w:].to(torch.bfloat16).contiguous()
    return a, b


def _gpu_fit(a, b, r, center, lam_rel, device, out_dtype=None):
    from paper_2606_07684_b200 import binding as B
    n, w = a.shape
    od = B.SCD_F32 if out_dtype is None else out_dtype
    td = torch.float32 if od == B.SCD_F32 else torch.bfloat16
    desc = B.FitDesc(w, r, int(center), lam_rel, B.SCD_BF16, od)
    ws = torch.empty(B.scd_fit_query(desc, n), dtype=torch.uint8, device=device)
    out = dict(w_enc=torch.zeros(w, r, dtype=td, device=device), w_dec_a=torch.zeros(r, w, dtype=td, device=device),
               w_dec_b=torch.zeros(r, w, dtype=td, device=device), mu_a=torch.zeros(w, device=device),
               mu_b=torch.zeros(w, device=device), sigma=torch.zeros(r, device=device))
    sweeps = B.scd_fit_reuse(desc, a.to(device), b.to(device), n, w, out["w_enc"], out["w_dec_a"], out["w_dec_b"],
                             out["mu_a"] if center else None, out["mu_b"] if center else None, out["sigma"], ws)
    torch.cuda.synchronize()
    return out, sweeps


def _check(a, b, r, center, lam_rel, device):
    out, sweeps = _gpu_fit(a, b, r, center, lam_rel, device)
    a64, b64 = a.double().numpy(), b.double().numpy()
    ref = F.fit_reuse(a64, b64, r, lam_rel=lam_rel, center=center)
    got = F.ReuseFit(out["w_enc"].double().cpu().numpy(), out["w_dec_a"].double().cpu().numpy(),
                     out["w_dec_b"].double().cpu().numpy(), out["sigma"].double().cpu().numpy(), None, None, ref.lam)
    x = np.concatenate([a64, b64], axis=1)
    if center:
        np.testing.assert_allclose(out["mu_a"].double().cpu().numpy(), ref.mu_a, rtol=1e-6, atol=1e-7)
        np.testing.assert_allclose(out["mu_b"].double().cpu().numpy(), ref.mu_b, rtol=1e-6, atol=1e-7)
        x = x - x.mean(axis=0)
    # error model of the Gram matrix
    ax = np.abs(np.concatenate([a64, b64], axis=1))
    e_fro = EPS_G * np.linalg.norm(ax.T @ ax)
    s_all = np.linalg.svd(x, compute_uv=False)
    lam = s_all ** 2
    gap = lam[r - 1] - lam[r]
    # singular values: |d lambda| <= ||E||_2 <= ||E||_F  ->  |d sigma| <= ||E|| / (2 sigma) (+ fp32 storage)
    d_sigma = np.abs(got.sigma - ref.sigma)
    bound_sigma = e_fro / (2 * ref.sigma) + 2.0 ** -23 * ref.sigma
    assert np.all(d_sigma <= bound_sigma), (d_sigma / bound_sigma).max()
    p_got, m_got = F.invariants(got)
    p_ref, m_ref = F.invariants(ref)
    d_p = np.linalg.norm(p_got - p_ref)
    bound_p = 2 * np.sqrt(2) * e_fro / gap + 1e-5          # + fp32 storage of the basis entries
    assert d_p <= bound_p, (d_p, bound_p)
    # rows of W_dec orthonormal (fp32 storage)
    vt = np.concatenate([got.w_dec_a, got.w_dec_b], axis=1)
    np.testing.assert_allclose(vt @ vt.T, np.eye(r), atol=5e-6)
    # encoder.  Coefficients of a ridge fit are ill-conditioned in directions where A has no energy (condition number
    # up to lambda_max / lam), its PREDICTIONS are not (the hat matrix has norm <= 1): compare A W_enc W_dec, the
    # reconstruction the codec actually produces from producer states, and report the coefficient error beside it.
    a_c = x[:, :a64.shape[1]]
    pred_got, pred_ref = a_c @ m_got, a_c @ m_ref
    rel_m = np.linalg.norm(pred_got - pred_ref) / np.linalg.norm(pred_ref)
    bound_m = 2 * bound_p + 1e-5
    assert rel_m <= bound_m, (rel_m, bound_m)
    coef_rel = np.linalg.norm(m_got - m_ref) / np.linalg.norm(m_ref)
    assert coef_rel <= 1e-2, coef_rel
    return {"sweeps": sweeps, "sigma_used": float((d_sigma / bound_sigma).max()), "proj_err": float(d_p),
            "proj_bound": float(bound_p), "enc_pred_rel": float(rel_m), "enc_bound": float(bound_m), "enc_coef_rel": float(coef_rel)}


@pytest.mark.parametrize("w,r,center", [(128, 32, False), (128, 32, True), (64, 16, True), (256, 64, True)])
def test_fit_matches_oracle(w, r, center, cuda_device):
    # planted rank = r: a clear gap between sigma_r and the noise floor
    a, b = _pair(3001, w, r, 0.93, 0.02, seed=w + r, offset=0.5 if center else 0.0)
    print(_check(a, b, r, center, 1e-3, cuda_device))


def test_fit_inside_a_decaying_spectrum(cuda_device):
    """r cuts a geometric spectrum (0.9^i): the gap is 19 % of lambda_r."""
    a, b = _pair(5000, 128, 48, 0.9, 0.01, seed=5)
    print(_check(a, b, 24, True, 1e-3, cuda_device))


@pytest.mark.slow
def test_fit_llama_width(cuda_device):
    """Per-layer width D = 1024 (n = 2048: the largest eigen-problem), r = 128 as in BASELINE config 2."""
    a, b = _pair(4100, 1024, 128, 0.97, 0.01, seed=11)
    print(_check(a, b, 128, True, 1e-3, cuda_device))


def test_fitted_pair_through_the_codec(cuda_device):
    """W_enc from the ridge fit is NOT W_dec^T, producer and consumer means differ.  One BASELINE-shaped
    REUSE problem (Llama geometry, r = 128) runs encode -> reuse_decode with artifacts fitted ON THE GPU from paired
    producer / consumer samples, and is checked against the oracle given the same artifact bits; end to end the decoded
    V must approximate the CONSUMER's states (Eq. 6, 9) to the truncation error."""
    from paper_2606_07684_b200 import binding as B
    from paper_2606_07684_b200.harness import CodecProblem
    cfg = W.CONFIGS["llama3_8b_8k"].scaled(n_layers=2, patch_layers=(), seqlens=(700,))
    D, r, T = cfg.D, cfg.rank, 700
    arts, prod, cons = [], [], []
    for l in range(cfg.n_layers):
        art = W.LayerArtifacts(W.REUSE)
        for br, name in ((0, "k"), (1, "v")):
            a, b = _pair(4096, D, r, 0.97, 0.01, seed=100 + 2 * l + br, offset=0.25)
            out, _ = _gpu_fit(a, b, r, True, 1e-3, cuda_device, out_dtype=B.SCD_BF16)
            setattr(art, f"enc_{name}", out["w_enc"])
            setattr(art, f"dec_{name}", out["w_dec_b"])
            setattr(art, f"mean_{name}", out["mu_a"])
            setattr(art, f"mean_dst_{name}", out["mu_b"])
            if br == 1:
                prod.append(a[:T].to(cuda_device))
                cons.append(b[:T].double().numpy())
            else:
                k_src = a[:T].to(cuda_device)
        assert not torch.equal(art.enc_v.t().contiguous(), art.dec_v)
        arts.append((art, k_src))
    prob = CodecProblem(cfg, cuda_device, artifacts=[a for a, _ in arts], k_is_roped=False, rope_on_reuse_k=False)
    k = [ks for _, ks in arts]                       # [T, D] = [T, H_kv, d_h] dense
    v = list(prod)
    h = [None] * cfg.n_layers
    prob.alloc_pools()
    prob.encode(k, v, h)
    prob.reuse_decode()
    torch.cuda.synchronize()
    P.check_encode(prob, k, v, h)
    P.check_reuse_decode(prob)
    slots = O.slot_mapping(P.oracle_batch(prob), cfg.block_size)
    for l in range(cfg.n_layers):
        got = prob.v_pool[l].view(-1, D)[torch.from_numpy(slots).to(cuda_device)].double().cpu().numpy()
        rel = np.linalg.norm(got - cons[l]) / np.linalg.norm(cons[l] - cons[l].mean(axis=0))
        assert rel < 0.1, rel            # noise floor 0.01 * sqrt(2W) against a planted signal of rank r


def test_fitted_per_head_translators_through_the_codec(cuda_device):
    """The paper-literal reading: heads flattened into the sample axis, ONE d_h x r translator per
    layer and branch.  Fitted on the GPU with width = head_dim from [T * H, d_h] paired samples, then run through the
    per-head mode of the codec (reuse_per_head) and checked against the oracle on the same artifact bits."""
    from paper_2606_07684_b200 import binding as B
    from paper_2606_07684_b200.harness import CodecProblem
    cfg = W.CONFIGS["llama3_8b_8k"].scaled(n_layers=1, patch_layers=(), seqlens=(333,))
    H, dh, T, r = cfg.n_kv_heads, cfg.head_dim, 333, 32
    art = W.LayerArtifacts(W.REUSE)
    src = {}
    for br, name in ((0, "k"), (1, "v")):
        a, b = _pair(T * H, dh, r, 0.9, 0.02, seed=300 + br, offset=0.1)
        out, sweeps = _gpu_fit(a, b, r, True, 1e-3, cuda_device, out_dtype=B.SCD_BF16)
        assert max(sweeps) < 60
        setattr(art, f"enc_{name}", out["w_enc"])
        setattr(art, f"dec_{name}", out["w_dec_b"])
        setattr(art, f"mean_{name}", out["mu_a"])
        setattr(art, f"mean_dst_{name}", out["mu_b"])
        src[name] = a.reshape(T, H * dh).to(cuda_device)
    prob = CodecProblem(cfg, cuda_device, artifacts=[art], per_head_rank=r, k_is_roped=False, rope_on_reuse_k=False)
    prob.alloc_pools()
    prob.encode([src["k"]], [src["v"]], [None])
    prob.reuse_decode()
    torch.cuda.synchronize()
    P.check_encode(prob, [src["k"]], [src["v"]], [None])
    P.check_reuse_decode(prob)


def test_fit_error_paths(cuda_device):
    from paper_2606_07684_b200 import binding as B
    ws = torch.empty(1 << 20, dtype=torch.uint8, device=cuda_device)
    x = torch.zeros(64, 64, dtype=torch.bfloat16, device=cuda_device)
    o = torch.zeros(64, 64, dtype=torch.float32, device=cuda_device)
    for desc, status in ((B.FitDesc(60, 8, 0, 1e-3, B.SCD_BF16, B.SCD_F32), 2),      # width not a multiple of 8
                         (B.FitDesc(2048, 8, 0, 1e-3, B.SCD_BF16, B.SCD_F32), 3),    # wider than the eigen-solver takes
                         (B.FitDesc(64, 200, 0, 1e-3, B.SCD_BF16, B.SCD_F32), 2),    # rank > 2 W
                         (B.FitDesc(64, 8, 0, 1e-3, B.SCD_F32, B.SCD_F32), 3),       # fp32 states
                         (B.FitDesc(64, 8, 0, -1.0, B.SCD_BF16, B.SCD_F32), 1)):     # negative ridge
        with pytest.raises(B.ScdError) as e:
            B.scd_fit_query(desc, 64)
        assert e.value.status == status
    desc = B.FitDesc(64, 8, 1, 1e-3, B.SCD_BF16, B.SCD_F32)
    with pytest.raises(B.ScdError) as e:                                             # centring without mean outputs
        B.scd_fit_reuse(desc, x, x, 64, 64, o, None, o, None, None, None, ws)
    assert e.value.status == 1
    with pytest.raises(B.ScdError) as e:                                             # workspace too small
        B.scd_fit_reuse(B.FitDesc(64, 8, 0, 1e-3, B.SCD_BF16, B.SCD_F32), x, x, 64, 64, o, None, o, None, None, None, ws[:1024])
    assert e.value.status == 5
