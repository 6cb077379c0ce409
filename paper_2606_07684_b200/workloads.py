"""Seeded synthetic workloads for the SCD codec (shared by tests, bench and smoke).

This module holds NONE of the method's arithmetic (no RoPE, no encode/decode/patch, no
packing): it only draws random tensors with the shapes, sizes and spectral structure of
the paper's workloads ("empirical low-rank structure of KV tensors",
:251-255 prefix lengths / model geometry) and fits the calibration-time artifacts the
codec is handed (a PCA basis via a library eigen-solver, random predictor weights).
The five configurations are the ones BASELINE.json names; the recipe is SURVEY.md §8(d)
and is restated in DESIGN.md ("Input recipe").

Everything is generated with torch on the device it is asked for, from `seed` and a
per-tensor sub-key, so that the CUDA path and the CPU oracle can be handed the same
bits (tests copy the tensors to the host for the oracle).
"""
from __future__ import annotations

import dataclasses
from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import torch

# enum values mirror include/scd.h (plain ints; no import of the binding on purpose)
F32, BF16, E4M3_ROWSCALE = 0, 1, 2
REUSE, PATCH = 0, 1


@dataclass(frozen=True)
class WorkloadConfig:
    name: str
    n_layers: int
    d_model: int
    n_kv_heads: int
    head_dim: int
    seqlens: Tuple[int, ...]              # explicit lengths, or () when ragged_range is set
    rank: int
    patch_layers: Tuple[int, ...]
    state_dtype: int
    code_dtype: int
    rope_theta: float
    spectrum_k: int                       # planted rank k
    spectrum_decay: float                 # s_i = decay^i
    noise_sigma: float                    # std of the iid noise
    ragged_range: Optional[Tuple[int, int, int]] = None   # (n_seqs, lo, hi): UniformInt[lo, hi]
    permute_pages: bool = False
    block_size: int = 16
    d_aligner: Optional[int] = None       # default d_model
    seed: int = 0
    rms_eps: float = 1e-5

    @property
    def D(self) -> int:
        return self.n_kv_heads * self.head_dim

    @property
    def d_a(self) -> int:
        return self.d_model if self.d_aligner is None else self.d_aligner

    def scaled(self, **kw) -> "WorkloadConfig":
        """A reduced copy (fewer layers / tokens / narrower model) for oracle-sized tests."""
        return dataclasses.replace(self, **kw)


# BASELINE.json `configs` [0..4]; * values are SURVEY §8(d) proposals where BASELINE is silent.
CONFIGS: Dict[str, WorkloadConfig] = {
    "tiny": WorkloadConfig("tiny", 4, 256, 4, 64, (512,), 32, (3,), F32, F32, 1e4, 48, 0.9, 0.01),
    "llama3_8b_8k": WorkloadConfig("llama3_8b_8k", 32, 4096, 8, 128, (8192,), 128, (8, 16, 24),
                                   BF16, BF16, 5e5, 256, 0.97, 0.01),
    "llama3_8b_ragged": WorkloadConfig("llama3_8b_ragged", 32, 4096, 8, 128, (), 64, (10, 21),
                                       BF16, BF16, 5e5, 256, 0.97, 0.01,
                                       ragged_range=(16, 256, 2048), permute_pages=True),
    "mistral_7b_32k_fp8": WorkloadConfig("mistral_7b_32k_fp8", 32, 4096, 8, 128, (32768,), 256,
                                         (4, 12, 20, 28), BF16, E4M3_ROWSCALE, 1e6, 512, 0.98, 0.02),
    "llama3_70b_2x16k": WorkloadConfig("llama3_70b_2x16k", 80, 8192, 8, 128, (16384, 16384), 128,
                                       tuple(range(0, 80, 10)), BF16, BF16, 5e5, 256, 0.97, 0.01),
}
CONFIG_ORDER = ["tiny", "llama3_8b_8k", "llama3_8b_ragged", "mistral_7b_32k_fp8", "llama3_70b_2x16k"]


def torch_state_dtype(cfg: WorkloadConfig) -> torch.dtype:
    return torch.float32 if cfg.state_dtype == F32 else torch.bfloat16


def _gen(cfg: WorkloadConfig, device, *key: int) -> torch.Generator:
    g = torch.Generator(device=device)
    s = cfg.seed
    for k in key:
        s = (s * 1000003 + 7919 * (k + 1)) % (2 ** 62)
    g.manual_seed(s)
    return g


# --------------------------------------------------------------------------------------
# batch geometry: lengths, page tables
# --------------------------------------------------------------------------------------
@dataclass
class BatchSpec:
    seqlens: List[int]
    cu_seqlens: torch.Tensor          # int32 [n_seqs + 1]   (device)
    page_table: torch.Tensor          # int32 [n_seqs, max_pages], unused = -1   (device)
    pos_offset: Optional[torch.Tensor]
    n_blocks: int
    max_pages: int

    @property
    def n_seqs(self) -> int:
        return len(self.seqlens)

    @property
    def total_tokens(self) -> int:
        return int(sum(self.seqlens))

    @property
    def max_seqlen(self) -> int:
        return max(self.seqlens) if self.seqlens else 0


def make_batch(cfg: WorkloadConfig, device="cpu", pos_offset: Optional[Sequence[int]] = None) -> BatchSpec:
    """Lengths (fixed or UniformInt[lo, hi]) and page tables over a shared block pool.
    Pool = sum(ceil(len/bs)) blocks + 10 % spare; with `permute_pages` the block ids are a
    random permutation dealt to requests (config 3), else identity order."""
    g = _gen(cfg, "cpu", 101)
    if cfg.ragged_range is not None:
        n, lo, hi = cfg.ragged_range
        seqlens = torch.randint(lo, hi + 1, (n,), generator=g).tolist()
    else:
        seqlens = list(cfg.seqlens)
    bs = cfg.block_size
    pages = [(l + bs - 1) // bs for l in seqlens]
    used = sum(pages)
    n_blocks = used + max(1, used // 10)
    ids = torch.randperm(n_blocks, generator=g) if cfg.permute_pages else torch.arange(n_blocks)
    max_pages = max(pages) if pages else 1
    table = torch.full((len(seqlens), max_pages), -1, dtype=torch.int32)
    at = 0
    for b, p in enumerate(pages):
        table[b, :p] = ids[at:at + p].to(torch.int32)
        at += p
    cu = torch.zeros(len(seqlens) + 1, dtype=torch.int32)
    if seqlens:
        cu[1:] = torch.cumsum(torch.tensor(seqlens, dtype=torch.int64), 0).to(torch.int32)
    po = None if pos_offset is None else torch.tensor(list(pos_offset), dtype=torch.int32, device=device)
    return BatchSpec(seqlens, cu.to(device), table.to(device), po, n_blocks, max_pages)


# --------------------------------------------------------------------------------------
# states: low-rank-plus-noise  X = (G diag(s)) Q^T + sigma E
# --------------------------------------------------------------------------------------
def planted_q(cfg: WorkloadConfig, layer: int, branch: int, width: int, device) -> torch.Tensor:
    """Q in R^{width x k}: Q-factor of a Gaussian matrix, diag(R) > 0."""
    k = min(cfg.spectrum_k, width)
    a = torch.randn(width, k, generator=_gen(cfg, device, layer, branch, 1), device=device,
                    dtype=torch.float32)
    q, r = torch.linalg.qr(a.double())
    return (q * torch.sign(torch.diagonal(r))[None, :]).float()


def make_state(cfg: WorkloadConfig, layer: int, branch: int, n_rows: int, device,
               row_offset: int = 0) -> torch.Tensor:
    """One [n_rows, width] state tensor in the state dtype (branch 0=K content-space keys,
    1=V, 2=H normalised hidden).  Rows are drawn in fixed 4096-row chunks keyed by the
    chunk index, so any row range of the same tensor can be regenerated."""
    width = cfg.d_model if branch == 2 else cfg.D
    q = planted_q(cfg, layer, branch, width, device)
    k = q.shape[1]
    s = cfg.spectrum_decay ** torch.arange(k, device=device, dtype=torch.float32)
    out = torch.empty(n_rows, width, device=device, dtype=torch_state_dtype(cfg))
    chunk = 4096
    first = row_offset // chunk
    last = (row_offset + n_rows - 1) // chunk if n_rows else first - 1
    for c in range(first, last + 1):
        gg = _gen(cfg, device, layer, branch, 2, c)
        g = torch.randn(chunk, k, generator=gg, device=device, dtype=torch.float32)
        e = torch.randn(chunk, width, generator=gg, device=device, dtype=torch.float32)
        x = (g * s[None, :]) @ q.t() + cfg.noise_sigma * e
        lo = max(row_offset, c * chunk)
        hi = min(row_offset + n_rows, (c + 1) * chunk)
        out[lo - row_offset:hi - row_offset] = x[lo - c * chunk:hi - c * chunk].to(out.dtype)
    return out


def fit_basis(x_cal: torch.Tensor, r: int) -> Tuple[torch.Tensor, torch.Tensor]:
    """Calibration fit (offline): mu = column mean, B = top-r right
    singular vectors of X_cal - mu, from the eigen-decomposition of the Gram matrix in
    fp64.  Returns (B [r, width] fp64 with orthonormal rows, mu [width] fp64)."""
    x = x_cal.double()
    mu = x.mean(dim=0)
    xc = x - mu[None, :]
    gram = xc.t() @ xc
    w, v = torch.linalg.eigh(gram)                      # ascending
    b = v[:, -r:].flip(1).t().contiguous()              # [r, width], descending eigenvalue
    return b, mu


@dataclass
class LayerArtifacts:
    """Device tensors handed to scd_plan for one layer (state dtype unless noted)."""
    kind: int
    enc_k: Optional[torch.Tensor] = None      # [D, r]
    enc_v: Optional[torch.Tensor] = None
    dec_k: Optional[torch.Tensor] = None      # [r, D]
    dec_v: Optional[torch.Tensor] = None
    mean_k: Optional[torch.Tensor] = None     # [D] fp32 (src = dst)
    mean_v: Optional[torch.Tensor] = None
    mean_dst_k: Optional[torch.Tensor] = None # [D] fp32 consumer-side mean when it differs from the producer's (fitted pairs)
    mean_dst_v: Optional[torch.Tensor] = None
    enc_h: Optional[torch.Tensor] = None      # [d, r]
    mean_h: Optional[torch.Tensor] = None     # [d] fp32
    w1: Optional[torch.Tensor] = None         # [r, d_a]
    b1: Optional[torch.Tensor] = None         # [d_a]
    w2: Optional[torch.Tensor] = None         # [d_a, d]
    b2: Optional[torch.Tensor] = None
    gamma: Optional[torch.Tensor] = None      # [d]
    w_k: Optional[torch.Tensor] = None        # [D, d]
    w_v: Optional[torch.Tensor] = None
    b_k: Optional[torch.Tensor] = None
    b_v: Optional[torch.Tensor] = None

    def to(self, device) -> "LayerArtifacts":
        """The same artifacts on another device (e.g. drawn on the CPU, used on the GPU)."""
        return LayerArtifacts(**{f.name: (v.to(device) if isinstance(v, torch.Tensor) else v)
                                 for f in dataclasses.fields(self) for v in (getattr(self, f.name),)})


def make_layer_artifacts(cfg: WorkloadConfig, layer: int, device, cal_rows: int = 8192,
                         total_rows: Optional[int] = None, per_head_rank: int = 0) -> LayerArtifacts:
    """Artifacts of one layer.  REUSE: one orthonormal-row PCA basis per branch, W_dec = B,
    W_enc = B^T, mu_src = mu_dst = calibration mean.  PATCH: W1 = B_H and
    b1 = mu_H (d_a = d_model) or Gaussian W1/b1 when d_a != d_model; W2, W_k, W_v ~
    N(0, 1/fan_in); gamma = 1 + 0.1 N(0,1); no b2 / b_k / b_v.
    `per_head_rank` > 0: the paper's per-head reading for REUSE layers: the calibration rows are
    flattened to [rows * H, d_h] and ONE basis [r, d_h] / mean [d_h] is fitted for all heads."""
    sd = torch_state_dtype(cfg)
    n_cal = cal_rows if total_rows is None else min(cal_rows, total_rows)
    if layer not in cfg.patch_layers:
        art = LayerArtifacts(REUSE)
        for branch, name in ((0, "k"), (1, "v")):
            x_cal = make_state(cfg, layer, branch, n_cal, device)
            if per_head_rank:
                b, mu = fit_basis(x_cal.reshape(-1, cfg.head_dim), per_head_rank)
            else:
                b, mu = fit_basis(x_cal, cfg.rank)
            setattr(art, f"dec_{name}", b.to(sd).contiguous())
            setattr(art, f"enc_{name}", b.t().to(sd).contiguous())
            setattr(art, f"mean_{name}", mu.float().contiguous())
        return art
    art = LayerArtifacts(PATCH)
    d, d_a, D = cfg.d_model, cfg.d_a, cfg.D
    b, mu = fit_basis(make_state(cfg, layer, 2, n_cal, device), cfg.rank)
    art.enc_h = b.t().to(sd).contiguous()
    art.mean_h = mu.float().contiguous()
    g = _gen(cfg, device, layer, 7)
    rn = lambda *shape: torch.randn(*shape, generator=g, device=device, dtype=torch.float32)
    if d_a == d:
        art.w1 = b.to(sd).contiguous()
        art.b1 = mu.to(sd).contiguous()
    else:
        art.w1 = (rn(cfg.rank, d_a) / cfg.rank ** 0.5).to(sd)
        art.b1 = (0.1 * rn(d_a)).to(sd)
    art.w2 = (rn(d_a, d) / d_a ** 0.5).to(sd)
    art.gamma = (1.0 + 0.1 * rn(d)).to(sd)
    art.w_k = (rn(D, d) / d ** 0.5).to(sd)
    art.w_v = (rn(D, d) / d ** 0.5).to(sd)
    return art


def make_sentinel_pool(cfg: WorkloadConfig, n_blocks: int, device) -> torch.Tensor:
    """A pool [n_blocks, bs, H_kv, d_h] filled with a recognisable bit pattern (bf16
    0x7FC1 / fp32 0x7FC00001: quiet NaNs no computation produces)."""
    shape = (n_blocks, cfg.block_size, cfg.n_kv_heads, cfg.head_dim)
    if cfg.state_dtype == F32:
        return torch.full(shape, 0x7FC00001, dtype=torch.int32, device=device).view(torch.float32)
    return torch.full(shape, 0x7FC1, dtype=torch.int16, device=device).view(torch.bfloat16)
