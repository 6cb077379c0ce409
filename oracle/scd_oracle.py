"""CPU oracle for the SCD KV state codec (arxiv/paper_2606_07684).

TEST INFRASTRUCTURE ONLY.  This module is the plain, slow, fp64 definition of what
`scd_encode`, `scd_reuse_decode`, `scd_patch` and `scd_plan` compute.  It shares no
code with the CUDA path (`paper_2606_07684_b200/`), imports nothing from it, and may be
imported only by `tests/`, `__graft_entry__.smoke()` and `bench.py`'s CPU-baseline
legs.  Every function cites the passage of `/root/reference/PAPER.md` it restates
(`PAPER.md:<line>`, section / equation) or, for build extensions the paper does not
have, the SURVEY.md §8(c) reading (U-number) it follows.

Conventions
-----------
* All arithmetic is numpy float64; a matmul is `a @ b` (library primitive used as one
  step, no blocking / fusion / reordering).
* Inputs stored in a narrower type (bf16 / fp32 / e4m3 bits) are widened exactly by
  the caller or by `unpack_codes`; outputs stay fp64.
* Rows are packed: request b owns rows cu_seqlens[b] .. cu_seqlens[b+1]-1; token t of
  request b has position id pos_offset[b] + t  ("cache_position").
* Layer indices are 0-based.

Parity pins: every function below is pinned by tests/test_oracle_*.py (closed forms,
invariants, independent library routines, brute force).  Nothing here is "parity
unpinned".
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

# --------------------------------------------------------------------------------------
# enums (plain ints so the oracle depends on nothing)
# --------------------------------------------------------------------------------------
F32, BF16, E4M3_ROWSCALE = 0, 1, 2          # code / state dtypes
REUSE, PATCH = 0, 1                         # layer kinds  (L_reuse / L_patch)
ROPE_HALF, ROPE_INTERLEAVED = 0, 1          # pairing convention
ACT_IDENTITY, ACT_SILU = 0, 1               # aligner non-linearity
NORM_NONE, NORM_RMS = 0, 1                  # NORM_NONE = paper-literal Eq. 11-12
BRANCH_K, BRANCH_V, BRANCH_H = 0, 1, 2


# --------------------------------------------------------------------------------------
# descriptors
# --------------------------------------------------------------------------------------
@dataclass
class Model:
    """Model-pair geometry: producer and consumer share the architecture."""
    n_layers: int
    d_model: int
    n_kv_heads: int
    head_dim: int
    block_size: int = 16
    rope_theta_producer: float = 10000.0
    rope_theta_consumer: float = 10000.0
    rope_style: int = ROPE_HALF
    k_is_roped: bool = True          # producer K arrives post-RoPE -> deRoPE first (Eq. 5)
    rope_on_reuse_k: bool = True     # re-apply RoPE after decode
    code_dtype: int = F32
    patch_act: int = ACT_SILU
    patch_norm: int = NORM_RMS
    rms_eps: float = 1e-5
    # Paper-literal REUSE translator: batch x heads x tokens are flattened into
    # one sample axis and ONE map W_enc in R^{d_h x r} / W_dec in R^{r x d_h} serves every head of the layer.
    # Codes of a token are the heads' codes side by side, [H * r].  False = per-layer basis over D.
    reuse_per_head: bool = False

    @property
    def D(self) -> int:
        return self.n_kv_heads * self.head_dim


@dataclass
class Layer:
    """Per-layer artifacts.  All arrays fp64 (already widened)."""
    kind: int
    # REUSE (Eq. 6-9): enc [D, r], dec [r, D], optional means [D] (None = 0)
    enc_k: Optional[np.ndarray] = None
    enc_v: Optional[np.ndarray] = None
    dec_k: Optional[np.ndarray] = None
    dec_v: Optional[np.ndarray] = None
    mean_src_k: Optional[np.ndarray] = None
    mean_src_v: Optional[np.ndarray] = None
    mean_dst_k: Optional[np.ndarray] = None
    mean_dst_v: Optional[np.ndarray] = None
    # PATCH (Eq. 10-12): enc_h [d, r_h]; aligner w1 [r_h, d_a], b1 [d_a], w2 [d_a, d], b2 [d]
    enc_h: Optional[np.ndarray] = None
    mean_src_h: Optional[np.ndarray] = None
    w1: Optional[np.ndarray] = None
    b1: Optional[np.ndarray] = None
    w2: Optional[np.ndarray] = None
    b2: Optional[np.ndarray] = None
    norm_gamma: Optional[np.ndarray] = None      # [d] consumer RMSNorm weight (NORM_RMS)
    w_k: Optional[np.ndarray] = None             # [D, d]  HF layout [out, in]
    w_v: Optional[np.ndarray] = None
    b_k: Optional[np.ndarray] = None
    b_v: Optional[np.ndarray] = None


@dataclass
class Batch:
    """Ragged batch + page tables."""
    cu_seqlens: np.ndarray                       # int [n_seqs + 1]
    page_table: np.ndarray                       # int [n_seqs, max_pages], unused = -1
    pos_offset: Optional[np.ndarray] = None      # int [n_seqs] or None (= 0)

    @property
    def n_seqs(self) -> int:
        return len(self.cu_seqlens) - 1

    @property
    def total_tokens(self) -> int:
        return int(self.cu_seqlens[-1])


# --------------------------------------------------------------------------------------
# a1 / A14 / D4: plan = static routing table + payload accounting
# --------------------------------------------------------------------------------------
def route(layers: Sequence[Layer]) -> Tuple[List[int], List[int]]:
    """(L_reuse, L_patch): fixed sets, membership by layer index."""
    l_reuse = [i for i, l in enumerate(layers) if l.kind == REUSE]
    l_patch = [i for i, l in enumerate(layers) if l.kind == PATCH]
    return l_reuse, l_patch


def code_elem_bytes(code_dtype: int) -> int:
    return {F32: 4, BF16: 2, E4M3_ROWSCALE: 1}[code_dtype]


def payload_bytes(model: Model, layers: Sequence[Layer], total_tokens: int) -> int:
    """|Z| of Eq. 3: {Z_K, Z_V} for reuse layers, {Z_H} for patch layers
    (Alg. 1 :180); e4m3 adds one fp32 scale per (segment, token) (U11)."""
    cb = code_elem_bytes(model.code_dtype)
    sb = 4 if model.code_dtype == E4M3_ROWSCALE else 0
    n = 0
    for l in layers:
        if l.kind == REUSE:
            hm = model.n_kv_heads if model.reuse_per_head else 1      # per-head: r codes per head
            n += total_tokens * (hm * l.enc_k.shape[1] * cb + sb)
            n += total_tokens * (hm * l.enc_v.shape[1] * cb + sb)
        else:
            n += total_tokens * (l.enc_h.shape[1] * cb + sb)
    return n


# --------------------------------------------------------------------------------------
# positions and paging (a8)
# --------------------------------------------------------------------------------------
def positions(batch: Batch) -> np.ndarray:
    """Position id of every packed row: p = pos_offset[b] + t."""
    pos = np.zeros(batch.total_tokens, dtype=np.int64)
    for b in range(batch.n_seqs):
        s, e = int(batch.cu_seqlens[b]), int(batch.cu_seqlens[b + 1])
        off = 0 if batch.pos_offset is None else int(batch.pos_offset[b])
        pos[s:e] = off + np.arange(e - s)
    return pos


def slot_mapping(batch: Batch, block_size: int) -> np.ndarray:
    """slot(b, t) = page_table[b][t // bs] * bs + t % bs for every packed row."""
    slots = np.zeros(batch.total_tokens, dtype=np.int64)
    for b in range(batch.n_seqs):
        s, e = int(batch.cu_seqlens[b]), int(batch.cu_seqlens[b + 1])
        t = np.arange(e - s)
        slots[s:e] = batch.page_table[b][t // block_size].astype(np.int64) * block_size + t % block_size
    return slots


def read_paged(pool: np.ndarray, slots: np.ndarray) -> np.ndarray:
    """Packed rows of a batch read back from a paged pool [n_blocks, bs, H_kv, d_h] (or [n_slots, D]): row n of the
    batch is the pool row at slots[n].  The producer's cache may be paged too ("native cache semantics",
    PAPER.md:610): encode then reads K_A / V_A through the producer's own page table."""
    flat = pool.reshape(-1, pool.shape[-2] * pool.shape[-1]) if pool.ndim == 4 else pool
    return flat[np.asarray(slots, dtype=np.int64)]


def write_paged(pool: np.ndarray, slots: np.ndarray, rows: np.ndarray) -> None:
    """Pool element (slot, head, c) lives at ((slot*H_kv)+head)*d_h + c, i.e. the pool
    viewed as [n_blocks*bs, D] takes row `rows[n]` at index slots[n]."""
    flat = pool.reshape(-1, rows.shape[1])
    flat[slots] = rows


# --------------------------------------------------------------------------------------
# A5: RoPE / deRoPE (Eq. 5, re-apply)
# --------------------------------------------------------------------------------------
def rope(x: np.ndarray, pos: np.ndarray, theta: float, sign: int,
         n_heads: int, head_dim: int, style: int = ROPE_HALF) -> np.ndarray:
    """Rotate every head of every row by its position.  sign=+1 RoPE, -1 deRoPE.

    phi_j = sign * p * theta^(-2j/d_h), j in [0, d_h/2).
    HALF pairs (x_j, x_{j+d_h/2}); INTERLEAVED pairs (x_{2j}, x_{2j+1}):
      x'_a = x_a cos(phi) - x_b sin(phi);  x'_b = x_b cos(phi) + x_a sin(phi).
    """
    T = x.shape[0]
    half = head_dim // 2
    xh = np.asarray(x, dtype=np.float64).reshape(T, n_heads, head_dim)
    j = np.arange(half, dtype=np.float64)
    inv_freq = np.float64(theta) ** (-2.0 * j / head_dim)
    phi = sign * np.asarray(pos, dtype=np.float64)[:, None] * inv_freq[None, :]   # [T, half]
    c, s = np.cos(phi)[:, None, :], np.sin(phi)[:, None, :]
    out = np.empty_like(xh)
    if style == ROPE_HALF:
        a, b = xh[..., :half], xh[..., half:]
        out[..., :half] = a * c - b * s
        out[..., half:] = b * c + a * s
    else:
        a, b = xh[..., 0::2], xh[..., 1::2]
        out[..., 0::2] = a * c - b * s
        out[..., 1::2] = b * c + a * s
    return out.reshape(T, n_heads * head_dim)


# --------------------------------------------------------------------------------------
# a5 / D1: code packing
# --------------------------------------------------------------------------------------
def round_to_bf16(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp64 -> bf16, returned as fp64 values that bf16 holds
    exactly.  bf16 = sign, 8 exponent bits, 7 fraction bits: ulp(x) = 2^(e-7) for
    2^e <= |x| < 2^(e+1) (normal range).  Inputs are assumed finite and within the bf16
    normal range (true for every tensor on this path)."""
    x = np.asarray(x, dtype=np.float64)
    out = np.zeros_like(x)
    nz = x != 0
    m, e = np.frexp(x[nz])                  # x = m * 2^e, 0.5 <= |m| < 1
    # 8 significant bits: scale mantissa to [128, 256), rint is ties-to-even
    out[nz] = np.ldexp(np.rint(m * 256.0), e - 8)
    return out


def _e4m3_values() -> np.ndarray:
    """All 256 byte codes of OCP e4m3fn -> value (NaN for 0x7F / 0xFF).
    1 sign, 4 exponent (bias 7), 3 mantissa; exponent 0 = subnormal m/8 * 2^-6;
    no infinities; S.1111.111 = NaN; max finite = 1.75 * 2^8 = 448."""
    v = np.zeros(256, dtype=np.float64)
    for b in range(256):
        s = -1.0 if b & 0x80 else 1.0
        e = (b >> 3) & 0xF
        m = b & 0x7
        if e == 0xF and m == 0x7:
            v[b] = np.nan
        elif e == 0:
            v[b] = s * (m / 8.0) * 2.0 ** (-6)
        else:
            v[b] = s * (1.0 + m / 8.0) * 2.0 ** (e - 7)
    return v


E4M3_VALUES = _e4m3_values()
E4M3_MAX = 448.0


def e4m3_quantize(x: np.ndarray) -> np.ndarray:
    """fp64 -> e4m3fn byte, round-to-nearest-even, saturating to +-448.
    Written as the definition: pick the nearest representable magnitude; on a tie pick
    the one whose byte code is even (even mantissa LSB)."""
    x = np.asarray(x, dtype=np.float64)
    mags = E4M3_VALUES[:0x7F]                         # 0x00..0x7E: ascending non-negative
    a = np.minimum(np.abs(x), E4M3_MAX)
    hi = np.searchsorted(mags, a, side="left")        # first code with value >= a
    hi = np.minimum(hi, 0x7E)
    lo = np.maximum(hi - 1, 0)
    d_lo, d_hi = a - mags[lo], mags[hi] - a
    pick_hi = (d_hi < d_lo) | ((d_hi == d_lo) & (hi % 2 == 0))
    code = np.where(pick_hi, hi, lo).astype(np.uint8)
    return np.where(np.signbit(x), code | 0x80, code).astype(np.uint8)


def pack_codes(z: np.ndarray, code_dtype: int) -> Tuple[np.ndarray, Optional[np.ndarray]]:
    """fp64 codes [T, r] -> (stored codes, per-row scales or None).
    F32: (float) z.  BF16: RNE(z).  E4M3_ROWSCALE: s = max_i |z_i| / 448 rounded to fp32
    (s = 1 for an all-zero row), q_i = e4m3(z_i / s)."""
    if code_dtype == F32:
        return z.astype(np.float32), None
    if code_dtype == BF16:
        return round_to_bf16(z), None
    amax = np.max(np.abs(z), axis=1)
    s = np.where(amax > 0, amax / E4M3_MAX, 1.0).astype(np.float32)
    q = e4m3_quantize(z / s.astype(np.float64)[:, None])
    return q, s


def quantize_pool(y: np.ndarray, n_heads: int) -> Tuple[np.ndarray, np.ndarray]:
    """fp8 K/V pools (build extension, DESIGN.md section 2 U20).  y [T, D] = the K or V rows the
    consumer stores (fp64).  Per (token, head): x = bf16(y) (the value a bf16 pool would hold), s = amax / 448 in fp32
    (1 for an all-zero head), byte = e4m3_rne_sat(x * (1 / s)) with 1 / s and the product rounded to fp32 -- the
    decision is taken in the kernel's precision.  Returns (bytes [T, D] uint8, scales [T, n_heads] fp32)."""
    T, D = y.shape
    x = round_to_bf16(y).astype(np.float32).reshape(T, n_heads, D // n_heads)
    amax = np.max(np.abs(x), axis=2)
    s = np.where(amax > 0, (amax / np.float32(E4M3_MAX)).astype(np.float32), np.float32(1.0)).astype(np.float32)
    inv = (np.float32(1.0) / s).astype(np.float32)
    t = (x * inv[:, :, None]).astype(np.float32)
    return e4m3_quantize(t.astype(np.float64)).reshape(T, D), s


def dequantize_pool(q: np.ndarray, s: np.ndarray) -> np.ndarray:
    """bytes [T, D], scales [T, H] -> fp64 values (exact): s * value(byte)."""
    T, D = q.shape
    H = s.shape[1]
    return (E4M3_VALUES[q].reshape(T, H, D // H) * s.astype(np.float64)[:, :, None]).reshape(T, D)


def unpack_codes(q: np.ndarray, scale: Optional[np.ndarray], code_dtype: int) -> np.ndarray:
    """Stored codes -> fp64 (exact).  e4m3: s * value(q)."""
    if code_dtype == E4M3_ROWSCALE:
        return E4M3_VALUES[q] * scale.astype(np.float64)[:, None]
    return np.asarray(q, dtype=np.float64)


# --------------------------------------------------------------------------------------
# a2-a4 / A8, A10: producer encode  (Eq. 8, H branch PAPER.md:165)
# --------------------------------------------------------------------------------------
def _sub(x: np.ndarray, mu: Optional[np.ndarray]) -> np.ndarray:
    return x if mu is None else x - mu[None, :]


def _add(x: np.ndarray, mu: Optional[np.ndarray]) -> np.ndarray:
    return x if mu is None else x + mu[None, :]


def _translate(model: Model, x: np.ndarray, mu: Optional[np.ndarray], w: np.ndarray, mu_after: bool) -> np.ndarray:
    """One linear REUSE map on rows of x.  Per-layer reading: x [T, in] (in = D or r).  Per-head reading
    (model.reuse_per_head): every head of every token is a sample, w is [d_h, r] or [r, d_h], mu is [d_h];
    the result is laid out per token again, heads side by side."""
    if not model.reuse_per_head:
        return _add(x @ w, mu) if mu_after else _sub(x, mu) @ w
    t = x.shape[0]
    xs = x.reshape(t * model.n_kv_heads, w.shape[0])
    ys = _add(xs @ w, mu) if mu_after else _sub(xs, mu) @ w
    return ys.reshape(t, model.n_kv_heads * w.shape[1])


def encode_k(model: Model, layer: Layer, k_a: np.ndarray, pos: np.ndarray) -> np.ndarray:
    """Z_K = (deRoPE(K_A) - mu_src,K) W_enc,K   (Eq. 5, Eq. 8, Alg. 1 :178)."""
    k = np.asarray(k_a, dtype=np.float64)
    if model.k_is_roped:
        k = rope(k, pos, model.rope_theta_producer, -1, model.n_kv_heads, model.head_dim,
                 model.rope_style)
    return _translate(model, k, layer.mean_src_k, layer.enc_k, False)


def encode_v(model: Model, layer: Layer, v_a: np.ndarray) -> np.ndarray:
    """Z_V = (V_A - mu_src,V) W_enc,V   (Eq. 8; "Values V are processed directly" :127)."""
    return _translate(model, np.asarray(v_a, dtype=np.float64), layer.mean_src_v, layer.enc_v, False)


def encode_h(model: Model, layer: Layer, h_a: np.ndarray) -> np.ndarray:
    """Z_H = (x_norm,A - mu_src,H) W_enc,H   (Eq. 10, Alg. 1 :179)."""
    return _sub(np.asarray(h_a, dtype=np.float64), layer.mean_src_h) @ layer.enc_h


Codes = Dict[Tuple[int, int], Tuple[np.ndarray, Optional[np.ndarray]]]


def scd_encode(model: Model, layers: Sequence[Layer], batch: Batch,
               k: Dict[int, np.ndarray], v: Dict[int, np.ndarray],
               h: Dict[int, np.ndarray]) -> Codes:
    """Alg. 1 producer half.  Returns {(layer, branch): (q, scale)}.
    REUSE layers emit K and V codes; PATCH layers emit only the H code."""
    pos = positions(batch)
    out: Codes = {}
    for i, l in enumerate(layers):
        if l.kind == REUSE:
            out[(i, BRANCH_K)] = pack_codes(encode_k(model, l, k[i], pos), model.code_dtype)
            out[(i, BRANCH_V)] = pack_codes(encode_v(model, l, v[i]), model.code_dtype)
        else:
            out[(i, BRANCH_H)] = pack_codes(encode_h(model, l, h[i]), model.code_dtype)
    return out


# --------------------------------------------------------------------------------------
# a6-a7 / A9: consumer REUSE decode  (Eq. 9, RoPE :152, Alg. 1 :184)
# --------------------------------------------------------------------------------------
def reuse_decode_layer(model: Model, layer: Layer, z_k: np.ndarray, z_v: np.ndarray,
                       pos: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    """K_B = RoPE(Z_K W_dec,K + mu_dst,K);  V_B = Z_V W_dec,V + mu_dst,V."""
    k = _translate(model, z_k, layer.mean_dst_k, layer.dec_k, True)
    if model.rope_on_reuse_k:
        k = rope(k, pos, model.rope_theta_consumer, +1, model.n_kv_heads, model.head_dim,
                 model.rope_style)
    v = _translate(model, z_v, layer.mean_dst_v, layer.dec_v, True)
    return k, v


# --------------------------------------------------------------------------------------
# a9-a11 / A11, A12: consumer PATCH  (Eq. 11, Eq. 12a/b :190-193)
# --------------------------------------------------------------------------------------
def silu(x: np.ndarray) -> np.ndarray:
    """SiLU(x) = x / (1 + e^-x)."""
    return x / (1.0 + np.exp(-x))


def aligner(model: Model, layer: Layer, z_h: np.ndarray) -> np.ndarray:
    """g_theta (Eq. 11), read as a 2-layer MLP: u = act(z W1 + b1) W2 + b2."""
    a = z_h @ layer.w1
    if layer.b1 is not None:
        a = a + layer.b1[None, :]
    if model.patch_act == ACT_SILU:
        a = silu(a)
    u = a @ layer.w2
    if layer.b2 is not None:
        u = u + layer.b2[None, :]
    return u


def rms_consistent(model: Model, layer: Layer, u: np.ndarray) -> np.ndarray:
    """NORM_RMS: h = gamma * u / sqrt(mean_i u_i^2 + eps); NORM_NONE: h = u."""
    if model.patch_norm == NORM_NONE:
        return u
    ms = np.mean(u * u, axis=1, keepdims=True)
    return layer.norm_gamma[None, :] * u / np.sqrt(ms + model.rms_eps)


def patch_layer(model: Model, layer: Layer, z_h: np.ndarray,
                pos: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    """K^ = RoPE(H^ W_k^T + b_k);  V^ = H^ W_v^T + b_v   (Eq. 12a/b; HF weights are
    [out, in] so the paper's `H W_k` is `H @ w_k.T`)."""
    hhat = rms_consistent(model, layer, aligner(model, layer, z_h))
    k = hhat @ layer.w_k.T
    if layer.b_k is not None:
        k = k + layer.b_k[None, :]
    k = rope(k, pos, model.rope_theta_consumer, +1, model.n_kv_heads, model.head_dim,
             model.rope_style)
    v = hhat @ layer.w_v.T
    if layer.b_v is not None:
        v = v + layer.b_v[None, :]
    return k, v


# --------------------------------------------------------------------------------------
# whole-call forms (Alg. 1 consumer half PAPER.md:182-184; cache assembly F.2 :610-616)
# --------------------------------------------------------------------------------------
def scd_reuse_decode(model: Model, layers: Sequence[Layer], batch: Batch, codes: Codes,
                     k_pool: Dict[int, np.ndarray], v_pool: Dict[int, np.ndarray],
                     rows: Optional[np.ndarray] = None) -> None:
    """Decode every REUSE layer into the paged pools (fp64 pools [n_blocks, bs, H, d_h]).
    `rows` restricts the work to a subset of packed rows (rows are independent,
    PAPER.md:102); untouched slots keep whatever the pool held."""
    pos = positions(batch)
    slots = slot_mapping(batch, model.block_size)
    sel = np.arange(batch.total_tokens) if rows is None else np.asarray(rows)
    for i, l in enumerate(layers):
        if l.kind != REUSE:
            continue
        qk, sk = codes[(i, BRANCH_K)]
        qv, sv = codes[(i, BRANCH_V)]
        zk = unpack_codes(qk[sel], None if sk is None else sk[sel], model.code_dtype)
        zv = unpack_codes(qv[sel], None if sv is None else sv[sel], model.code_dtype)
        k, v = reuse_decode_layer(model, l, zk, zv, pos[sel])
        write_paged(k_pool[i], slots[sel], k)
        write_paged(v_pool[i], slots[sel], v)


def scd_patch(model: Model, layers: Sequence[Layer], batch: Batch, codes: Codes,
              k_pool: Dict[int, np.ndarray], v_pool: Dict[int, np.ndarray],
              rows: Optional[np.ndarray] = None) -> None:
    """Regenerate every PATCH layer's K/V into the paged pools."""
    pos = positions(batch)
    slots = slot_mapping(batch, model.block_size)
    sel = np.arange(batch.total_tokens) if rows is None else np.asarray(rows)
    for i, l in enumerate(layers):
        if l.kind != PATCH:
            continue
        qh, sh = codes[(i, BRANCH_H)]
        zh = unpack_codes(qh[sel], None if sh is None else sh[sel], model.code_dtype)
        k, v = patch_layer(model, l, zh, pos[sel])
        write_paged(k_pool[i], slots[sel], k)
        write_paged(v_pool[i], slots[sel], v)
