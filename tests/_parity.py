"""Helpers for the GPU-vs-oracle parity tests (SURVEY.md 8(c) "Parity protocol").

Each stage is checked on its own with the oracle fed the same input bits as the GPU:
codes produced by the GPU encode are copied back and become the oracle's decode / patch
input, so a rounding flip in one stage never leaks into the next stage's verdict.
"""
from __future__ import annotations

from typing import Dict, List, Optional, Sequence

import numpy as np
import torch

from oracle import scd_oracle as O
from paper_2606_07684_b200 import workloads as W

TOL = {W.F32: 1e-5, W.BF16: 2e-2}          # north_star: rel. Frobenius per layer (fp32 / bf16 outputs)


def np64(t: Optional[torch.Tensor]) -> Optional[np.ndarray]:
    return None if t is None else t.detach().to("cpu").double().numpy()


def rel_fro(a: np.ndarray, b: np.ndarray) -> float:
    den = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / den) if den > 0 else float(np.linalg.norm(a - b))


# ---------------------------------------------------------------------------------------------------------
# Under the per-layer Frobenius criterion (north_star) every comparison is also made block by block and
# element by element, so that one wrong head of one token, one wrong 16-column chunk or two swapped rows fail
# even in a batch of thousands of rows (a norm over the whole layer hides all three).
#   block   = one [row, head] slice (codes: the row, or the head's r codes in the per-head reading):
#             ||got - want|| <= tol * max(||want_block||, ||want_row|| / (4 sqrt(n_blocks)))
#   element = |got - want| <= rel * |want| + k_abs * rms(block reference) [+ extra]
# `rel` is the rounding of the stored value (bf16 half-ulp 2^-8 against an unrounded reference, one ulp 2^-7
# when both sides are rounded codes; 1e-5 on the fp32 path), `k_abs` the noise the arithmetic of the stage
# may add relative to the block's rms (derived per stage where it is used).
# ---------------------------------------------------------------------------------------------------------
FINE_TOL = {W.F32: 1e-5, W.BF16: 2e-2}


def fine_check(got: np.ndarray, want: np.ndarray, n_blocks: int, tol: float, rel: float, k_abs: float, what: str,
               extra: Optional[np.ndarray] = None) -> Dict[str, float]:
    """Block and element bounds described above.  Returns the largest used fraction of either bound."""
    T, W_ = want.shape
    if T == 0:
        return {"block": 0.0, "element": 0.0}
    bw = W_ // n_blocks
    g3, w3 = got.reshape(T, n_blocks, bw), want.reshape(T, n_blocks, bw)
    blk = np.linalg.norm(w3, axis=2)
    floor = np.linalg.norm(want, axis=1)[:, None] / (4.0 * np.sqrt(n_blocks))
    ref = np.maximum(blk, floor)                                       # [T, n_blocks]
    ref = np.where(ref > 0, ref, 1e-30)
    err = np.linalg.norm(g3 - w3, axis=2)
    used_b = err / (tol * ref)
    ib = np.unravel_index(np.argmax(used_b), used_b.shape)
    assert used_b[ib] <= 1.0, (f"{what}: block (row {ib[0]}, block {ib[1]}) off by {err[ib]:.3e} "
                               f"= {err[ib] / ref[ib]:.3e} of its reference norm (tol {tol})")
    bound = rel * np.abs(w3) + k_abs * (ref / np.sqrt(bw))[:, :, None]
    if extra is not None:
        bound = bound + extra.reshape(T, n_blocks, bw)
    used_e = np.abs(g3 - w3) / bound
    ie = np.unravel_index(np.argmax(used_e), used_e.shape)
    assert used_e[ie] <= 1.0, (f"{what}: element (row {ie[0]}, block {ie[1]}, col {ie[2]}) got {g3[ie]:.6g} want {w3[ie]:.6g}: "
                               f"|diff| {abs(g3[ie] - w3[ie]):.3e} > bound {bound[ie]:.3e}")
    return {"block": float(used_b[ib]), "element": float(used_e[ie])}


def _merge(stats: Dict[str, float], new: Dict[str, float], prefix: str = "") -> None:
    for k_, v_ in new.items():
        stats[prefix + k_] = max(stats.get(prefix + k_, 0.0), v_)


def oracle_model(prob) -> O.Model:
    m = prob.model
    return O.Model(n_layers=m.n_layers, d_model=m.d_model, n_kv_heads=m.n_kv_heads, head_dim=m.head_dim,
                   block_size=m.block_size, rope_theta_producer=m.rope_theta_producer,
                   rope_theta_consumer=m.rope_theta_consumer, rope_style=m.rope_style,
                   k_is_roped=bool(m.k_is_roped), rope_on_reuse_k=bool(m.rope_on_reuse_k), code_dtype=m.code_dtype,
                   patch_act=m.patch_act, patch_norm=m.patch_norm, rms_eps=float(m.rms_eps),
                   reuse_per_head=bool(m.reuse_per_head))


def oracle_layer(prob, l: int) -> O.Layer:
    a = prob.arts[l]
    mk = (lambda t: np64(t)) if prob.use_means else (lambda t: None)
    if a.kind == W.REUSE:
        return O.Layer(O.REUSE, enc_k=np64(a.enc_k), enc_v=np64(a.enc_v), dec_k=np64(a.dec_k), dec_v=np64(a.dec_v),
                       mean_src_k=mk(a.mean_k), mean_src_v=mk(a.mean_v),
                       mean_dst_k=mk(a.mean_k if a.mean_dst_k is None else a.mean_dst_k),
                       mean_dst_v=mk(a.mean_v if a.mean_dst_v is None else a.mean_dst_v))
    return O.Layer(O.PATCH, enc_h=np64(a.enc_h), mean_src_h=mk(a.mean_h), w1=np64(a.w1), b1=np64(a.b1), w2=np64(a.w2),
                   b2=np64(a.b2), norm_gamma=np64(a.gamma), w_k=np64(a.w_k), w_v=np64(a.w_v), b_k=np64(a.b_k),
                   b_v=np64(a.b_v))


def oracle_batch(prob) -> O.Batch:
    b = prob.batch
    return O.Batch(b.cu_seqlens.cpu().numpy().astype(np.int64), b.page_table.cpu().numpy().astype(np.int64),
                   None if b.pos_offset is None else b.pos_offset.cpu().numpy().astype(np.int64))


def roped_producer_k(prob, k: List[Optional[torch.Tensor]]) -> List[Optional[torch.Tensor]]:
    """The producer cache holds RoPE(content keys): build it with the oracle's
    RoPE on the host and hand the same (re-cast) bits to both sides."""
    om, pos = oracle_model(prob), O.positions(oracle_batch(prob))
    out: List[Optional[torch.Tensor]] = []
    for t in k:
        if t is None:
            out.append(None)
            continue
        r = O.rope(np64(t), pos, om.rope_theta_producer, +1, om.n_kv_heads, om.head_dim, om.rope_style)
        out.append(torch.from_numpy(r).to(t.dtype).to(t.device))
    return out


def gpu_codes(prob, layer: int, branch: int, rows: Optional[np.ndarray] = None):
    """Stored codes of a segment as the oracle's (q, scale) pair."""
    q, s = prob.code_view(layer, branch)
    if rows is not None:
        idx = torch.from_numpy(rows).to(q.device)
        q = q[idx]
        s = None if s is None else s[idx]
    cd = prob.cfg.code_dtype
    if cd == W.E4M3_ROWSCALE:
        return q.cpu().numpy().astype(np.uint8), s.cpu().numpy().astype(np.float32)
    if cd == W.F32:
        return q.cpu().numpy().astype(np.float32), None
    return q.double().cpu().numpy(), None


def _rerounded_operand_noise(om, ol, kt: np.ndarray) -> np.ndarray:
    """bf16 path, K branch (U15): the deRoPE'd operand k~ is re-rounded to bf16 for the MMA (each element
    moves by up to 2^-9 |k~_j|) with fp16 cos/sin (2^-12 abs on each, i.e. up to 2^-12 (|a| + |b|) per pair), so
    z_i = sum_j k~_j W_ji moves by sum_j delta_j W_ji with independent-sign delta_j: a random sum whose standard
    deviation is <= 2^-9 / sqrt(3) * sqrt(sum_j e_j W_ji^2), e_j = k~_j^2 + k~_partner(j)^2.  Returned: 2^-7 times that
    root (>= 5.5 sigma) per code -- the term added to the element bound and to the scale agreement for K codes."""
    T = len(kt)
    half = om.head_dim // 2
    k3 = kt.reshape(T, om.n_kv_heads, om.head_dim)
    if om.rope_style == O.ROPE_HALF:
        part = np.concatenate([k3[..., half:], k3[..., :half]], axis=2)
    else:
        part = k3.reshape(T, om.n_kv_heads, half, 2)[..., ::-1].reshape(T, om.n_kv_heads, om.head_dim)
    e = k3 ** 2 + part ** 2
    if om.reuse_per_head:       # code (t, h, i) sees head h only
        return 2.0 ** -7 * np.sqrt(e.reshape(T * om.n_kv_heads, om.head_dim) @ ol.enc_k ** 2).reshape(T, -1)
    return 2.0 ** -7 * np.sqrt(e.reshape(T, -1) @ ol.enc_k ** 2)


def e4m3_cell_check(z: np.ndarray, q: np.ndarray, s: np.ndarray, noise: np.ndarray, what: str) -> float:
    """Stored e4m3 codes q (bytes) with row scales s against the exact codes z: z / s must lie in the rounding cell of
    the stored code (between the midpoints to its two neighbours on the e4m3 grid; the outermost cell is open-ended),
    widened by noise / s.  Returns the largest fraction of the widening that was needed (0 = every code is the
    correctly rounded one of the oracle's own z under the stored scale)."""
    mags = O.E4M3_VALUES[:0x7F]                                    # 0 .. 448 ascending
    code = (q & 0x7F).astype(np.int64)
    assert (code != 0x7F).all(), f"{what}: NaN code stored"
    sg = s.astype(np.float64)[:, None]
    sign = np.where((q & 0x80) != 0, -1.0, 1.0)
    a = np.where(code == 0, z / sg, sign * z / sg)                  # coordinate along the stored code's own sign
    m = mags[code]
    lower = np.where(code == 0, -mags[1] / 2.0, (mags[np.maximum(code - 1, 0)] + m) / 2.0)
    upper = np.where(code == 0x7E, np.inf, (m + mags[np.minimum(code + 1, 0x7E)]) / 2.0)
    outside = np.maximum(np.maximum(lower - a, a - upper), 0.0) * sg     # distance outside the cell, in z units
    used = outside / noise
    i = np.unravel_index(np.argmax(used), used.shape)
    assert used[i] <= 1.0, (f"{what}: code at (row {i[0]}, col {i[1]}) = {sign[i] * m[i]:g} x {sg[i[0], 0]:.6g} is not a rounding of "
                            f"z = {z[i]:.8g}: {outside[i]:.3e} outside its cell, allowance {noise[i]:.3e}")
    return float(used[i])


def check_encode(prob, k, v, h, rows: Optional[np.ndarray] = None) -> Dict:
    """GPU codes vs oracle codes per (layer, branch) on dequantised values: Frobenius per segment (north_star), then
    per row (per head's codes in the per-head reading) and per element (fine_check)."""
    om, ob = oracle_model(prob), oracle_batch(prob)
    pos = O.positions(ob)
    sel = np.arange(prob.T) if rows is None else rows
    sd = prob.cfg.state_dtype
    tol = TOL[sd]
    worst = 0.0
    stats: Dict[str, float] = {}
    tsel = torch.from_numpy(sel).to(prob.device)
    for l in range(prob.cfg.n_layers):
        ol = oracle_layer(prob, l)
        if ol.kind == O.REUSE:
            zs = {O.BRANCH_K: O.encode_k(om, ol, np64(k[l][tsel]), pos[sel]), O.BRANCH_V: O.encode_v(om, ol, np64(v[l][tsel]))}
        else:
            zs = {O.BRANCH_H: O.encode_h(om, ol, np64(h[l][tsel]))}
        for br, z in zs.items():
            what = f"encode layer {l} branch {br}"
            q_o, s_o = O.pack_codes(z, om.code_dtype)
            want = O.unpack_codes(q_o, s_o, om.code_dtype)
            q_g, s_g = gpu_codes(prob, l, br, None if rows is None else sel)
            got = O.unpack_codes(q_g, s_g, om.code_dtype)
            err = rel_fro(got, want)
            worst = max(worst, err)
            assert err <= tol, f"{what}: rel fro {err:.3e} > {tol}"
            n_blk = om.n_kv_heads if (om.reuse_per_head and br != O.BRANCH_H) else 1
            # the K operand of the bf16 path is re-rounded after the rotation: its own noise term (see above)
            rerounded = br == O.BRANCH_K and om.k_is_roped and sd == W.BF16
            extra, kt = None, None
            if br == O.BRANCH_K:
                kt = np64(k[l][tsel])
                if om.k_is_roped:
                    kt = O.rope(kt, pos[sel], om.rope_theta_producer, -1, om.n_kv_heads, om.head_dim, om.rope_style)
            if rerounded:
                extra = _rerounded_operand_noise(om, ol, kt)
            if om.code_dtype == O.E4M3_ROWSCALE:
                # fp32 accumulation of x W - c on the GPU against fp64: 2^-16 of sum_j |x_j| |W_ji| + |mu|.|W_i| is a
                # generous cover (K <= 8192 products at 2^-24 each, signs random)
                x_in = kt if br == O.BRANCH_K else (np64(v[l][tsel]) if br == O.BRANCH_V else np64(h[l][tsel]))
                w_enc = {O.BRANCH_K: ol.enc_k, O.BRANCH_V: ol.enc_v, O.BRANCH_H: ol.enc_h}[br]
                mu = {O.BRANCH_K: ol.mean_src_k, O.BRANCH_V: ol.mean_src_v, O.BRANCH_H: ol.mean_src_h}[br]
                if n_blk > 1:
                    acc = (np.abs(x_in).reshape(-1, om.head_dim) @ np.abs(w_enc)).reshape(len(x_in), -1)
                    acc = acc + (0.0 if mu is None else np.tile(np.abs(mu) @ np.abs(w_enc), n_blk)[None, :])
                else:
                    acc = np.abs(x_in) @ np.abs(w_enc) + (0.0 if mu is None else (np.abs(mu) @ np.abs(w_enc))[None, :])
                noise = 2.0 ** -16 * acc + (extra if rerounded else 0.0)
                # scale = row amax / 448; amax is 1-Lipschitz in the sup norm, so it moves by at most the largest
                # element perturbation of the row
                s_tol = 2.0 ** -22 * s_o.astype(np.float64) + noise.max(axis=1) / 448.0
                s_used = np.abs(s_g.astype(np.float64) - s_o) / s_tol
                assert s_used.max() <= 1.0, f"{what}: e4m3 scale of row {int(np.argmax(s_used))} off by {s_used.max():.2f} x its bound"
                _merge(stats, {"scale": float(s_used.max())}, "e4m3K_" if rerounded else "e4m3_")
                # every stored code must be THE correctly rounded code of a value within `noise` of the oracle's exact
                # z under the stored scale (a code may differ from the oracle's own only where z / s sits that close to
                # a rounding boundary, SURVEY U14 ii); how much of the noise allowance is used is reported
                used = e4m3_cell_check(z, q_g, s_g, noise, what)
                _merge(stats, {"noise_used": used}, "e4m3K_" if rerounded else "e4m3_")
            else:
                # both sides rounded to the code dtype: one ulp (2^-7 for bf16) where the two straddle a rounding
                # boundary; fp32 accumulation of K products: 2^-10 of the row rms covers it with a wide margin
                rel = 2.0 ** -7 * 1.001 if om.code_dtype == O.BF16 else 1e-5
                k_abs = 2.0 ** -10 if om.code_dtype == O.BF16 else 1e-5
                _merge(stats, fine_check(got, want, n_blk, FINE_TOL[sd], rel, k_abs, what, extra), "encK_" if rerounded else "enc_")
    return {"worst_rel_fro": worst, **stats}


def _gather(pool: torch.Tensor, slots: np.ndarray) -> np.ndarray:
    D = pool.shape[2] * pool.shape[3]
    flat = pool.view(-1, D)
    return flat[torch.from_numpy(slots).to(pool.device)].double().cpu().numpy()


def check_untouched(prob, layers: Sequence[int], written_slots: np.ndarray, also_untouched_layers: Sequence[int] = ()):
    """Bit-exact: every pool element outside the written slot set still holds the sentinel."""
    cfg = prob.cfg
    n_slots = prob.batch.n_blocks * cfg.block_size
    mask = torch.ones(n_slots, dtype=torch.bool, device=prob.device)
    mask[torch.from_numpy(written_slots).to(prob.device)] = False
    int_t = torch.int32 if cfg.state_dtype == W.F32 else torch.int16
    sent = 0x7FC00001 if cfg.state_dtype == W.F32 else 0x7FC1
    for l in layers:
        for pool in (prob.k_pool[l], prob.v_pool[l]):
            bits = pool.view(int_t).view(n_slots, -1)
            assert bool((bits[mask] == sent).all()), f"layer {l}: a slot outside the page table was written"
            assert not bool((bits[~mask] == sent).any()), f"layer {l}: an addressed slot was left unwritten"
    for l in also_untouched_layers:
        for pool in (prob.k_pool[l], prob.v_pool[l]):
            assert bool((pool.view(int_t) == sent).all()), f"layer {l} must not be touched by this call"


# Element noise allowed on top of the output rounding, relative to the rms of the element's [row, head] block:
#   REUSE decode: fp32 accumulation of r products and the RoPE mix with (cos, sin) good to 3e-5 (Q0.32 phase + MUFU):
#     3e-5 ||pair|| <= 3e-5 sqrt(d_h) rms = 2^-11.5 rms at d_h = 128 -> 2^-9.
#   PATCH: a and u^ are rounded to bf16 on the way (U15) and SiLU uses tanh.approx (2^-11): the chain's
#     measured relative error is 3.3e-3 of the row; an element may see ~10 sigma of it -> 2^-5.
#   fp32 path: 1e-5 throughout (the north_star tolerance).
K_ABS = {"reuse": {W.BF16: 2.0 ** -9, W.F32: 1e-5}, "patch": {W.BF16: 2.0 ** -5, W.F32: 1e-5}}
REL_OUT = {W.BF16: 2.0 ** -8 * 1.001, W.F32: 1e-5}      # stored K/V against the unrounded oracle value


def check_reuse_decode(prob, rows: Optional[np.ndarray] = None) -> Dict:
    om, ob = oracle_model(prob), oracle_batch(prob)
    pos, slots = O.positions(ob), O.slot_mapping(ob, om.block_size)
    sel = np.arange(prob.T) if rows is None else rows
    sd = prob.cfg.state_dtype
    tol = TOL[sd]
    worst = 0.0
    stats: Dict[str, float] = {}
    for l in range(prob.cfg.n_layers):
        if prob.arts[l].kind != W.REUSE:
            continue
        ol = oracle_layer(prob, l)
        qk, sk = gpu_codes(prob, l, O.BRANCH_K, None if rows is None else sel)
        qv, sv = gpu_codes(prob, l, O.BRANCH_V, None if rows is None else sel)
        k_o, v_o = O.reuse_decode_layer(om, ol, O.unpack_codes(qk, sk, om.code_dtype),
                                        O.unpack_codes(qv, sv, om.code_dtype), pos[sel])
        for name, want, pool in (("K", k_o, prob.k_pool[l]), ("V", v_o, prob.v_pool[l])):
            got = _gather(pool, slots[sel])
            err = rel_fro(got, want)
            worst = max(worst, err)
            assert err <= tol, f"reuse_decode layer {l} {name}: rel fro {err:.3e} > {tol}"
            _merge(stats, fine_check(got, want, om.n_kv_heads, FINE_TOL[sd], REL_OUT[sd], K_ABS["reuse"][sd],
                                     f"reuse_decode layer {l} {name}"), "dec_")
    return {"worst_rel_fro": worst, "slots": slots, **stats}


def check_patch(prob, rows: Optional[np.ndarray] = None) -> Dict:
    om, ob = oracle_model(prob), oracle_batch(prob)
    pos, slots = O.positions(ob), O.slot_mapping(ob, om.block_size)
    sel = np.arange(prob.T) if rows is None else rows
    sd = prob.cfg.state_dtype
    tol = TOL[sd]
    worst = 0.0
    stats: Dict[str, float] = {}
    for l in range(prob.cfg.n_layers):
        if prob.arts[l].kind != W.PATCH:
            continue
        ol = oracle_layer(prob, l)
        qh, sh = gpu_codes(prob, l, O.BRANCH_H, None if rows is None else sel)
        k_o, v_o = O.patch_layer(om, ol, O.unpack_codes(qh, sh, om.code_dtype), pos[sel])
        for name, want, pool in (("K", k_o, prob.k_pool[l]), ("V", v_o, prob.v_pool[l])):
            got = _gather(pool, slots[sel])
            err = rel_fro(got, want)
            worst = max(worst, err)
            assert err <= tol, f"patch layer {l} {name}: rel fro {err:.3e} > {tol}"
            _merge(stats, fine_check(got, want, om.n_kv_heads, FINE_TOL[sd], REL_OUT[sd], K_ABS["patch"][sd],
                                     f"patch layer {l} {name}"), "patch_")
    return {"worst_rel_fro": worst, "slots": slots, **stats}


def sample_rows(prob, n_random: int, seed: int = 0) -> np.ndarray:
    """First and last 128-row tile of every request, every ragged tail, plus a seeded sample."""
    cu = prob.batch.cu_seqlens.cpu().numpy().astype(np.int64)
    rows = []
    for b in range(len(cu) - 1):
        s, e = cu[b], cu[b + 1]
        rows += list(range(s, min(e, s + 8))) + list(range(max(s, e - 24), e))
    rng = np.random.default_rng(seed)
    if prob.T:
        rows += list(rng.integers(0, prob.T, n_random))
    return np.unique(np.array(rows, dtype=np.int64))
