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
                       mean_src_k=mk(a.mean_k), mean_src_v=mk(a.mean_v), mean_dst_k=mk(a.mean_k), mean_dst_v=mk(a.mean_v))
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


def check_encode(prob, k, v, h, rows: Optional[np.ndarray] = None) -> Dict:
    """GPU codes vs oracle codes per (layer, branch) on dequantised values."""
    om, ob = oracle_model(prob), oracle_batch(prob)
    pos = O.positions(ob)
    sel = np.arange(prob.T) if rows is None else rows
    tol = TOL[prob.cfg.state_dtype]
    worst = 0.0
    tsel = torch.from_numpy(sel).to(prob.device)
    for l in range(prob.cfg.n_layers):
        ol = oracle_layer(prob, l)
        if ol.kind == O.REUSE:
            zs = {O.BRANCH_K: O.encode_k(om, ol, np64(k[l][tsel]), pos[sel]), O.BRANCH_V: O.encode_v(om, ol, np64(v[l][tsel]))}
        else:
            zs = {O.BRANCH_H: O.encode_h(om, ol, np64(h[l][tsel]))}
        for br, z in zs.items():
            q_o, s_o = O.pack_codes(z, om.code_dtype)
            want = O.unpack_codes(q_o, s_o, om.code_dtype)
            q_g, s_g = gpu_codes(prob, l, br, None if rows is None else sel)
            got = O.unpack_codes(q_g, s_g, om.code_dtype)
            err = rel_fro(got, want)
            worst = max(worst, err)
            assert err <= tol, f"encode layer {l} branch {br}: rel fro {err:.3e} > {tol}"
            if om.code_dtype == O.E4M3_ROWSCALE:
                # scale = row amax / 448: agrees to fp32 accumulation noise, except for K on the bf16 path,
                # where the deRoPE'd operand is re-rounded to bf16 before the MMA (U15): 2^-8
                s_rtol = 2.0 ** -8 if (br == O.BRANCH_K and om.k_is_roped and prob.cfg.state_dtype == W.BF16) else 1e-5
                np.testing.assert_allclose(s_g, s_o, rtol=s_rtol, err_msg=f"e4m3 scales layer {l} branch {br}")
                # each element within one e4m3 step (2^-3 relative in the normal range, 2^-9*s absolute below).
                # K on the bf16 path: the rotated operand k~ is re-rounded to bf16 (2^-9 rel. per element) with
                # fp16 cos/sin, so z_i may move by up to 2^-8 * ||k~||_2 * ||W_enc[:, i]||_2 on top of that step.
                step = np.maximum(np.abs(want) * 2.0 ** -3, s_o.astype(np.float64)[:, None] * 2.0 ** -9)
                if s_rtol > 1e-5:
                    kt = O.rope(np64(k[l][tsel]), pos[sel], om.rope_theta_producer, -1, om.n_kv_heads, om.head_dim,
                                om.rope_style)
                    if om.reuse_per_head:     # code (t, h, i) sees head h of the row only
                        hn = np.linalg.norm(kt.reshape(len(kt), om.n_kv_heads, om.head_dim), axis=2)
                        extra = hn[:, :, None] * np.linalg.norm(ol.enc_k, axis=0)[None, None, :]
                        step = step + 2.0 ** -8 * extra.reshape(len(kt), -1)
                    else:
                        step = step + 2.0 ** -8 * np.linalg.norm(kt, axis=1)[:, None] * np.linalg.norm(ol.enc_k, axis=0)[None, :]
                assert np.all(np.abs(got - want) <= step * 1.001), f"e4m3 code off by more than one step, layer {l} branch {br}"
    return {"worst_rel_fro": worst}


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


def check_reuse_decode(prob, rows: Optional[np.ndarray] = None) -> Dict:
    om, ob = oracle_model(prob), oracle_batch(prob)
    pos, slots = O.positions(ob), O.slot_mapping(ob, om.block_size)
    sel = np.arange(prob.T) if rows is None else rows
    tol = TOL[prob.cfg.state_dtype]
    worst = 0.0
    for l in range(prob.cfg.n_layers):
        if prob.arts[l].kind != W.REUSE:
            continue
        ol = oracle_layer(prob, l)
        qk, sk = gpu_codes(prob, l, O.BRANCH_K, None if rows is None else sel)
        qv, sv = gpu_codes(prob, l, O.BRANCH_V, None if rows is None else sel)
        k_o, v_o = O.reuse_decode_layer(om, ol, O.unpack_codes(qk, sk, om.code_dtype),
                                        O.unpack_codes(qv, sv, om.code_dtype), pos[sel])
        for name, want, pool in (("K", k_o, prob.k_pool[l]), ("V", v_o, prob.v_pool[l])):
            err = rel_fro(_gather(pool, slots[sel]), want)
            worst = max(worst, err)
            assert err <= tol, f"reuse_decode layer {l} {name}: rel fro {err:.3e} > {tol}"
    return {"worst_rel_fro": worst, "slots": slots}


def check_patch(prob, rows: Optional[np.ndarray] = None) -> Dict:
    om, ob = oracle_model(prob), oracle_batch(prob)
    pos, slots = O.positions(ob), O.slot_mapping(ob, om.block_size)
    sel = np.arange(prob.T) if rows is None else rows
    tol = TOL[prob.cfg.state_dtype]
    worst = 0.0
    for l in range(prob.cfg.n_layers):
        if prob.arts[l].kind != W.PATCH:
            continue
        ol = oracle_layer(prob, l)
        qh, sh = gpu_codes(prob, l, O.BRANCH_H, None if rows is None else sel)
        k_o, v_o = O.patch_layer(om, ol, O.unpack_codes(qh, sh, om.code_dtype), pos[sel])
        for name, want, pool in (("K", k_o, prob.k_pool[l]), ("V", v_o, prob.v_pool[l])):
            err = rel_fro(_gather(pool, slots[sel]), want)
            worst = max(worst, err)
            assert err <= tol, f"patch layer {l} {name}: rel fro {err:.3e} > {tol}"
    return {"worst_rel_fro": worst, "slots": slots}


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
