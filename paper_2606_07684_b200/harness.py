"""Problem set-up around the C ABI: turns a WorkloadConfig into device buffers, a plan and
the three hot calls.  Allocation and marshalling only -- used by tests, bench.py and
__graft_entry__.smoke().  No arithmetic of the method lives here."""
from __future__ import annotations

from typing import Dict, List, Optional, Sequence

import torch

from . import binding as B
from . import workloads as W


GUARD_BYTES, GUARD_BYTE = 4096, 0xA5


class CodecProblem:
    """One synthetic workload resident on `device`: artifacts, plan, batch, code buffer,
    workspace and sentinel-filled paged pools."""

    def __init__(self, cfg: W.WorkloadConfig, device, pos_offset: Optional[Sequence[int]] = None,
                 k_is_roped: bool = True, rope_on_reuse_k: bool = True, patch_norm: int = B.SCD_NORM_RMS,
                 patch_act: int = B.SCD_ACT_SILU, rope_style: int = B.SCD_ROPE_HALF,
                 rope_theta_consumer: Optional[float] = None, use_means: bool = True,
                 artifacts: Optional[List[W.LayerArtifacts]] = None, per_head_rank: int = 0, gen_device=None):
        """`gen_device`: where the synthetic tensors are drawn and the bases fitted (default: `device`).  "cpu" keeps
        the library eigen-solver / QR kernels off the GPU, so that a launch trace of a short run (smoke) shows the
        codec's own kernels."""
        self.cfg = cfg
        self.device = torch.device(device)
        self.gen_device = self.device if gen_device is None else torch.device(gen_device)
        self.batch = W.make_batch(cfg, self.device, pos_offset)
        self.T = self.batch.total_tokens
        self.use_means = use_means
        self.arts = artifacts if artifacts is not None else [
            W.make_layer_artifacts(cfg, l, self.gen_device, total_rows=max(self.T, 1), per_head_rank=per_head_rank).to(self.device)
            for l in range(cfg.n_layers)]
        self.per_head_rank = per_head_rank
        max_off = max(pos_offset) if pos_offset is not None else 0
        self.max_position = max(16, (self.batch.max_seqlen + max_off + 15) // 16 * 16)
        self.model = B.model_desc(
            n_layers=cfg.n_layers, d_model=cfg.d_model, n_kv_heads=cfg.n_kv_heads, head_dim=cfg.head_dim,
            max_position=self.max_position, state_dtype=cfg.state_dtype, code_dtype=cfg.code_dtype,
            rope_theta_producer=cfg.rope_theta, rope_theta_consumer=rope_theta_consumer, block_size=cfg.block_size,
            rope_style=rope_style, k_is_roped=int(k_is_roped), rope_on_reuse_k=int(rope_on_reuse_k),
            patch_act=patch_act, patch_norm=patch_norm, rms_eps=cfg.rms_eps, reuse_per_head=int(per_head_rank > 0))
        self.layer_descs = [self._desc(a) for a in self.arts]
        self.plan = B.scd_plan(self.model, self.layer_descs)
        torch.cuda.synchronize(self.device)
        self.code_bytes, self.ws_bytes, self.payload_bytes = self.plan.query(self.T)
        # both buffers sit in front of GUARD_BYTES of guard and start out filled with GUARD_BYTE, so that tests can see
        # writes into the padding between code segments, past the last scale segment or past the workspace
        self._codes_alloc = torch.full((max(self.code_bytes, 128) + GUARD_BYTES,), GUARD_BYTE, dtype=torch.uint8, device=self.device)
        self.codes = self._codes_alloc[:max(self.code_bytes, 128)]
        self._ws_alloc = torch.full((max(self.ws_bytes, 128) + GUARD_BYTES,), GUARD_BYTE, dtype=torch.uint8, device=self.device)
        self.workspace = self._ws_alloc[:max(self.ws_bytes, 128)]
        self.k_pool: List[torch.Tensor] = []
        self.v_pool: List[torch.Tensor] = []
        self.bdesc = B.batch_desc(self.batch.cu_seqlens, self.batch.page_table, self.batch.pos_offset,
                                  self.batch.seqlens, max_off)

    def _desc(self, a: W.LayerArtifacts) -> B.LayerDesc:
        mk = lambda t: t if self.use_means else None
        if a.kind == W.REUSE:
            return B.reuse_layer_desc(enc_k=a.enc_k, enc_v=a.enc_v, dec_k=a.dec_k, dec_v=a.dec_v,
                                      mean_src_k=mk(a.mean_k), mean_src_v=mk(a.mean_v),
                                      mean_dst_k=mk(a.mean_k if a.mean_dst_k is None else a.mean_dst_k),
                                      mean_dst_v=mk(a.mean_v if a.mean_dst_v is None else a.mean_dst_v))
        return B.patch_layer_desc(enc_h=a.enc_h, mean_src_h=mk(a.mean_h), w1=a.w1, b1=a.b1, w2=a.w2, b2=a.b2,
                                  norm_gamma=a.gamma, w_k=a.w_k, w_v=a.w_v, b_k=a.b_k, b_v=a.b_v)

    # ---- buffers -------------------------------------------------------------------
    def alloc_pools(self) -> None:
        self.k_pool = [W.make_sentinel_pool(self.cfg, self.batch.n_blocks, self.device) for _ in range(self.cfg.n_layers)]
        self.v_pool = [W.make_sentinel_pool(self.cfg, self.batch.n_blocks, self.device) for _ in range(self.cfg.n_layers)]

    def make_sources(self):
        """Producer states: K, V for REUSE layers (content-space low-rank-plus-noise; the
        caller decides whether to treat K as post-RoPE), H for PATCH layers."""
        cfg, L = self.cfg, self.cfg.n_layers
        k: List[Optional[torch.Tensor]] = [None] * L
        v: List[Optional[torch.Tensor]] = [None] * L
        h: List[Optional[torch.Tensor]] = [None] * L
        for l in range(L):
            if l in cfg.patch_layers:
                h[l] = W.make_state(cfg, l, 2, self.T, self.gen_device).to(self.device)
            else:
                k[l] = W.make_state(cfg, l, 0, self.T, self.gen_device).to(self.device)
                v[l] = W.make_state(cfg, l, 1, self.T, self.gen_device).to(self.device)
        return k, v, h

    # ---- the three hot calls ---------------------------------------------------------
    def encode(self, k, v, h, stream=None, layers=None, src_page_table=None, src_n_blocks=0) -> int:
        cfg = self.cfg
        return B.scd_encode(self.plan, self.bdesc, k, v, h, self.codes, cfg.D, cfg.head_dim, cfg.d_model, stream, layers,
                            src_page_table, src_n_blocks)

    def reuse_decode(self, stream=None, layers=None) -> int:
        return B.scd_reuse_decode(self.plan, self.bdesc, self.codes, self.k_pool, self.v_pool, self.batch.n_blocks, stream,
                                  layers)

    def patch(self, stream=None, layers=None) -> int:
        return B.scd_patch(self.plan, self.bdesc, self.codes, self.k_pool, self.v_pool, self.batch.n_blocks,
                           self.workspace, stream, layers)

    # ---- views ---------------------------------------------------------------------
    def code_ranges(self):
        """Byte ranges [begin, end) of the code buffer that scd_encode may write: every segment's codes and scales."""
        cb = {W.F32: 4, W.BF16: 2, W.E4M3_ROWSCALE: 1}[self.cfg.code_dtype]
        out = []
        for l in range(self.cfg.n_layers):
            for br in ((2,) if self.arts[l].kind == W.PATCH else (0, 1)):
                off, soff, r = self.plan.code_segment(l, br, self.T)
                out.append((off, off + self.T * r * cb))
                if self.cfg.code_dtype == W.E4M3_ROWSCALE:
                    out.append((soff, soff + self.T * 4))
        return sorted(out)

    def guard_violations(self):
        """Bytes outside the writable ranges that no longer hold GUARD_BYTE: (in the code buffer's padding and guard,
        in the guard after the workspace)."""
        bad_c, at = 0, 0
        for b, e in self.code_ranges() + [(self._codes_alloc.numel(), self._codes_alloc.numel())]:
            if b > at:
                bad_c += int((self._codes_alloc[at:b] != GUARD_BYTE).sum())
            at = max(at, e)
        bad_w = int((self._ws_alloc[self.workspace.numel():] != GUARD_BYTE).sum())
        return bad_c, bad_w

    def code_view(self, layer: int, branch: int):
        """(codes [T, r] tensor view in the code dtype, scales [T] fp32 or None)."""
        off, soff, r = self.plan.code_segment(layer, branch, self.T)
        cd = self.cfg.code_dtype
        dt, eb = {W.F32: (torch.float32, 4), W.BF16: (torch.bfloat16, 2), W.E4M3_ROWSCALE: (torch.uint8, 1)}[cd]
        q = self.codes[off:off + self.T * r * eb].view(dt).view(self.T, r)
        s = None
        if cd == W.E4M3_ROWSCALE:
            s = self.codes[soff:soff + self.T * 4].view(torch.float32)
        return q, s
