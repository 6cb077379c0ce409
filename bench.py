#!/usr/bin/env python
"""bench.py -- SCD KV state codec on B200: one "step" = one pass of the whole hot path
(scd_encode -> scd_reuse_decode -> scd_patch, every row of SURVEY.md 8(a)) over one batch of
synthetic input.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config NAME] [--impl ours|reference]

Prints ONE JSON line (rank 0).  `value` = packed tokens whose K/V were rebuilt for all layers
per second of device time (CUDA events around the three C-ABI calls, L2 flushed between calls
outside the events, max over ranks).  `e2e` = the same with HOST buffers: pinned producer
states copied H2D, the three calls, the reconstructed pools copied D2H, all inside the timed
region.  `roofline` = the dominant kernel of the step, timed live with CUDA events on its
launching stream (scd_profile_* hooks).  `cpu_baseline` / `--impl reference` = the fp64 oracle
timed on the box's host cores on a bounded row sample.  Multi-GPU: the path has no exchange
step, so N ranks run N independent replicas ("replicas only") -- weak scaling.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "reconstructed KV tokens/s (REUSE+PATCH hybrid cache, encode->reuse_decode->patch)"
UNIT = "tokens/s"
KERNEL_NAMES = {100: "tc_gemm<codes,plain> (encode V/H)", 101: "tc_gemm<codes,derope> (encode K)",
                110: "tc_kv_kernel / tc_gemm<paged_kv> (reuse decode)", 120: "tc_gemm<aligner_in> (patch GEMM-1)",
                130: "tc_gemm<aligner_out> (patch GEMM-2)", 140: "tc_kv_kernel<dyn> (patch GEMM-3)"}     # 120-140: one launch per group of PATCH layers


# ------------------------------------------------------------------------------ helpers
def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16_tflops": d["bf16_tflops"],
                "bf16_tflops_sustained": d.get("bf16_tflops_sustained", d["bf16_tflops"]), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in self.rows if len(r) >= 6 for n, v in zip(names, r[2:6]) if v == "Active"})
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def workload_costs(cfg, T, reuse_rank=None):
    """Algorithmic bytes / FLOPs per call (stated in DESIGN.md)."""
    cb = {0: 4, 1: 2, 2: 1}[cfg.code_dtype]
    sb = 4 if cfg.code_dtype == 2 else 0
    ob = 4 if cfg.state_dtype == 0 else 2
    D, d, d_a, r = cfg.D, cfg.d_model, cfg.d_a, cfg.rank
    rr = reuse_rank or r              # codes per token and REUSE branch (per-head reading: H * r_head)
    P = len(cfg.patch_layers)
    R = cfg.n_layers - P
    c = {}
    c["reuse_bytes"] = R * T * (2 * (rr * cb + sb) + 2 * D * ob)
    c["reuse_bytes_written"] = R * T * 2 * D * ob
    c["reuse_flops"] = R * T * 4 * rr * D
    c["encode_bytes"] = R * T * (2 * D * ob + 2 * (rr * cb + sb)) + P * T * (d * ob + r * cb + sb)
    c["encode_flops"] = R * T * 4 * D * rr + P * T * 2 * d * r
    c["patch_flops"] = P * T * 2 * (r * d_a + d_a * d + 2 * d * D)
    c["patch_bytes"] = P * T * (r * cb + sb + 2 * D * ob)
    c["kv_bytes_written"] = cfg.n_layers * T * 2 * D * ob
    c["gemm2_flops_per_launch"] = T * 2 * d_a * d
    c["gemm3_flops_per_launch"] = T * 2 * d * 2 * D
    c["gemm1_flops_per_launch"] = T * 2 * r * d_a
    c["gemm1_bytes_per_layer"] = T * (r * cb + sb + d_a * ob)
    return c


# ------------------------------------------------------------------------------ oracle arm
def oracle_sample_rate(cfg, n_rows: int, seed: int = 0):
    """Time the oracle (as it stands) on `n_rows` sampled rows of the workload, all layers:
    encode + pack + reuse_decode + patch.  Returns (rows per second, seconds, threads)."""
    import numpy as np
    import torch
    from oracle import scd_oracle as O
    from paper_2606_07684_b200 import workloads as W
    try:
        from threadpoolctl import threadpool_info
        threads = max([i.get("num_threads", 1) for i in threadpool_info() if i.get("user_api") == "blas"] or [1])
    except Exception:
        threads = os.cpu_count() or 1
    n64 = lambda t: None if t is None else t.double().numpy()
    om = O.Model(n_layers=cfg.n_layers, d_model=cfg.d_model, n_kv_heads=cfg.n_kv_heads, head_dim=cfg.head_dim,
                 block_size=cfg.block_size, rope_theta_producer=cfg.rope_theta, rope_theta_consumer=cfg.rope_theta,
                 code_dtype=cfg.code_dtype, rms_eps=cfg.rms_eps)
    pos = np.random.default_rng(seed).integers(0, max(1, max(cfg.seqlens or (2048,))), n_rows)
    elapsed = 0.0
    for l in range(cfg.n_layers):
        a = W.make_layer_artifacts(cfg, l, "cpu", cal_rows=1024)      # untimed: calibration artifacts
        if a.kind == W.REUSE:
            lay = O.Layer(O.REUSE, enc_k=n64(a.enc_k), enc_v=n64(a.enc_v), dec_k=n64(a.dec_k), dec_v=n64(a.dec_v),
                          mean_src_k=n64(a.mean_k), mean_src_v=n64(a.mean_v), mean_dst_k=n64(a.mean_k), mean_dst_v=n64(a.mean_v))
            k, v = n64(W.make_state(cfg, l, 0, n_rows, "cpu")), n64(W.make_state(cfg, l, 1, n_rows, "cpu"))
            t0 = time.perf_counter()
            qk, sk = O.pack_codes(O.encode_k(om, lay, k, pos), om.code_dtype)
            qv, sv = O.pack_codes(O.encode_v(om, lay, v), om.code_dtype)
            O.reuse_decode_layer(om, lay, O.unpack_codes(qk, sk, om.code_dtype), O.unpack_codes(qv, sv, om.code_dtype), pos)
            elapsed += time.perf_counter() - t0
        else:
            lay = O.Layer(O.PATCH, enc_h=n64(a.enc_h), mean_src_h=n64(a.mean_h), w1=n64(a.w1), b1=n64(a.b1), w2=n64(a.w2),
                          norm_gamma=n64(a.gamma), w_k=n64(a.w_k), w_v=n64(a.w_v))
            h = n64(W.make_state(cfg, l, 2, n_rows, "cpu"))
            t0 = time.perf_counter()
            qh, sh = O.pack_codes(O.encode_h(om, lay, h), om.code_dtype)
            O.patch_layer(om, lay, O.unpack_codes(qh, sh, om.code_dtype), pos)
            elapsed += time.perf_counter() - t0
    return n_rows / elapsed, elapsed, threads


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores, each step a bounded row sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n_rows = args.ref_rows
    for _ in range(args.warmup):
        oracle_sample_rate(cfg, min(n_rows, 16))
    times, threads = [], 1
    for s in range(args.steps):
        rate, sec, threads = oracle_sample_rate(cfg, n_rows, seed=s)
        times.append(sec)
    sec = sum(times) / len(times)
    val = n_rows / sec
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "sample": f"{n_rows} seeded rows x all {cfg.n_layers} layers per step"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle",
                             "sample": f"{n_rows} rows x {cfg.n_layers} layers (encode+reuse_decode+patch), numpy fp64"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# ------------------------------------------------------------------------------ rank aggregation
def reduce_max_over_ranks(values, device="cpu"):
    """Element-wise MAX over ranks (times are reported as the slowest rank's); identity when
    torch.distributed is not initialised.  Works on gloo (CPU tests) and nccl."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def whole_job_throughput(tokens_per_rank: int, world: int, step_ms_max: float) -> float:
    """Replicas only: every rank rebuilds `tokens_per_rank` tokens per step; the job's rate is all
    ranks' tokens over the slowest rank's step time."""
    return tokens_per_rank * world / (step_ms_max * 1e-3)


# ------------------------------------------------------------------------------ beside the hot path
def run_extras(prob, cfg, k, v, peaks, flush, stream, iters=10):
    """Same-box numbers for the two SURVEY 8(f) items that sit beside the hot path (N = 1 only, outside the step):
    the group-wise INT4 comparison codec (the paper's fastest transport baseline) on the same
    geometry, and the GPU calibration fit (stack-SVD + ridge, Eq. 6-7) for one (layer, branch)."""
    import torch
    from paper_2606_07684_b200 import binding as B
    ev = lambda: torch.cuda.Event(enable_timing=True)
    out = {}
    if cfg.state_dtype != 1 or cfg.head_dim % 32:
        return out
    T, D, L = prob.T, cfg.D, cfg.n_layers
    dev = prob.device

    def timed(fn):
        fn(); fn()
        ts = []
        for _ in range(iters):
            flush.fill_(1)
            a, b = ev(), ev()
            a.record(stream); fn(); b.record(stream)
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return sum(ts) / len(ts), min(ts)

    # ---- INT4: every layer's K and V (the raw-KV transports ship all L layers; PATCH layers borrow a REUSE layer's
    # states as stand-ins, the kernels' work does not depend on the values)
    donor = next(l for l in range(L) if k[l] is not None)
    src = [t if t is not None else k[donor] for t in k] + [t if t is not None else v[donor] for t in v]
    pools = list(prob.k_pool) + list(prob.v_pool)
    for group in (32, 128):
        desc = B.Int4Desc(cfg.n_kv_heads, cfg.head_dim, cfg.block_size, group)
        stride_b, moff, total, payload = B.scd_int4_layout(desc, T, len(src))
        packed = torch.empty(total, dtype=torch.uint8, device=dev)
        q_ms, q_best = timed(lambda: B.scd_int4_quantize(desc, T, src, D, packed))
        d_ms, d_best = timed(lambda: B.scd_int4_dequantize_paged(desc, prob.bdesc, packed, pools, prob.batch.n_blocks))
        raw = len(src) * T * D * 2
        out[f"int4_g{group}"] = {
            "quantize_ms": q_ms, "dequantize_paged_ms": d_ms, "payload_bytes": payload, "scd_payload_bytes": prob.payload_bytes,
            "raw_kv_bytes": raw, "quantize_gbs": (raw + payload) / (q_ms * 1e-3) / 1e9,
            "dequantize_gbs": (raw + payload) / (d_ms * 1e-3) / 1e9,
            "quantize_frac_of_hbm_peak": (raw + payload) / (q_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
            "dequantize_frac_of_hbm_peak": (raw + payload) / (d_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
            "kv_tokens_per_s_dequantize": T / (d_ms * 1e-3), "tensors": len(src)}
        del packed
    # ---- encode with the producer's cache paged (identity table over the packed states: the same bytes, gathered)
    if T % cfg.block_size == 0 and not cfg.permute_pages and prob.per_head_rank == 0:
        h_src = [None] * L
        for l in cfg.patch_layers:
            h_src[l] = prob._bench_h[l]
        p_ms, p_best = timed(lambda: prob.encode(k, v, h_src, src_page_table=prob.batch.page_table, src_n_blocks=T // cfg.block_size))
        e_ms, e_best = timed(lambda: prob.encode(k, v, h_src))
        out["encode_paged_source"] = {"packed_ms": e_ms, "paged_ms": p_ms, "note": "K_A / V_A read through a producer page table (TMA: one 16-row box per page where rows align with pages, tile::gather4 otherwise)"}
    # ---- REUSE decode into fp8 pools (e4m3 bytes + one fp32 scale per (slot, head))
    if cfg.head_dim == 128 and D % 256 == 0:
        nb = prob.batch.n_blocks
        k8 = [torch.empty(nb, cfg.block_size, cfg.n_kv_heads, cfg.head_dim, dtype=torch.uint8, device=dev) for _ in range(L)]
        v8 = [torch.empty_like(t) for t in k8]
        ks = [torch.empty(nb, cfg.block_size, cfg.n_kv_heads, device=dev) for _ in range(L)]
        vs = [torch.empty_like(t) for t in ks]
        f_ms, f_best = timed(lambda: B.scd_reuse_decode(prob.plan, prob.bdesc, prob.codes, k8, v8, nb, k_scale=ks, v_scale=vs))
        R = L - len(cfg.patch_layers)
        cbytes = {0: 4, 1: 2, 2: 1}[cfg.code_dtype]
        fb = R * T * (2 * (cfg.rank * cbytes + (4 if cfg.code_dtype == 2 else 0)) + 2 * (D + 4 * cfg.n_kv_heads))
        out["reuse_decode_fp8_pools"] = {"ms": f_ms, "algorithmic_bytes": fb, "gbs": fb / (f_ms * 1e-3) / 1e9,
                                         "frac_of_hbm_peak": fb / (f_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                                         "kv_tokens_per_s": T / (f_ms * 1e-3)}
        del k8, v8, ks, vs
    # ---- calibration fit of one (layer, branch): A, B = two layers' K states (paired samples stand-in)
    others = [l for l in range(L) if k[l] is not None]
    if len(others) >= 2 and D <= 1024:
        a_s, b_s = k[others[0]].view(T, D), k[others[1]].view(T, D)
        desc = B.FitDesc(D, cfg.rank, 1, 1e-3, B.SCD_BF16, B.SCD_BF16)
        ws = torch.empty(B.scd_fit_query(desc, T), dtype=torch.uint8, device=dev)
        w_enc = torch.empty(D, cfg.rank, dtype=torch.bfloat16, device=dev)
        w_dec = torch.empty(cfg.rank, D, dtype=torch.bfloat16, device=dev)
        mu_a, mu_b = torch.empty(D, device=dev), torch.empty(D, device=dev)
        sig = torch.empty(cfg.rank, device=dev)
        B.profile_enable(True)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        sweeps = B.scd_fit_reuse(desc, a_s, b_s, T, D, w_enc, None, w_dec, mu_a, mu_b, sig, ws)
        torch.cuda.synchronize()
        fit_s = time.perf_counter() - t0
        gram = [ms for kid, ms in B.profile_fetch() if kid == 300]
        B.profile_enable(False)
        gram_ms = gram[0] if gram else None
        np_ = (T + 63) // 64 * 64
        mt_, nt_ = (2 * D + 127) // 128, (2 * D + 255) // 256
        kept_frac = sum(min(mt_, 2 * tn + 2) for tn in range(nt_)) / float(mt_ * nt_)
        # the same fit on 10^5 paired rows (the states repeated: the eigen-problem is the same, the Gram pass is 12 x longer)
        big = None
        try:
            reps = (100000 + T - 1) // T
            a_b, b_b = a_s.repeat(reps, 1)[:100000].contiguous(), b_s.repeat(reps, 1)[:100000].contiguous()
            ws_b = torch.empty(B.scd_fit_query(desc, 100000), dtype=torch.uint8, device=dev)
            B.profile_enable(True)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            sw_b = B.scd_fit_reuse(desc, a_b, b_b, 100000, D, w_enc, None, w_dec, mu_a, mu_b, sig, ws_b)
            torch.cuda.synchronize()
            big_s = time.perf_counter() - t0
            g_b = [ms for kid, ms in B.profile_fetch() if kid == 300]
            B.profile_enable(False)
            big = {"rows": 100000, "seconds": big_s, "jacobi_sweeps": list(sw_b), "gram_ms": g_b[0] if g_b else None,
                   "gram_tflops_full_matrix_equivalent": (2.0 * (2 * D) ** 2 * 100032 / (g_b[0] * 1e-3) / 1e12) if g_b else None,
                   "gram_tflops_executed": (kept_frac * 2.0 * (2 * D) ** 2 * 100032 / (g_b[0] * 1e-3) / 1e12) if g_b else None}
            del a_b, b_b, ws_b
        except Exception as e:
            big = {"error": f"{type(e).__name__}: {e}"}
        out["calibration_fit"] = {
            "at_1e5_rows": big,
            "rows": T, "width": D, "rank": cfg.rank, "seconds": fit_s, "jacobi_sweeps": list(sweeps), "gram_ms": gram_ms,
            "gram_tflops_full_matrix_equivalent": (2.0 * (2 * D) ** 2 * np_ / (gram_ms * 1e-3) / 1e12) if gram_ms else None,
            "gram_tflops_executed": (kept_frac * 2.0 * (2 * D) ** 2 * np_ / (gram_ms * 1e-3) / 1e12) if gram_ms else None,
            "gram_note": "G is symmetric: only the 128 x 256 tiles touching the upper triangle are computed (kept fraction below)",
            "gram_tiles_kept_fraction": kept_frac,
            "paper_reuse_fitting_s_all_layers": 905.5,
            "note": "one (layer, branch); wall clock incl. one host sync per Jacobi sweep; the paper's figure is for all layers of a 7B pair on its GPU (PAPER.md:602)"}
    return out


def run_other_configs(args):
    from paper_2606_07684_b200 import workloads as W
    out = {}
    for name in W.CONFIG_ORDER:
        if name == "llama3_8b_8k":
            continue
        cmd = [sys.executable, os.path.abspath(__file__), "--config", name, "--no-e2e", "--no-cpu-baseline", "--no-extras",
               "--no-other-configs", "--steps", "5", "--warmup", "3"]
        try:
            r = subprocess.run(cmd, capture_output=True, text=True, timeout=600)
            d = json.loads(r.stdout.strip().splitlines()[-1])
            out[name] = {"value": d["value"], "unit": d["unit"], "ms_per_step": d["ms_per_step"], "stages_ms": d["stages_ms"],
                         "kv_tokens_per_s_reuse_plus_patch": d["kv_tokens_per_s_reuse_plus_patch"], "config": d["config"],
                         "clocks": d["clocks"], "gpu_launches": d["gpu_launches"],
                         "rooflines": {k_: {x: v_[x] for x in ("bound", "achieved", "peak", "unit", "frac", "ms") if x in v_}
                                       for k_, v_ in d["rooflines"].items()}}
        except Exception as e:                                   # a side run never takes the headline line down
            out[name] = {"error": f"{type(e).__name__}: {e}"}
    return out


# ------------------------------------------------------------------------------ our arm
def run_ours(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_2606_07684_b200 import binding as B
    from paper_2606_07684_b200.harness import CodecProblem

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("NCCL_DEBUG", "WARN")          # keep NCCL's communicator messages in the log
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = torch.device(f"cuda:{local}")
    torch.cuda.set_device(dev)

    prob = CodecProblem(cfg, dev, per_head_rank=args.per_head_rank)
    T = prob.T
    k, v, h = prob.make_sources()          # content-space states stand in for the post-RoPE cache
    prob.alloc_pools()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def one_step(timed):
        """encode -> decode -> patch with L2 flushed before each call; returns per-call ms."""
        evs = []
        launches = 0
        for fn in (lambda: prob.encode(k, v, h), prob.reuse_decode, prob.patch):
            flush.fill_(1)
            a, b = ev(), ev()
            a.record(stream)
            launches += fn()
            b.record(stream)
            evs.append((a, b))
        return evs, launches

    for _ in range(max(args.warmup, 3)):
        one_step(False)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    t_wall = time.perf_counter()
    all_evs, launches = [], 0
    for _ in range(args.steps):
        evs, n = one_step(True)
        all_evs.append(evs)
        launches += n
    barrier()
    t_wall = time.perf_counter() - t_wall
    per_call = [[a.elapsed_time(b) for a, b in evs] for evs in all_evs]
    enc_ms, dec_ms, pat_ms = (sum(c[i] for c in per_call) / len(per_call) for i in range(3))
    step_ms = enc_ms + dec_ms + pat_ms

    # ---- per-kernel times (events inside the library, same stream), for the roofline ----
    B.profile_enable(True)
    for _ in range(min(args.steps, 5)):
        one_step(False)
    torch.cuda.synchronize()
    recs = B.profile_fetch()
    B.profile_enable(False)
    by_kernel = {}
    for kid, ms in recs:
        by_kernel.setdefault(kid, []).append(ms)

    # ---- optional: layer-streamed pipeline (scd_*_layers) ----
    # Producer encodes a group of layers, the group's code segments cross a stand-in link (device-to-device copy into
    # the consumer's code buffer), the consumer decodes / patches the group -- on three streams, against the same four
    # steps run whole and back to back.  One GPU plays both sides, so only the copy can truly overlap.
    streamed = None
    if args.stream_layers > 0:
        G, L = args.stream_layers, cfg.n_layers
        segs = {l: [prob.plan.code_segment(l, br, T) for br in ((2,) if l in cfg.patch_layers else (0, 1))] for l in range(L)}
        cb = {0: 4, 1: 2, 2: 1}[cfg.code_dtype]
        rx_codes = torch.zeros_like(prob.codes)

        def link(l0, l1):
            for l in range(l0, l1):
                for off, soff, r in segs[l]:
                    n = T * r * cb
                    rx_codes[off:off + n].copy_(prob.codes[off:off + n], non_blocking=True)
                    if cfg.code_dtype == 2:
                        rx_codes[soff:soff + 4 * T].copy_(prob.codes[soff:soff + 4 * T], non_blocking=True)

        s_link, s_rx = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
        tx_codes = prob.codes

        def whole():
            prob.codes = tx_codes
            prob.encode(k, v, h)
            link(0, L)
            prob.codes = rx_codes
            prob.reuse_decode(); prob.patch()
            prob.codes = tx_codes

        def pipelined():
            for l0 in range(0, L, G):
                l1 = min(L, l0 + G)
                prob.codes = tx_codes
                prob.encode(k, v, h, layers=(l0, l1))
                e1 = ev(); e1.record(stream)
                s_link.wait_event(e1)
                with torch.cuda.stream(s_link):
                    link(l0, l1)
                    e2 = ev(); e2.record(s_link)
                s_rx.wait_event(e2)
                prob.codes = rx_codes
                prob.reuse_decode(stream=s_rx, layers=(l0, l1))
                prob.patch(stream=s_rx, layers=(l0, l1))
            prob.codes = tx_codes
            e3 = ev(); e3.record(s_rx)
            stream.wait_event(e3)

        res = {}
        for name_, fn_ in (("whole_calls_ms", whole), ("pipelined_ms", pipelined)):
            fn_(); fn_()
            torch.cuda.synchronize()
            a, b = ev(), ev()
            a.record(stream)
            for _ in range(5):
                fn_()
            b.record(stream)
            torch.cuda.synchronize()
            res[name_] = a.elapsed_time(b) / 5
        streamed = {"layers_per_group": G, **res, "link": "device-to-device copy of the group's code segments"}

    # ---- e2e: host buffers in, host buffers out ----
    e2e = None
    if not args.no_e2e:
        # Every step copies its inputs host -> device from pinned memory, runs the three C-ABI calls and copies the
        # pools device -> host.  Inputs and pools are double-buffered and the copies run on their own streams, so
        # step i's D2H and step i+1's H2D overlap (PCIe is full duplex) with step i+1's compute waiting only on
        # its own inputs; every step's copies are inside the timed region.
        # The per-layer tensors the C ABI takes are views into ONE device slab per direction (and the host side is one
        # pinned buffer per direction), so a step's transfer is one copy each way: 67 per-tensor copies each way reach
        # 41.6 GB/s per direction on this box, one copy 50 GB/s (both directions busy).
        def slab_views(ts):
            nb = [0 if t is None else (t.numel() * t.element_size() + 255) // 256 * 256 for t in ts]
            slab = torch.empty(sum(nb), dtype=torch.uint8, device=dev)
            views, off = [], 0
            for t, n in zip(ts, nb):
                if t is None:
                    views.append(None)
                    continue
                vw = slab[off:off + t.numel() * t.element_size()].view(t.dtype).view(t.shape)
                vw.copy_(t)
                views.append(vw)
                off += n
            return slab, views
        sets = []
        for _ in range(2):
            src_slab, sv = slab_views(list(k) + list(v) + list(h))
            pool_slab, pv = slab_views(list(prob.k_pool) + list(prob.v_pool))
            L_ = len(k)
            sets.append({"k": sv[:L_], "v": sv[L_:2 * L_], "h": sv[2 * L_:], "kp": pv[:len(prob.k_pool)], "vp": pv[len(prob.k_pool):],
                         "src_slab": src_slab, "pool_slab": pool_slab})
        host_in = torch.empty(sets[0]["src_slab"].shape, dtype=torch.uint8, pin_memory=True).copy_(sets[0]["src_slab"])
        host_out = torch.empty(sets[0]["pool_slab"].shape, dtype=torch.uint8, pin_memory=True)
        h2d = sum(t.numel() * t.element_size() for t in (list(k) + list(v) + list(h)) if t is not None)
        d2h = sum(p.numel() * p.element_size() for p in (list(prob.k_pool) + list(prob.v_pool)) if p is not None)
        orig_pools = (prob.k_pool, prob.v_pool)
        s_in, s_out = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
        in_done, comp_done, out_done = [ev(), ev()], [ev(), ev()], [ev(), ev()]

        def e2e_step(i):
            st, bi = sets[i % 2], i % 2
            if i >= 2:
                s_in.wait_event(comp_done[bi])            # step i-2 has consumed this input buffer
            with torch.cuda.stream(s_in):
                st["src_slab"].copy_(host_in, non_blocking=True)
                in_done[bi].record(s_in)
            stream.wait_event(in_done[bi])
            if i >= 2:
                stream.wait_event(out_done[bi])           # step i-2's pools have been read back
            prob.k_pool, prob.v_pool = st["kp"], st["vp"]
            prob.encode(st["k"], st["v"], st["h"]); prob.reuse_decode(); prob.patch()
            comp_done[bi].record(stream)
            s_out.wait_event(comp_done[bi])
            with torch.cuda.stream(s_out):
                host_out.copy_(st["pool_slab"], non_blocking=True)
                out_done[bi].record(s_out)

        e2e_step(0); e2e_step(1)
        torch.cuda.synchronize()
        barrier()
        a, b = ev(), ev()
        n_e2e = max(4, args.steps)                 # the same K steps as the device-timed region (pipeline fill and drain included)
        a.record(stream)
        for i in range(n_e2e):
            e2e_step(i + 2)
        stream.wait_event(out_done[0]); stream.wait_event(out_done[1])
        b.record(stream)
        barrier()
        e2e_ms = a.elapsed_time(b) / n_e2e
        prob.k_pool, prob.v_pool = orig_pools
        del sets, host_in, host_out
        e2e = {"ms": e2e_ms, "h2d": h2d, "d2h": d2h}
    clocks = sampler.stop() if sampler else None
    extras = None
    if world == 1 and not args.no_extras:
        prob._bench_h = h
        extras = run_extras(prob, cfg, k, v, load_peaks(), flush, stream)

    # ---- max over ranks ----
    step_ms, enc_ms, dec_ms, pat_ms, e2e_ms = reduce_max_over_ranks(
        [step_ms, enc_ms, dec_ms, pat_ms, e2e["ms"] if e2e else 0.0], dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks = load_peaks()
    costs = workload_costs(cfg, T, cfg.n_kv_heads * args.per_head_rank if args.per_head_rank else None)
    # DRAM bytes per launch from the committed `ncu --set full` captures (profiles/): {kernel: bytes}
    traffic = {}
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(tpath):
        for ln in open(tpath).read().splitlines()[1:]:
            f = [x.strip() for x in ln.split(",")]
            if len(f) >= 3 and f[0] == cfg.name:
                traffic[f[1]] = float(f[2])
    tokens = T * world
    value = whole_job_throughput(T, world, step_ms)

    # dominant kernel of the step = largest total time over the profiled passes
    tot = {kid: sum(v_) for kid, v_ in by_kernel.items()}
    dom = max(tot, key=tot.get) if tot else None
    rooflines = {}
    n_prof = max(1, min(args.steps, 5))
    for kid, ts in by_kernel.items():
        avg_ms = sum(ts) / len(ts)
        per_pass = len(ts) / n_prof
        if kid == 110:      # REUSE decode: one launch per call (per rank run), HBM-bound
            # one launch per call (all REUSE segments of equal rank): the call's own events in the timed region
            # are the kernel's duration; several launches: sum of the in-library per-launch events
            call_ms = dec_ms if per_pass == 1 else avg_ms * per_pass
            ach = costs["reuse_bytes"] / (call_ms * 1e-3) / 1e9
            wr = costs["reuse_bytes_written"] / (call_ms * 1e-3) / 1e9
            rooflines["reuse_decode"] = {"kernel": KERNEL_NAMES[kid], "bound": "hbm", "achieved": ach,
                                         "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": ach / peaks["hbm_gbs"],
                                         "traffic": traffic.get("reuse_decode"), "ms": call_ms,
                                         "share_of_step": call_ms / step_ms, "write_gbs": wr}
            # t_roof = max(FLOP / P_tensor, bytes / P_hbm) -- wide ranks (r >= 256) are tensor-bound
            t_hbm = costs["reuse_bytes"] / (peaks["hbm_gbs"] * 1e9)
            t_tc = costs["reuse_flops"] / (peaks["bf16_tflops"] * 1e12)
            if t_tc > t_hbm:
                ach_tf = costs["reuse_flops"] / (call_ms * 1e-3) / 1e12
                rooflines["reuse_decode"].update({"bound": "tensor", "achieved": ach_tf, "peak": peaks["bf16_tflops"], "unit": "TFLOP/s",
                                                  "frac": ach_tf / peaks["bf16_tflops"], "hbm_gbs": ach, "frac_of_hbm_peak": ach / peaks["hbm_gbs"]})
        elif kid in (120, 130, 140):
            # PATCH GEMM-1 / GEMM-2 / GEMM-3: a launch covers a group of PATCH layers (one segment per layer), so the
            # algorithmic FLOPs per launch are the per-layer figure x layers per launch; `ms` is the launch average
            name = {120: "patch_gemm1", 130: "patch_gemm2", 140: "patch_gemm3"}[kid]
            per_layer = costs[{120: "gemm1_flops_per_launch", 130: "gemm2_flops_per_launch", 140: "gemm3_flops_per_launch"}[kid]]
            layers_per_launch = len(cfg.patch_layers) / per_pass
            if kid == 120:      # K = r is small: the write of the [T, d_a] activation bounds GEMM-1
                ach = costs["gemm1_bytes_per_layer"] * layers_per_launch / (avg_ms * 1e-3) / 1e9
                rooflines[name] = {"kernel": KERNEL_NAMES[kid], "bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"],
                                   "unit": "GB/s", "frac": ach / peaks["hbm_gbs"], "traffic": traffic.get(name),
                                   "ms": avg_ms, "layers_per_launch": layers_per_launch,
                                   "share_of_step": avg_ms * per_pass / step_ms}
                continue
            ach = per_layer * layers_per_launch / (avg_ms * 1e-3) / 1e12
            rooflines[name] = {"kernel": KERNEL_NAMES[kid], "bound": "tensor", "achieved": ach,
                               # each launch is timed on its own (events around it, a 0.3-0.6 ms kernel after an L2
                               # flush): the burst figure is the peak that applies; the sustained one is reported beside it
                               "peak": peaks["bf16_tflops"], "unit": "TFLOP/s",
                               "frac": ach / peaks["bf16_tflops"], "frac_of_sustained_peak": ach / peaks["bf16_tflops_sustained"],
                               "traffic": traffic.get(name), "ms": avg_ms,
                               "layers_per_launch": layers_per_launch, "share_of_step": avg_ms * per_pass / step_ms}
        elif kid in (100, 101):
            pass
    if enc_ms > 0:
        ach = costs["encode_bytes"] / (enc_ms * 1e-3) / 1e9
        rooflines["encode_call"] = {"kernel": "scd_encode (all launches)", "bound": "hbm", "achieved": ach,
                                    "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": ach / peaks["hbm_gbs"],
                                    "traffic": None, "ms": enc_ms, "share_of_step": enc_ms / step_ms}
        t_tc = costs["encode_flops"] / (peaks["bf16_tflops"] * 1e12)
        if t_tc > costs["encode_bytes"] / (peaks["hbm_gbs"] * 1e9):
            ach_tf = costs["encode_flops"] / (enc_ms * 1e-3) / 1e12
            rooflines["encode_call"].update({"bound": "tensor", "achieved": ach_tf, "peak": peaks["bf16_tflops"], "unit": "TFLOP/s",
                                             "frac": ach_tf / peaks["bf16_tflops"], "hbm_gbs": ach, "frac_of_hbm_peak": ach / peaks["hbm_gbs"]})
    dom_key = max(rooflines, key=lambda n: rooflines[n]["share_of_step"]) if rooflines else None
    roofline = dict(rooflines[dom_key]) if dom_key else None
    if roofline:
        roofline["name"] = dom_key
        roofline["peak_source"] = peaks["source"] + (" burst bf16 (kernel timed alone)" if roofline["bound"] == "tensor" else " copy")

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16" if cfg.state_dtype == 1 else "f32", "data": "synthetic",
        "config": {"workload": cfg.name, "tokens": T, "layers": cfg.n_layers, "patch_layers": list(cfg.patch_layers),
                   "rank": cfg.rank, "reuse_per_head_rank": args.per_head_rank or None, "code_dtype": {0: "f32", 1: "bf16", 2: "e4m3+f32 rowscale"}[cfg.code_dtype],
                   "l2": "flushed (256 MiB fill) before every C-ABI call, outside the events; inputs 2.2 GB >> L2",
                   "parallelism": "replicas only" if world > 1 else "1 gpu"},
        "stages_ms": {"encode": enc_ms, "reuse_decode": dec_ms, "patch": pat_ms},
        "kv_tokens_per_s_reuse_plus_patch": tokens / ((dec_ms + pat_ms) * 1e-3),
        "kv_gbs_written": costs["kv_bytes_written"] * world / ((dec_ms + pat_ms) * 1e-3) / 1e9,
        "reuse_decode_tokens_per_s": tokens / (dec_ms * 1e-3) if dec_ms else None,
        "gpu_launches": launches, "wall_s_timed_region": t_wall, "layer_streamed": streamed,
        "clocks": clocks, "roofline": roofline, "rooflines": rooflines,
    }
    if extras:
        line["beside_the_hot_path"] = extras
    if world == 1 and args.config == "llama3_8b_8k" and not args.no_other_configs and not args.rank and not args.per_head_rank:
        # the other BASELINE configs (parity-test cases, not the headline): stage times and roofline fractions, each run
        # by this same script in a process of its own after this one has released the GPU's memory
        del prob, k, v, h, flush
        torch.cuda.empty_cache()
        line["other_configs"] = run_other_configs(args)
    if e2e:
        line["e2e"] = {"value": tokens / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": e2e["h2d"],
                       "d2h_bytes_per_step": e2e["d2h"], "ms_per_step": e2e_ms}
    if world == 1 and not args.no_cpu_baseline:
        rate, sec, threads = oracle_sample_rate(cfg, args.ref_rows)
        line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": threads, "kind": "oracle",
                                "sample": f"{args.ref_rows} seeded rows x all {cfg.n_layers} layers "
                                          f"(encode+reuse_decode+patch), numpy fp64, {sec:.1f} s"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="llama3_8b_8k")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-rows", type=int, default=4096)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the short runs of the other BASELINE configs")
    ap.add_argument("--no-extras", action="store_true", help="skip the INT4 comparison codec and the calibration-fit timings")
    ap.add_argument("--rank", type=int, default=0, help="override the config's rank (config 5 rank sweep)")
    ap.add_argument("--stream-layers", type=int, default=0,
                    help="also time the layer-streamed pipeline (scd_*_layers) with this many layers per group")
    ap.add_argument("--per-head-rank", type=int, default=0,
                    help="REUSE layers in the paper's per-head reading (one d_h x r map per layer, PAPER.md:102) with this r")
    args = ap.parse_args()
    from paper_2606_07684_b200 import workloads as W
    cfg = W.CONFIGS[args.config]
    if args.rank:
        cfg = cfg.scaled(rank=args.rank)
    if args.impl == "reference":
        run_reference(args, cfg)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started as plain `python bench.py --gpus N`: start the N ranks ourselves (one process per GPU), exactly as the
        # driver would; rank 0 prints the line
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    import __graft_entry__ as ge
    ge.build()
    run_ours(args, cfg)


if __name__ == "__main__":
    main()
