"""GPU parity: the CUDA path behind the C ABI vs the fp64 oracle, element by element on the
same seeded inputs (SURVEY.md 8(c) protocol).  Tolerances (BASELINE.json north_star):
rel. Frobenius per layer <= 2e-2 for bf16 outputs, <= 1e-5 for fp32; page / slot indexing
bit-exact (sentinel-filled pools)."""
import numpy as np
import pytest
import torch

from oracle import scd_oracle as O
from paper_2606_07684_b200 import workloads as W
from tests import _parity as P

pytestmark = pytest.mark.gpu

C = W.CONFIGS
# oracle-sized versions of BASELINE configs 2-5: same head geometry / dtypes / rank / page size,
# fewer layers and tokens; lengths chosen to span several 128-row tiles and a ragged tail
MINI = {
    "tiny": C["tiny"],
    "llama3_8b_8k": C["llama3_8b_8k"].scaled(n_layers=4, patch_layers=(1,), seqlens=(1000,), d_model=1024),
    "llama3_8b_ragged": C["llama3_8b_ragged"].scaled(n_layers=3, patch_layers=(1,), ragged_range=(6, 20, 300),
                                                     d_model=512),
    "mistral_7b_32k_fp8": C["mistral_7b_32k_fp8"].scaled(n_layers=3, patch_layers=(2,), seqlens=(700,), d_model=1024),
    "llama3_70b_2x16k": C["llama3_70b_2x16k"].scaled(n_layers=3, patch_layers=(0,), seqlens=(300, 333), d_model=2048),
}


def _problem(cfg, device, **kw):
    from paper_2606_07684_b200.harness import CodecProblem
    # small cases draw their inputs and fit their bases on the host: only the codec's kernels launch on the device
    small = cfg.d_model <= 1024 and (sum(cfg.seqlens) if cfg.seqlens else 8192) <= 4096
    kw.setdefault("gen_device", "cpu" if small else None)
    return CodecProblem(cfg, device, **kw)


def _run_all(prob, rows=None, roped=True):
    """encode -> reuse_decode -> patch, each checked against the oracle on the same bits."""
    k, v, h = prob.make_sources()
    if roped and prob.model.k_is_roped:
        k = P.roped_producer_k(prob, k)
    prob.alloc_pools()
    prob.encode(k, v, h)
    torch.cuda.synchronize()
    enc = P.check_encode(prob, k, v, h, rows)
    reuse = [l for l in range(prob.cfg.n_layers) if prob.arts[l].kind == W.REUSE]
    patch = [l for l in range(prob.cfg.n_layers) if prob.arts[l].kind == W.PATCH]
    prob.reuse_decode()
    torch.cuda.synchronize()
    slots = O.slot_mapping(P.oracle_batch(prob), prob.cfg.block_size)
    P.check_untouched(prob, reuse, slots, also_untouched_layers=patch)     # REUSE call leaves PATCH layers alone
    dec = P.check_reuse_decode(prob, rows)
    prob.patch()
    torch.cuda.synchronize()
    P.check_untouched(prob, reuse + patch, slots)
    pat = P.check_patch(prob, rows)
    P.check_reuse_decode(prob, rows)                                       # and PATCH left REUSE layers alone
    # nothing outside the code segments / scale segments / workspace was written (padding, tails, guards)
    assert prob.guard_violations() == (0, 0), f"guard bytes overwritten (code buffer, workspace): {prob.guard_violations()}"
    used = {k_: round(v_, 3) for d_ in (enc, dec, pat) for k_, v_ in d_.items() if k_ not in ("worst_rel_fro", "slots")}
    return {"encode": enc["worst_rel_fro"], "reuse": dec["worst_rel_fro"], "patch": pat["worst_rel_fro"], "bounds_used": used}


@pytest.mark.parametrize("name", list(MINI))
def test_config_parity(name, cuda_device):
    prob = _problem(MINI[name], cuda_device)
    res = _run_all(prob)
    print(name, res)


def test_tiny_round_trip_matches_truncation_closed_form(cuda_device):
    """Encode -> decode of V equals the rank-r truncation: ||X - X^||_F^2 = sum_{i>r} sigma_i^2
    (Eckart-Young), sigma from numpy's SVD of the centred input bits; and the
    round trip of K returns the roped K up to the same truncation."""
    cfg = C["tiny"]
    prob = _problem(cfg, cuda_device)
    k, v, h = prob.make_sources()
    kr = P.roped_producer_k(prob, k)
    prob.alloc_pools()
    prob.encode(kr, v, h)
    prob.reuse_decode()
    torch.cuda.synchronize()
    slots = O.slot_mapping(P.oracle_batch(prob), cfg.block_size)
    for l in (0, 1, 2):
        for src, pool, mu in ((v[l], prob.v_pool[l], prob.arts[l].mean_v), (k[l], prob.k_pool[l], prob.arts[l].mean_k)):
            x = P.np64(src)
            s = np.linalg.svd(x - P.np64(mu)[None, :], compute_uv=False)
            want = np.sqrt((s[cfg.rank:] ** 2).sum())
            y = P._gather(pool, slots)
            if pool is prob.k_pool[l]:      # compare in content space: deRoPE the reconstruction with the oracle
                y = O.rope(y, O.positions(P.oracle_batch(prob)), cfg.rope_theta, -1, cfg.n_kv_heads, cfg.head_dim)
            got = np.linalg.norm(x - y)
            assert abs(got - want) <= 2e-4 * want, (l, got, want)
            # population value quoted in SURVEY 8(c): ~0.073 relative for Tiny, r = 32
            assert 0.05 < got / np.linalg.norm(x - P.np64(mu)[None, :]) < 0.10


def test_e4m3_operand_expansion_is_exact_for_every_code(cuda_device):
    """The tcgen05 path widens e4m3 codes to bf16 in shared memory; that must be exact for all 254 finite
    codes, subnormals included (a flush-to-zero would wipe rows made of small codes only).  Hand-written
    code bytes and power-of-two scales go through scd_reuse_decode; each output element must agree with
    the oracle (same code bits) to bf16 output rounding."""
    cfg = MINI["mistral_7b_32k_fp8"].scaled(n_layers=1, patch_layers=(), seqlens=(256,))
    prob = _problem(cfg, cuda_device, use_means=False)
    prob.alloc_pools()
    finite = np.array([b for b in range(256) if (b & 0x7F) != 0x7F], dtype=np.uint8)
    small = np.array([b for b in range(256) if (b & 0x78) == 0], dtype=np.uint8)       # zero + subnormals, both signs
    rng = np.random.default_rng(0)
    for br in (O.BRANCH_K, O.BRANCH_V):
        q, s = prob.code_view(0, br)
        T, r = q.shape
        codes = np.empty((T, r), np.uint8)
        for t in range(T):
            pool = small if t % 4 == 3 else finite            # every 4th row: small codes only
            codes[t] = np.roll(np.resize(pool, r), t)
        q.copy_(torch.from_numpy(codes).to(cuda_device))
        s.copy_(torch.from_numpy((2.0 ** rng.integers(-6, 3, T)).astype(np.float32)).to(cuda_device))
    prob.reuse_decode()
    torch.cuda.synchronize()
    om, ob = P.oracle_model(prob), P.oracle_batch(prob)
    pos, slots = O.positions(ob), O.slot_mapping(ob, om.block_size)
    ol = P.oracle_layer(prob, 0)
    qk, sk = P.gpu_codes(prob, 0, O.BRANCH_K)
    qv, sv = P.gpu_codes(prob, 0, O.BRANCH_V)
    zk, zv = O.unpack_codes(qk, sk, om.code_dtype), O.unpack_codes(qv, sv, om.code_dtype)
    k_o, v_o = O.reuse_decode_layer(om, ol, zk, zv, pos)
    for name, z, dec, want, pool in (("K", zk, ol.dec_k, k_o, prob.k_pool[0]), ("V", zv, ol.dec_v, v_o, prob.v_pool[0])):
        got = P._gather(pool, slots)
        # bf16 output rounding (2^-9 relative) + fp32 accumulation of r products (and the RoPE mix for K)
        bound = 2.0 ** -8 * np.abs(want) + 1e-5 * (np.abs(z) @ np.abs(dec)) + 1e-30
        if name == "K":
            bound = bound + 2.0 ** -8 * np.sqrt((want.reshape(len(want), -1, cfg.head_dim) ** 2).sum(-1)).repeat(cfg.head_dim, axis=1)
        bad = np.abs(got - want) > bound
        assert not bad.any(), f"{name}: {int(bad.sum())} elements off, first at {np.argwhere(bad)[0]}"
        assert np.abs(want[3::4]).max() > 0          # the small-code rows are not trivially zero


@pytest.mark.parametrize("name,r_h", [("tiny", 8), ("llama3_8b_8k", 16), ("llama3_8b_8k", 24), ("llama3_8b_8k", 32),
                                       ("llama3_8b_8k", 64), ("llama3_8b_ragged", 16), ("mistral_7b_32k_fp8", 32)])
def test_per_head_reuse_mode(name, r_h, cuda_device):
    """The paper's own Sec. 4.1 translator: one d_h x r map per layer and branch shared by all
    KV heads, heads flattened into the sample axis (scd_model_desc_t.reuse_per_head).  The code row of a token is
    H * r wide; the decode kernel skips the zero blocks of I_H (x) W (k-block range per n-tile), which r = 24 / 32 / 64
    exercise with ranges that straddle, equal and span k-blocks."""
    prob = _problem(MINI[name], cuda_device, per_head_rank=r_h)
    assert prob.plan.code_segment(0, 0, prob.T)[2] == MINI[name].n_kv_heads * r_h
    res = _run_all(prob)
    print(name, r_h, res)


@pytest.mark.parametrize("rank", [96, 192])
def test_ranks_that_are_not_powers_of_two(rank, cuda_device):
    """Tile widths that are not powers of two (the encode tile is the rank rounded up to 16).  192 = two 96-column
    warp groups once had its copy-out overwrite the neighbouring group's first 32 columns (sporadic NaNs)."""
    cfg = MINI["llama3_8b_8k"].scaled(rank=rank, seqlens=(700,), n_layers=2, patch_layers=(1,))
    _run_all(_problem(cfg, cuda_device))


@pytest.mark.parametrize("rank", [32, 64, 128, 256, 512])
def test_config5_rank_sweep_mini(rank, cuda_device):
    """BASELINE.json configs[4] sweeps the per-layer rank over {32, 64, 128, 256, 512}: every one of them on config-5
    geometry (2 requests, REUSE layers and one PATCH layer).  r = 256 fills the encode's widest tile; r = 512 is the
    distinct path where a segment's codes span two 256-wide n-tiles of the encode and the decode runs K = 512
    (8 k-blocks)."""
    cfg = MINI["llama3_70b_2x16k"].scaled(rank=rank, seqlens=(300, 333), n_layers=3, patch_layers=(1,), d_model=2048)
    res = _run_all(_problem(cfg, cuda_device))
    print(rank, res)


@pytest.mark.parametrize("rank,d_model", [(16, 1024), (48, 1024), (48, 80), (80, 1024), (112, 528)])
def test_tile_widths_that_are_not_multiples_of_32_on_dirty_tmem(rank, d_model, cuda_device):
    """The epilogue reads TMEM 32 columns at a time and TMEM is not cleared between kernels: a tile narrower than the
    last chunk it reads (e4m3 rank 16 / 48 / 80 / 112 in the row-amax pass; d_model = 80 / 528 in GEMM-2's row sum of
    squares) must not pick up a previous kernel's accumulators.  A 256-column decode runs first, so every SM's TMEM
    holds large stale values; a stale value in the amax would show as a wrong e4m3 scale, in the sum of squares as a
    wrong RMS scale of the PATCH layer."""
    dirty = _problem(MINI["llama3_8b_8k"].scaled(n_layers=1, patch_layers=(), seqlens=(2048,)), cuda_device)
    k, v, h = dirty.make_sources()
    dirty.alloc_pools()
    dirty.encode(k, v, h)
    q, _ = dirty.code_view(0, 0)
    q.mul_(1e4)                                                   # large accumulators left behind in TMEM
    dirty.reuse_decode()
    cfg = MINI["mistral_7b_32k_fp8"].scaled(rank=rank, d_model=d_model, n_layers=2, patch_layers=(1,), seqlens=(300,),
                                            spectrum_k=min(512, d_model))
    res = _run_all(_problem(cfg, cuda_device))
    print(rank, d_model, res)


def test_plan_built_on_a_non_blocking_stream(cuda_device):
    """scd_plan enqueues its zero-fills and repacks on the caller's stream; on a non-blocking stream (every
    torch.cuda.Stream) a legacy-stream memset would be unordered with them and could wipe artifacts.  Busy work on the
    default stream makes a misordering likely to show."""
    from paper_2606_07684_b200.harness import CodecProblem
    cfg = MINI["llama3_8b_8k"].scaled(n_layers=3, patch_layers=(1,), seqlens=(300,), d_model=512)
    side = torch.cuda.Stream(device=cuda_device)
    busy = torch.randn(4096, 4096, device=cuda_device)
    for _ in range(20):
        busy = busy @ busy * 1e-3                                 # keeps the default (blocking) stream occupied
    with torch.cuda.stream(side):
        prob = CodecProblem(cfg, cuda_device)                    # plan on `side` (the binding passes the current stream)
        res = _run_all(prob)
    torch.cuda.synchronize()
    print(res)


def test_page_ids_outside_the_pool_are_skipped_not_written(cuda_device):
    """Page tables live on the device, so the host cannot validate them (include/scd.h): a row whose page id is -1 or
    >= n_blocks is left unwritten -- never a store outside the pool."""
    cfg = MINI["llama3_8b_8k"].scaled(n_layers=2, patch_layers=(1,), seqlens=(300, 200), d_model=512)
    prob = _problem(cfg, cuda_device)
    k, v, h = prob.make_sources()
    prob.alloc_pools()
    prob.encode(k, v, h)
    torch.cuda.synchronize()
    slots = O.slot_mapping(P.oracle_batch(prob), cfg.block_size)           # from the intact table
    prob.batch.page_table[0, 3] = prob.batch.n_blocks + 7                  # rows 48..63 of request 0
    prob.batch.page_table[1, 0] = -1                                       # rows 0..15 of request 1
    prob.reuse_decode()
    prob.patch()
    torch.cuda.synchronize()
    bad = np.r_[48:64, 300:316]
    good = np.setdiff1d(np.arange(prob.T), bad)
    P.check_untouched(prob, [0, 1], slots[good])                           # the bad rows' slots still hold the sentinel
    P.check_reuse_decode(prob, good)
    P.check_patch(prob, good)


def test_all_layers_patch_with_mixed_code_ranks(cuda_device):
    """L_patch = all layers (legal), with PATCH layers whose r_h differ: scd_patch runs each GEMM stage for a
    group of consecutive layers of equal (r_h, d_a) as one launch, so ranks 128, 64, 64, 128 exercise groups of 1, 2, 1."""
    cfg = MINI["llama3_8b_8k"].scaled(seqlens=(333,), n_layers=4, patch_layers=(0, 1, 2, 3), d_model=512)
    arts = [W.make_layer_artifacts(cfg, l, cuda_device, total_rows=333) for l in range(4)]
    g = torch.Generator(device=cuda_device).manual_seed(5)
    for l in (1, 2):                                   # a narrower H code for the two middle layers (random W1: d_a != width of B_H)
        a = arts[l]
        a.enc_h = a.enc_h[:, :64].contiguous()
        a.w1 = (torch.randn(64, cfg.d_a, generator=g, device=cuda_device) / 8.0).to(a.w1.dtype)
    prob = _problem(cfg, cuda_device, artifacts=arts)
    assert [prob.plan.code_segment(l, 2, prob.T)[2] for l in range(4)] == [128, 64, 64, 128]
    res = _run_all(prob)
    print(res)


@pytest.mark.parametrize("seed", range(6))
def test_random_ragged_batches(seed, cuda_device):
    """Seeded random draws over what the tests above fix by hand (tier 4): request count and lengths (1 ... 700,
    so tiles straddle requests and pages are partial), permuted pages, position offsets, the PATCH set (empty, some, all),
    rank, per-head vs per-layer REUSE, bf16 vs e4m3 codes."""
    rng = np.random.default_rng(1000 + seed)
    n_layers = int(rng.integers(1, 5))
    patch = tuple(int(l) for l in range(n_layers) if rng.random() < 0.4)
    seqlens = tuple(int(x) for x in rng.integers(1, 700, int(rng.integers(1, 6))))
    e4 = bool(rng.random() < 0.35)
    base = MINI["mistral_7b_32k_fp8"] if e4 else MINI["llama3_8b_8k"]
    per_head = 0 if rng.random() < 0.6 else int(rng.choice([16, 32]))
    rank = int(rng.choice([64, 128, 256] if e4 else [32, 64, 96, 128, 256]))
    cfg = base.scaled(n_layers=n_layers, patch_layers=patch, seqlens=seqlens, ragged_range=None, permute_pages=True,
                      d_model=int(rng.choice([512, 1024])), rank=rank)
    offs = [int(x) for x in rng.integers(0, 3000, len(seqlens))]
    prob = _problem(cfg, cuda_device, pos_offset=offs, per_head_rank=per_head)
    res = _run_all(prob)
    print(seed, n_layers, patch, seqlens, rank, per_head, "e4m3" if e4 else "bf16", res)


def test_patch_with_a_one_layer_workspace(cuda_device):
    """scd_patch prefers a workspace for a whole group of PATCH layers (one launch per GEMM stage and group) but must
    accept one that holds a single layer's intermediates, and produce the same bits."""
    from paper_2606_07684_b200 import binding as B
    cfg = MINI["llama3_8b_8k"].scaled(seqlens=(400,), n_layers=3, patch_layers=(0, 1, 2), d_model=512)
    prob = _problem(cfg, cuda_device)
    k, v, h = prob.make_sources()
    prob.alloc_pools()
    prob.encode(k, v, h)
    n_full = prob.patch()
    torch.cuda.synchronize()
    want = [(kp.clone(), vp.clone()) for kp, vp in zip(prob.k_pool, prob.v_pool)]
    prob.alloc_pools()
    one = prob.ws_bytes // 3
    assert one % 128 == 0
    n_one = B.scd_patch(prob.plan, prob.bdesc, prob.codes, prob.k_pool, prob.v_pool, prob.batch.n_blocks,
                        prob.workspace[:one])
    torch.cuda.synchronize()
    assert n_full == 3 and n_one == 9                   # 3 stages x 1 group  vs  3 stages x 3 groups of one layer
    for (kw, vw), kp, vp in zip(want, prob.k_pool, prob.v_pool):
        assert torch.equal(kw.view(torch.int16), kp.view(torch.int16)) and torch.equal(vw.view(torch.int16), vp.view(torch.int16))
    P.check_patch(prob)


@pytest.mark.parametrize("name", ["tiny", "llama3_8b_8k", "mistral_7b_32k_fp8"])
def test_layer_streamed_calls_give_the_same_bits(name, cuda_device):
    """scd_*_layers: the path run window by window -- [0,1), [1,3), [3,L), with the source pointers
    of the other layers withheld -- writes exactly the code and pool bits of the three whole calls; an empty window and a
    window without REUSE / PATCH layers are no-ops; a bad window is SCD_E_ARG."""
    from paper_2606_07684_b200 import binding as B
    cfg = MINI[name] if name == "tiny" else MINI[name].scaled(n_layers=5, patch_layers=(1, 4), seqlens=(300, 45))
    L = cfg.n_layers
    prob = _problem(cfg, cuda_device)
    k, v, h = prob.make_sources()
    if prob.model.k_is_roped:
        k = P.roped_producer_k(prob, k)
    prob.alloc_pools()
    prob.encode(k, v, h); prob.reuse_decode(); prob.patch()
    torch.cuda.synchronize()
    codes_full = prob.codes.clone()
    pools_full = [t.clone() for t in prob.k_pool + prob.v_pool]
    prob.codes.fill_(0xA5)                               # the harness' guard pattern (padding bytes are compared too)
    prob.alloc_pools()
    only = lambda ts, b, e: [t if b <= i < e else None for i, t in enumerate(ts)]
    windows = [(0, 1), (1, 3), (3, L)] if L > 3 else [(0, 1), (1, L)]
    for b, e in windows:                                 # producer side, group by group
        prob.encode(only(k, b, e), only(v, b, e), only(h, b, e), layers=(b, e))
    for b, e in reversed(windows):                       # consumer side, any order
        prob.reuse_decode(layers=(b, e))
        prob.patch(layers=(b, e))
    assert prob.encode(k, v, h, layers=(2, 2)) == 0      # empty window: nothing launched
    torch.cuda.synchronize()
    assert torch.equal(prob.codes, codes_full)
    for want, got in zip(pools_full, prob.k_pool + prob.v_pool):
        bits = torch.int32 if want.dtype == torch.float32 else torch.int16
        assert torch.equal(want.view(bits), got.view(bits))
    with pytest.raises(B.ScdError) as err:
        prob.reuse_decode(layers=(3, L + 1))
    assert err.value.status == 1


@pytest.mark.parametrize("state", ["f32", "bf16"])
def test_edge_batches(state, cuda_device):
    """Ragged lengths that are not multiples of 16 / 128, a 1-token request, position offsets,
    permuted pages."""
    base = C["tiny"] if state == "f32" else MINI["llama3_8b_ragged"]
    cfg = base.scaled(seqlens=(1, 17, 129, 16, 255), ragged_range=None, permute_pages=True, n_layers=2,
                      patch_layers=(1,))
    prob = _problem(cfg, cuda_device, pos_offset=[0, 5, 1000, 31, 2])
    _run_all(prob)


def test_empty_batch_is_a_noop(cuda_device):
    cfg = C["tiny"].scaled(seqlens=(), n_layers=2, patch_layers=(1,))
    prob = _problem(cfg, cuda_device)
    prob.alloc_pools()
    assert prob.T == 0
    prob.encode(*[[None] * 2] * 3)
    prob.reuse_decode()
    prob.patch()
    torch.cuda.synchronize()
    P.check_untouched(prob, [], np.zeros(0, np.int64), also_untouched_layers=[0, 1])


@pytest.mark.parametrize("state", ["f32", "bf16"])
def test_variants_paper_literal_and_interleaved(state, cuda_device):
    """Paper-literal options: no mean vectors, NORM_NONE, identity activation; INTERLEAVED RoPE;
    different producer / consumer theta."""
    base = C["tiny"] if state == "f32" else MINI["llama3_8b_8k"].scaled(seqlens=(200,), n_layers=2, patch_layers=(1,))
    from paper_2606_07684_b200 import binding as B
    prob = _problem(base, cuda_device, use_means=False, patch_norm=B.SCD_NORM_NONE, patch_act=B.SCD_ACT_IDENTITY,
                    rope_theta_consumer=1e4 if base.rope_theta != 1e4 else 5e5)
    _run_all(prob)
    prob = _problem(base, cuda_device, rope_style=B.SCD_ROPE_INTERLEAVED, k_is_roped=(state == "f32"))
    _run_all(prob)


def test_independent_ranks_r_k_ne_r_v(cuda_device):
    """K and V are compressed independently with their own ranks."""
    cfg = MINI["llama3_8b_8k"].scaled(seqlens=(300,), n_layers=2, patch_layers=())
    arts = [W.make_layer_artifacts(cfg, l, cuda_device, total_rows=300) for l in range(2)]
    for a in arts:                                     # truncate the V translators to rank 64
        a.enc_v = a.enc_v[:, :64].contiguous()
        a.dec_v = a.dec_v[:64].contiguous()
    prob = _problem(cfg, cuda_device, artifacts=arts)
    _run_all(prob)
    assert prob.plan.code_segment(0, 0, prob.T)[2] == 128 and prob.plan.code_segment(0, 1, prob.T)[2] == 64


def test_error_paths(cuda_device):
    from paper_2606_07684_b200 import binding as B
    cfg = MINI["llama3_8b_8k"].scaled(seqlens=(64,), n_layers=2, patch_layers=(1,))
    prob = _problem(cfg, cuda_device)
    prob.alloc_pools()
    k, v, h = prob.make_sources()
    with pytest.raises(B.ScdError) as e:               # workspace too small
        B.scd_patch(prob.plan, prob.bdesc, prob.codes, prob.k_pool, prob.v_pool, prob.batch.n_blocks,
                    prob.workspace[:128])
    assert e.value.status == 5
    with pytest.raises(B.ScdError) as e:               # misaligned code buffer
        B.scd_reuse_decode(prob.plan, prob.bdesc, prob.codes[16:], prob.k_pool, prob.v_pool, prob.batch.n_blocks)
    assert e.value.status == 4
    bad = B.batch_desc(prob.batch.cu_seqlens, prob.batch.page_table, None, prob.batch.seqlens, max_pos_offset=10 ** 6)
    with pytest.raises(B.ScdError) as e:               # positions beyond the RoPE table
        B.scd_reuse_decode(prob.plan, bad, prob.codes, prob.k_pool, prob.v_pool, prob.batch.n_blocks)
    assert e.value.status == 1
    with pytest.raises(B.ScdError) as e:               # PATCH layers receive only Z_H
        prob.plan.code_segment(1, 0, prob.T)
    assert e.value.status == 1
    P.check_untouched(prob, [], np.zeros(0, np.int64), also_untouched_layers=[0, 1])   # nothing was enqueued


# ------------------------------------------------------------------ full BASELINE sizes
FULL_SAMPLE = {"llama3_8b_8k": 384, "llama3_8b_ragged": 256, "mistral_7b_32k_fp8": 256, "llama3_70b_2x16k": 128}


@pytest.mark.slow
@pytest.mark.parametrize("name,rank", [("llama3_8b_8k", 0), ("llama3_8b_ragged", 0), ("mistral_7b_32k_fp8", 0),
                                       ("llama3_70b_2x16k", 0), ("llama3_70b_2x16k", 512)])
def test_full_size_sampled_parity(name, rank, cuda_device):
    """BASELINE.json's full sizes in the launch configuration bench.py times (rank 0 = the config's own; 512 = the
    widest rank of the config-5 sweep); the oracle recomputes a row sample (first / last rows of every request,
    ragged tails, seeded random rows -- rows are independent); sentinels checked over the whole pool."""
    cfg = C[name] if not rank else C[name].scaled(rank=rank)
    prob = _problem(cfg, cuda_device)
    rows = P.sample_rows(prob, FULL_SAMPLE[name])
    res = _run_all(prob, rows=rows, roped=False)
    print(name, rank, res)


@pytest.mark.parametrize("name", ["llama3_8b_ragged", "mistral_7b_32k_fp8"])
def test_paged_producer_source(name, cuda_device):
    """the producer's K / V live in ITS paged cache (own page table, own permutation, junk in
    the unused slots) and scd_encode gathers them through that table (TMA tile::gather4).  The codes must equal,
    bit for bit, those of the same rows handed over packed, and match the oracle reading the pool through
    O.read_paged."""
    cfg = MINI[name].scaled(ragged_range=(5, 1, 400), permute_pages=True) if name == "llama3_8b_ragged" else MINI[name]
    prob = _problem(cfg, cuda_device)
    k, v, h = prob.make_sources()
    k = P.roped_producer_k(prob, k)
    prob.encode(k, v, h)
    torch.cuda.synchronize()
    want = prob.codes.clone()
    # the producer's own paging: a different permutation over a larger pool
    bs, T = cfg.block_size, prob.T
    g = torch.Generator().manual_seed(99)
    pages = [(l + bs - 1) // bs for l in prob.batch.seqlens]
    n_blocks = sum(pages) + 7
    ids = torch.randperm(n_blocks, generator=g)
    table = torch.full((len(pages), max(pages) + 2), -1, dtype=torch.int32)
    at = 0
    for i, n in enumerate(pages):
        table[i, :n] = ids[at:at + n].to(torch.int32)
        at += n
    ob = O.Batch(prob.batch.cu_seqlens.cpu().numpy().astype(np.int64), table.numpy().astype(np.int64), None)
    slots = torch.from_numpy(O.slot_mapping(ob, bs)).to(cuda_device)
    kp, vp = [None] * cfg.n_layers, [None] * cfg.n_layers
    for l in range(cfg.n_layers):
        if k[l] is None:
            continue
        for src, dst in ((k, kp), (v, vp)):
            pool = torch.randn(n_blocks * bs, cfg.D, generator=g).to(torch.bfloat16).to(cuda_device)
            pool[slots] = src[l].reshape(T, cfg.D)
            dst[l] = pool
            # the oracle's reading of the pool gives back the packed rows
            np.testing.assert_array_equal(O.read_paged(pool.float().cpu().numpy(), slots.cpu().numpy()),
                                          src[l].reshape(T, cfg.D).float().cpu().numpy())
    prob.codes.fill_(0xA5)
    prob.encode(kp, vp, h, src_page_table=table.to(cuda_device), src_n_blocks=n_blocks)
    torch.cuda.synchronize()
    for b, e in prob.code_ranges():
        assert torch.equal(prob.codes[b:e], want[b:e]), "codes gathered through the producer's page table differ"
    assert prob.guard_violations() == (0, 0)
    P.check_encode(prob, k, v, h)


@pytest.mark.parametrize("rank", [64, 192, 256])
def test_e4m3_decode_with_several_tiles_per_cta(rank, cuda_device):
    """e4m3 codes keep the code tile of an (m-tile, segment) resident across its four n-tiles.  The mini configs give every CTA at
    most one tile; here 21 m-tiles x 6 segments x 4 n-tiles = 504 tiles on 148 CTAs, so CTAs walk several tiles, enter and leave
    (m-tile, segment) groups in the middle, and reuse a widened tile -- with ragged requests and permuted pages."""
    cfg = MINI["mistral_7b_32k_fp8"].scaled(n_layers=4, patch_layers=(3,), seqlens=(1500, 1100, 7), d_model=512, rank=rank,
                                            permute_pages=True)
    prob = _problem(cfg, cuda_device, pos_offset=[0, 40, 3])
    res = _run_all(prob)
    print(rank, res)


@pytest.mark.parametrize("rank", [32, 64, 192, 256])
def test_bf16_decode_with_a_resident_code_tile_and_several_tiles_per_cta(rank, cuda_device):
    """bf16 codes with one, three or four k-blocks per tile decode on the resident-code-tile variant too (two k-blocks keep
    the plain kernel).  Same geometry as the e4m3 case above: 504 tiles on 148 CTAs, groups entered and left mid-way, the slot
    table shared per lane quadrant and the mean slices shared per column group, ragged requests, permuted pages."""
    cfg = MINI["llama3_8b_8k"].scaled(n_layers=4, patch_layers=(3,), seqlens=(1500, 1100, 7), d_model=512, rank=rank,
                                      permute_pages=True)
    prob = _problem(cfg, cuda_device, pos_offset=[0, 40, 3])
    res = _run_all(prob)
    print(rank, res)


def test_patch_gemms_on_cta_pairs_with_several_tiles_per_pair(cuda_device):
    """PATCH GEMM-2 / GEMM-3 run as CTA pairs (tcgen05 cta_group::2).  39 m-tiles (odd: the last pair has an out-of-range
    partner) x 4 n-tiles x 2 layers = 160 / 320 pair tiles on 74 pairs: every pair walks several tiles, through the L2
    super-block order and both accumulator buffers."""
    cfg = MINI["llama3_8b_8k"].scaled(n_layers=2, patch_layers=(0, 1), seqlens=(3000, 1990), d_model=1024)
    prob = _problem(cfg, cuda_device)
    res = _run_all(prob)
    print(res)


def test_patch_gemm1_b_resident_walk_with_a_ragged_tail(cuda_device):
    """PATCH GEMM-1 with enough tiles for the B-resident walk (4 layers x 4 n-tiles x 39 m-tiles = 624 >= 4 x 148): every CTA
    owns a contiguous run of ~4 m-tiles, runs cross (layer, n-tile) boundaries -- the resident W1 tile is swapped mid-run, the
    staged bias slice with it -- and the last m-tile has 126 valid rows.  All layers are PATCH layers."""
    cfg = MINI["llama3_8b_8k"].scaled(n_layers=4, patch_layers=(0, 1, 2, 3), seqlens=(3000, 1990), d_model=1024)
    prob = _problem(cfg, cuda_device)
    res = _run_all(prob)
    print(res)
