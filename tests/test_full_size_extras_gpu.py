"""Full BASELINE sizes, in the launch configuration bench.py times, for the items beside the hot path: the INT4
comparison codec (all 64 K/V tensors of config 2 in one launch), the paged producer source and the fp8 pools (config 2
geometry).  The oracle recomputes a row sample (rows are independent); sentinels / guard bytes are checked
over the whole buffers.  Marked slow."""
import numpy as np
import pytest
import torch

from oracle import int4_oracle as Q
from oracle import scd_oracle as O
from paper_2606_07684_b200 import workloads as W
from tests import _parity as P

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

C = W.CONFIGS


def test_int4_full_size_sampled(cuda_device):
    from paper_2606_07684_b200 import binding as B
    cfg = C["llama3_8b_8k"]
    batch = W.make_batch(cfg, cuda_device)
    T, D, L = batch.total_tokens, cfg.D, cfg.n_layers
    g = torch.Generator(device=cuda_device).manual_seed(7)
    src = [(torch.randn(T, D, generator=g, device=cuda_device) * (1 + 0.1 * i) + 0.3).to(torch.bfloat16) for i in range(2 * L)]
    desc = B.Int4Desc(cfg.n_kv_heads, cfg.head_dim, cfg.block_size, 32)
    stride_b, moff, total, payload = B.scd_int4_layout(desc, T, len(src))
    assert payload == Q.payload_bytes(T, D, 32, len(src))
    packed = torch.full((total + 4096,), 0xA5, dtype=torch.uint8, device=cuda_device)
    pools = [torch.full((batch.n_blocks, cfg.block_size, cfg.n_kv_heads, cfg.head_dim), 0x7FC1, dtype=torch.int16,
                        device=cuda_device).view(torch.bfloat16) for _ in src]
    bdesc = B.batch_desc(batch.cu_seqlens, batch.page_table, None, batch.seqlens, 0)
    assert B.scd_int4_quantize(desc, T, src, D, packed) == 1           # one launch for all tensors
    assert B.scd_int4_dequantize_paged(desc, bdesc, packed, pools, batch.n_blocks) == 1
    torch.cuda.synchronize()
    assert bool((packed[total:] == 0xA5).all())
    ob = O.Batch(batch.cu_seqlens.cpu().numpy().astype(np.int64), batch.page_table.cpu().numpy().astype(np.int64), None)
    slots = O.slot_mapping(ob, cfg.block_size)
    rng = np.random.default_rng(3)
    rows = np.unique(np.concatenate([np.arange(0, 8), np.arange(T - 24, T), rng.integers(0, T, 200)]))
    rt = torch.from_numpy(rows).to(cuda_device)
    for i in (0, 1, L - 1, L, 2 * L - 1):
        x = src[i][rt].float().cpu().numpy()
        q, want_packed, s, z = Q.quantize(x, 32)
        base = i * stride_b
        got_q = packed[base:base + T * D // 2].view(T, D // 2)[rt].cpu().numpy()
        meta = packed[base + moff:base + moff + T * (D // 32) * 4].view(torch.bfloat16).view(T, D // 32, 2)[rt].float().cpu().numpy()
        np.testing.assert_array_equal(got_q, want_packed)
        np.testing.assert_array_equal(meta[:, :, 0], s)
        np.testing.assert_array_equal(meta[:, :, 1], z)
        want = torch.from_numpy(Q.dequantize(q, s, z, 32)).to(torch.bfloat16).view(torch.int16).numpy()
        pool = pools[i].view(torch.int16).view(-1, D)
        np.testing.assert_array_equal(pool[torch.from_numpy(slots[rows]).to(cuda_device)].cpu().numpy(), want)
        mask = torch.ones(pool.shape[0], dtype=torch.bool, device=cuda_device)
        mask[torch.from_numpy(slots).to(cuda_device)] = False
        assert bool((pool[mask] == 0x7FC1).all()) and not bool((pool[~mask] == 0x7FC1).all(dim=1).any())


def test_paged_source_and_fp8_pools_full_size(cuda_device):
    """Config 2 at full size: encode through a producer page table must give the bits of the packed encode; REUSE
    decode into fp8 pools must give, on every row, the oracle quantiser's bytes of the bf16 pool the plain call writes."""
    from paper_2606_07684_b200 import binding as B
    from paper_2606_07684_b200.harness import CodecProblem
    cfg = C["llama3_8b_8k"]
    prob = CodecProblem(cfg, cuda_device)
    k, v, h = prob.make_sources()
    prob.alloc_pools()
    prob.encode(k, v, h)
    torch.cuda.synchronize()
    want = prob.codes.clone()
    T, bs = prob.T, cfg.block_size
    # the packed states ARE a paged pool under an identity table; permute the pages to make it a real one
    g = torch.Generator().manual_seed(5)
    perm = torch.randperm(T // bs, generator=g)
    table = perm.to(torch.int32).view(1, -1).to(cuda_device)
    inv = torch.empty_like(perm)
    inv[perm] = torch.arange(T // bs)
    def paged(t):      # pool block perm[j] holds tokens of page j
        return t.view(T // bs, bs, -1)[inv.to(cuda_device)].reshape(T, -1).contiguous()
    kp = [None if t is None else paged(t.view(T, -1)) for t in k]
    vp = [None if t is None else paged(t.view(T, -1)) for t in v]
    prob.codes.fill_(0xA5)
    prob.encode(kp, vp, h, src_page_table=table, src_n_blocks=T // bs)
    torch.cuda.synchronize()
    for b, e in prob.code_ranges():
        assert torch.equal(prob.codes[b:e], want[b:e])
    assert prob.guard_violations() == (0, 0)
    # fp8 pools against the bf16 pools of the plain call
    prob.reuse_decode()
    nb, H, dh, D, L = prob.batch.n_blocks, cfg.n_kv_heads, cfg.head_dim, cfg.D, cfg.n_layers
    reuse = [l for l in range(L) if prob.arts[l].kind == W.REUSE]
    k8 = [torch.full((nb, bs, H, dh), 0xFF, dtype=torch.uint8, device=cuda_device) if l in reuse else None for l in range(L)]
    v8 = [None if t is None else t.clone() for t in k8]
    ks = [torch.full((nb, bs, H), float("nan"), device=cuda_device) if l in reuse else None for l in range(L)]
    vs = [None if t is None else t.clone() for t in ks]
    B.scd_reuse_decode(prob.plan, prob.bdesc, prob.codes, k8, v8, nb, k_scale=ks, v_scale=vs)
    torch.cuda.synchronize()
    slots = O.slot_mapping(P.oracle_batch(prob), bs)
    rows = P.sample_rows(prob, 256)
    st = torch.from_numpy(slots[rows]).to(cuda_device)
    for l in (reuse[0], reuse[len(reuse) // 2], reuse[-1]):
        for p16, p8, sc in ((prob.k_pool[l], k8[l], ks[l]), (prob.v_pool[l], v8[l], vs[l])):
            want_q, want_s = O.quantize_pool(p16.view(-1, D)[st].double().cpu().numpy(), H)
            got_q, got_s = p8.view(-1, D)[st].cpu().numpy(), sc.view(-1, H)[st].cpu().numpy()
            np.testing.assert_array_equal(got_s, want_s)
            same = (got_q == want_q) | ((O.E4M3_VALUES[got_q] == 0) & (O.E4M3_VALUES[want_q] == 0))
            assert same.all()
            written = ~torch.isnan(sc.view(-1, H)).any(dim=1)
            assert int(written.sum()) == T and bool(written[torch.from_numpy(slots).to(cuda_device)].all())
