"""GPU parity of the group-wise INT4 comparison codec (scd_int4_quantize / scd_int4_dequantize_paged,
PAPER.md:265) against oracle/int4_oracle.py: codes, metadata and dequantised pool rows BIT-EXACT (the codec is an
encoding; both sides decide in IEEE fp32), page / slot indexing bit-exact through sentinel pools."""
import numpy as np
import pytest
import torch

from oracle import int4_oracle as Q
from oracle import scd_oracle as O
from paper_2606_07684_b200 import workloads as W

pytestmark = pytest.mark.gpu

SENTINEL = 0x7FC1


def _case(cfg, group, device, n_layers, stride_pad=0, seed=0):
    from paper_2606_07684_b200 import binding as B
    batch = W.make_batch(cfg, device)
    T, D = batch.total_tokens, cfg.D
    g = torch.Generator().manual_seed(1234 + seed)
    stride = D + stride_pad
    src = []
    for i in range(2 * n_layers):
        x = torch.randn(T, stride, generator=g) * (0.5 + i)
        x[:, :D] += torch.randn(1, D, generator=g) * 2            # per-channel offsets: asymmetric ranges
        if T:
            x[T // 2, :group] = 0.375                             # a constant group
            x[0, 5] = 300.0                                       # an outlier
        src.append(x.to(torch.bfloat16).to(device))
    desc = B.Int4Desc(cfg.n_kv_heads, cfg.head_dim, cfg.block_size, group)
    stride_b, moff, total, payload = B.scd_int4_layout(desc, T, len(src))
    assert payload == Q.payload_bytes(T, D, group, len(src))
    packed = torch.full((total + 4096,), 0xA5, dtype=torch.uint8, device=device)
    pools = [torch.full((batch.n_blocks, cfg.block_size, cfg.n_kv_heads, cfg.head_dim), SENTINEL, dtype=torch.int16,
                        device=device).view(torch.bfloat16) for _ in src]
    bdesc = B.batch_desc(batch.cu_seqlens, batch.page_table, None, batch.seqlens, 0)
    n1 = B.scd_int4_quantize(desc, T, src, stride, packed)
    n2 = B.scd_int4_dequantize_paged(desc, bdesc, packed, pools, batch.n_blocks)
    torch.cuda.synchronize()
    assert n1 >= 1 and n2 >= 1
    ob = O.Batch(cu_seqlens=batch.cu_seqlens.cpu().numpy(), page_table=batch.page_table.cpu().numpy(), pos_offset=None)
    slots = O.slot_mapping(ob, cfg.block_size)
    pk = packed.cpu().numpy()
    written = np.zeros(pk.shape[0], bool)
    for i, x in enumerate(src):
        xf = x[:, :D].float().cpu().numpy()
        q, want_packed, s, z = Q.quantize(xf, group)
        base = i * stride_b
        got_q = pk[base:base + T * D // 2].reshape(T, D // 2)
        meta = torch.from_numpy(pk[base + moff:base + moff + T * (D // group) * 4].copy()).view(torch.bfloat16).float().numpy().reshape(T, -1, 2)
        got_s, got_z = meta[:, :, 0], meta[:, :, 1]
        np.testing.assert_array_equal(got_q, want_packed)
        np.testing.assert_array_equal(got_s, s)
        np.testing.assert_array_equal(got_z, z)
        for b0, n in ((base, T * D // 2), (base + moff, T * (D // group) * 4)):
            written[b0:b0 + n] = True
        want = Q.dequantize(q, s, z, group)
        pool = pools[i].view(torch.int16).cpu().numpy().reshape(-1, D)
        want_bits = torch.from_numpy(want).to(torch.bfloat16).view(torch.int16).numpy()
        np.testing.assert_array_equal(pool[slots], want_bits)
        mask = np.ones(pool.shape[0], bool)
        mask[slots] = False
        assert np.all(pool[mask] == np.int16(SENTINEL)), "a slot outside the batch was written"
    assert np.all(pk[~written] == 0xA5), "bytes outside the nibble / scale / zero segments were written"


@pytest.mark.parametrize("group", [32, 64, 128])
def test_int4_bit_exact_llama_geometry(group, cuda_device):
    cfg = W.CONFIGS["llama3_8b_8k"].scaled(seqlens=(1000,))
    _case(cfg, group, cuda_device, n_layers=2)


def test_int4_ragged_permuted_pages_and_strided_source(cuda_device):
    cfg = W.CONFIGS["llama3_8b_ragged"].scaled(ragged_range=(7, 1, 300))
    _case(cfg, 32, cuda_device, n_layers=2, stride_pad=64, seed=3)


def test_int4_small_heads_and_one_token(cuda_device):
    cfg = W.CONFIGS["tiny"].scaled(seqlens=(1, 17, 16), state_dtype=W.BF16, permute_pages=True)
    _case(cfg, 32, cuda_device, n_layers=1, seed=5)
    _case(cfg, 64, cuda_device, n_layers=3, seed=6)


def test_int4_empty_batch_and_bad_arguments(cuda_device):
    from paper_2606_07684_b200 import binding as B
    desc = B.Int4Desc(8, 128, 16, 32)
    packed = torch.zeros(1024, dtype=torch.uint8, device=cuda_device)
    assert B.scd_int4_quantize(desc, 0, [], 1024, packed) == 0
    with pytest.raises(B.ScdError):
        B.scd_int4_layout(B.Int4Desc(8, 128, 16, 48), 10, 1)             # group not supported
    with pytest.raises(B.ScdError):
        B.scd_int4_layout(B.Int4Desc(8, 64, 16, 128), 10, 1)             # group does not divide head_dim
    x = torch.zeros(4, 1024, dtype=torch.bfloat16, device=cuda_device)
    with pytest.raises(B.ScdError):
        B.scd_int4_quantize(desc, 4, [x], 1000, packed)                  # stride < width
