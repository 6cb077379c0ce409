"""GPU parity of fp8 K/V pools (second half; build extension U20): scd_reuse_decode / scd_patch
writing e4m3 bytes + one fp32 scale per (slot, head).

Two comparisons.  (1) The quantiser is an ENCODING, so it is checked bit-exactly: the kernel quantises the very bf16
values it would have stored, therefore bytes and scales must equal O.quantize_pool applied to the bits of the bf16
pool the same call produces (those bits are themselves parity-checked against the oracle by P.check_reuse_decode /
P.check_patch).  (2) End to end against the oracle alone: the dequantised fp8 pool vs the oracle's own quantised K/V,
relative Frobenius <= 2e-2 per layer (north_star's bf16 tolerance; the oracle's value is its QUANTISED value, as for
e4m3 codes), every element within one e4m3 step.  Slots outside the batch keep their sentinels."""
import numpy as np
import pytest
import torch

from oracle import scd_oracle as O
from paper_2606_07684_b200 import workloads as W
from tests import _parity as P

pytestmark = pytest.mark.gpu

C = W.CONFIGS
CASES = {
    "bf16_codes": C["llama3_8b_8k"].scaled(n_layers=3, patch_layers=(1,), seqlens=(300, 77, 1), d_model=1024, permute_pages=True),
    "e4m3_codes": C["mistral_7b_32k_fp8"].scaled(n_layers=3, patch_layers=(2,), seqlens=(450,), d_model=512),
    "short_k_patch": C["llama3_8b_8k"].scaled(n_layers=2, patch_layers=(0, 1), seqlens=(200, 200), d_model=256, rank=64),
}
SENT_BYTE, SENT_SCALE = 0xFF, 0x7FC00001


PER_HEAD = {"per_head_reuse": 32}        # the paper-literal per-head translator writing fp8 pools
CASES["per_head_reuse"] = C["llama3_8b_8k"].scaled(n_layers=2, patch_layers=(), seqlens=(260, 41), d_model=512)


@pytest.mark.parametrize("name", list(CASES))
def test_fp8_pools(name, cuda_device):
    from paper_2606_07684_b200 import binding as B
    from paper_2606_07684_b200.harness import CodecProblem
    cfg = CASES[name]
    prob = CodecProblem(cfg, cuda_device, pos_offset=[5 * i for i in range(len(cfg.seqlens))], per_head_rank=PER_HEAD.get(name, 0))
    k, v, h = prob.make_sources()
    k = P.roped_producer_k(prob, k)
    prob.alloc_pools()
    prob.encode(k, v, h)
    prob.reuse_decode()
    prob.patch()
    torch.cuda.synchronize()
    P.check_reuse_decode(prob)                                  # the bf16 pools are right ...
    P.check_patch(prob)
    nb, bs, H, dh, D, L = prob.batch.n_blocks, cfg.block_size, cfg.n_kv_heads, cfg.head_dim, cfg.D, cfg.n_layers
    mk8 = lambda: torch.full((nb, bs, H, dh), SENT_BYTE, dtype=torch.uint8, device=cuda_device)
    mks = lambda: torch.full((nb, bs, H), SENT_SCALE, dtype=torch.int32, device=cuda_device).view(torch.float32)
    k8, v8, ks, vs = [mk8() for _ in range(L)], [mk8() for _ in range(L)], [mks() for _ in range(L)], [mks() for _ in range(L)]
    B.scd_reuse_decode(prob.plan, prob.bdesc, prob.codes, k8, v8, nb, k_scale=ks, v_scale=vs)
    B.scd_patch(prob.plan, prob.bdesc, prob.codes, k8, v8, nb, prob.workspace, k_scale=ks, v_scale=vs)
    torch.cuda.synchronize()
    om, ob = P.oracle_model(prob), P.oracle_batch(prob)
    pos, slots = O.positions(ob), O.slot_mapping(ob, bs)
    st = torch.from_numpy(slots).to(cuda_device)
    mask = np.ones(nb * bs, bool)
    mask[slots] = False
    worst = 0.0
    for l in range(L):
        ol = P.oracle_layer(prob, l)
        if prob.arts[l].kind == W.REUSE:
            qk, sk = P.gpu_codes(prob, l, O.BRANCH_K, None)
            qv, sv = P.gpu_codes(prob, l, O.BRANCH_V, None)
            want_y = O.reuse_decode_layer(om, ol, O.unpack_codes(qk, sk, om.code_dtype), O.unpack_codes(qv, sv, om.code_dtype), pos)
        else:
            qh, sh = P.gpu_codes(prob, l, O.BRANCH_H, None)
            want_y = O.patch_layer(om, ol, O.unpack_codes(qh, sh, om.code_dtype), pos)
        for name_, y_o, p16, p8, sc in (("K", want_y[0], prob.k_pool[l], k8[l], ks[l]), ("V", want_y[1], prob.v_pool[l], v8[l], vs[l])):
            got_q = p8.view(-1, D)[st].cpu().numpy()
            got_s = sc.view(-1, H)[st].cpu().numpy()
            # (1) bit-exact against the oracle's quantiser on the bf16 bits this call stores
            x16 = p16.view(-1, D)[st].double().cpu().numpy()
            want_q, want_s = O.quantize_pool(x16, H)
            np.testing.assert_array_equal(got_s, want_s, err_msg=f"layer {l} {name_}: scales")
            same = (got_q == want_q) | ((O.E4M3_VALUES[got_q] == 0) & (O.E4M3_VALUES[want_q] == 0))
            assert same.all(), f"layer {l} {name_}: {np.count_nonzero(~same)} bytes differ from the oracle's quantiser"
            # (2) end to end against the oracle alone
            oq, os_ = O.quantize_pool(y_o, H)
            deq_o, deq_g = O.dequantize_pool(oq, os_), O.dequantize_pool(got_q, got_s)
            err = P.rel_fro(deq_g, deq_o)
            worst = max(worst, err)
            assert err <= 2e-2, f"layer {l} {name_}: rel fro {err:.3e}"
            # |deq_g - deq_o| <= |q(x_g) - x_g| + |x_g - x_o| + |x_o - q(x_o)|: half an e4m3 step on either side plus the
            # element noise of the stage that produced x (the model P.fine_check uses: output rounding + k_abs of the head's
            # rms), and the head's scale may move by the relative noise of its amax element
            stage = "reuse" if prob.arts[l].kind == W.REUSE else "patch"
            k_abs = P.K_ABS[stage][W.BF16]
            step = np.repeat(os_, dh, axis=1).astype(np.float64) * np.maximum(2.0 ** -3 * np.abs(O.E4M3_VALUES[oq]), 2.0 ** -9)
            rms = np.repeat(np.sqrt(np.mean(y_o.reshape(-1, H, dh) ** 2, axis=2)), dh, axis=1)
            noise = P.REL_OUT[W.BF16] * np.abs(y_o) + k_abs * rms
            rel_s = 2.0 ** -8 + k_abs
            bound = step * (1 + rel_s) + noise + np.abs(deq_o) * rel_s
            used = np.abs(deq_g - deq_o) / bound
            assert used.max() <= 1.0, f"layer {l} {name_}: element off by {used.max():.2f} of (one e4m3 step + stage noise)"
            flips = float(np.mean(got_q != oq))
            assert flips <= (0.05 if stage == "reuse" else 0.25), f"layer {l} {name_}: {flips:.3f} of the bytes differ from the oracle's"
            # sentinels
            assert np.all(p8.view(-1, D).cpu().numpy()[mask] == SENT_BYTE), f"layer {l} {name_}: a slot outside the batch was written"
            assert np.all(sc.view(torch.int32).view(-1, H).cpu().numpy()[mask] == SENT_SCALE)
    print(name, "worst rel fro (dequantised fp8 pool vs oracle's quantised K/V)", worst)


def test_fp8_pools_rejected_where_not_built(cuda_device):
    from paper_2606_07684_b200 import binding as B
    from paper_2606_07684_b200.harness import CodecProblem
    prob = CodecProblem(C["tiny"], cuda_device)
    k, v, h = prob.make_sources()
    prob.alloc_pools()
    prob.encode(k, v, h)
    sc = [torch.zeros(prob.batch.n_blocks, 16, 4, device=cuda_device) for _ in range(4)]
    with pytest.raises(B.ScdError) as e:
        B.scd_reuse_decode(prob.plan, prob.bdesc, prob.codes, prob.k_pool, prob.v_pool, prob.batch.n_blocks, k_scale=sc, v_scale=sc)
    assert e.value.status == 3
