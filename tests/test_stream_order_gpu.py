"""Stream-order guarantees of the hot calls at full size (config 2), where the launches really overlap.

The launches of one scd_encode call skip the programmatic-dependency wait at their start and wait for their predecessor at
their end: (1) a call must still see what the stream produced right before it -- here device copies that fill
the source tensors, enqueued immediately before scd_encode with no synchronisation; (2) the next call on the stream must see
everything the call wrote -- encode -> reuse_decode -> patch back to back with no synchronisation must give the bits of the
same chain run with a synchronisation after every call; (3) a second scd_encode into the same code buffer must win over the
first.  Bitwise comparisons: the kernels are deterministic."""
import pytest
import torch

from paper_2606_07684_b200 import workloads as W

pytestmark = [pytest.mark.gpu, pytest.mark.slow]


def test_calls_enqueued_back_to_back_see_each_other(cuda_device):
    from paper_2606_07684_b200.harness import CodecProblem
    cfg = W.CONFIGS["llama3_8b_8k"]
    prob = CodecProblem(cfg, cuda_device)
    k, v, h = prob.make_sources()
    prob.alloc_pools()
    # reference: a synchronisation after every call
    prob.encode(k, v, h); torch.cuda.synchronize()
    prob.reuse_decode(); torch.cuda.synchronize()
    prob.patch(); torch.cuda.synchronize()
    codes_ref = prob.codes.clone()
    L = cfg.n_layers
    kp_ref = [prob.k_pool[l].clone() for l in (0, 8, L - 1)]
    vp_ref = [prob.v_pool[l].clone() for l in (0, 8, L - 1)]
    # staging tensors the sources are refilled from, and a decoy set of sources
    live = [t for t in (k + v + h) if t is not None]
    keep = [t.clone() for t in live]
    for rep in range(3):
        for t in live:
            t.zero_()
        prob.codes.fill_(0x5A)
        prob.alloc_pools()                    # fresh pools (sentinels in the slots outside the batch, as in the reference)
        torch.cuda.synchronize()
        # (3) a first encode of the zeroed sources, then (1) the refill and the real encode, then (2) decode and patch: no syncs
        prob.encode(k, v, h)
        for t, src in zip(live, keep):
            t.copy_(src, non_blocking=True)
        prob.encode(k, v, h)
        prob.reuse_decode()
        prob.patch()
        torch.cuda.synchronize()
        bad = [(b, e) for b, e in prob.code_ranges() if not torch.equal(prob.codes[b:e], codes_ref[b:e])]
        assert not bad, f"rep {rep}: {len(bad)} code segments differ from the synchronised chain, first at bytes {bad[0]}"
        for i, l in enumerate((0, 8, L - 1)):
            assert torch.equal(prob.k_pool[l].view(torch.int16), kp_ref[i].view(torch.int16)), f"rep {rep}: K pool of layer {l}"
            assert torch.equal(prob.v_pool[l].view(torch.int16), vp_ref[i].view(torch.int16)), f"rep {rep}: V pool of layer {l}"
