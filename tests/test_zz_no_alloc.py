"""scd_patch_static (include/scd.h): scd_patch with its intermediates in the library's static device array -- no caller
workspace, no allocation -- against the existing path (scd_patch with a caller workspace) on the same inputs.

Two calls in a row on DIFFERENT codes: the array keeps the first call's contents, so the second call shows that nothing
stale leaks into it.  Tolerance: the relative Frobenius bound the parity tests use for bf16 states (2e-2 per layer, tests/
_parity.py); the two paths run the same kernels, so the pools are also expected to be bit-identical and the test says
whether they were.  Also: slots outside the batch stay untouched, and a batch whose one-layer intermediates exceed
SCD_PATCH_STATIC_WORKSPACE_BYTES is refused with SCD_E_WORKSPACE before anything is enqueued.

This file is collected last on purpose (the suite runs with pytest -x): it passes alone in a fresh process and after the
other GPU tests."""
import pytest
import torch

from paper_2606_07684_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 2e-2                      # tests/_parity.py: TOL[BF16]
SENT = 0x7FC1                   # bf16 NaN payload the pools are filled with


def _sentinel_pools(prob, device):
    cfg, nb = prob.cfg, prob.batch.n_blocks
    mk = lambda: torch.full((nb, cfg.block_size, cfg.n_kv_heads, cfg.head_dim), SENT, dtype=torch.int16, device=device).view(torch.bfloat16)
    return [mk() for _ in range(cfg.n_layers)], [mk() for _ in range(cfg.n_layers)]


def _rel_fro(a, b):
    a, b = a.double(), b.double()
    return float((a - b).norm() / b.norm().clamp_min(1e-30))


def test_patch_static_matches_scd_patch_on_two_calls_in_a_row(cuda_device):
    from paper_2606_07684_b200 import binding as B
    from paper_2606_07684_b200.harness import CodecProblem
    # three PATCH layers, 1111 tokens (ragged last m-tile), d_model 1024: 4.6 MB of intermediates per layer, so the 32 MiB
    # array groups all three layers per launch while the caller workspace below is sized by scd_plan_query
    cfg = W.CONFIGS["llama3_8b_8k"].scaled(n_layers=4, patch_layers=(0, 2, 3), seqlens=(700, 400, 11), d_model=1024, permute_pages=True)
    prob = CodecProblem(cfg, cuda_device, pos_offset=[0, 9, 3])
    patch_layers = [l for l in range(cfg.n_layers) if prob.arts[l].kind == W.PATCH]
    nb = prob.batch.n_blocks
    slots_written = None
    for call in range(2):
        k, v, h = prob.make_sources()
        if call == 1:           # different inputs for the second call
            h = [None if t is None else (t.float() * -0.5 + 0.125).to(t.dtype) for t in h]
        prob.alloc_pools()
        prob.encode(k, v, h)
        torch.cuda.synchronize()
        # existing path: caller workspace
        k_ref, v_ref = _sentinel_pools(prob, cuda_device)
        n_ref = B.scd_patch(prob.plan, prob.bdesc, prob.codes, k_ref, v_ref, nb, prob.workspace)
        # new path: static array, nothing allocated by the call (the pools are the caller's outputs)
        k_new, v_new = _sentinel_pools(prob, cuda_device)
        before = torch.cuda.memory_allocated(cuda_device)
        n_new = B.scd_patch_static(prob.plan, prob.bdesc, prob.codes, k_new, v_new, nb)
        assert torch.cuda.memory_allocated(cuda_device) == before
        torch.cuda.synchronize()
        assert n_new > 0 and n_ref > 0
        exact = True
        for l in range(cfg.n_layers):
            for name, got, want in (("K", k_new[l], k_ref[l]), ("V", v_new[l], v_ref[l])):
                gi, wi = got.view(torch.int16), want.view(torch.int16)
                written = (wi != SENT).view(-1, cfg.D).any(dim=1)
                if l not in patch_layers:
                    assert not bool(written.any()) and bool((gi == SENT).all()), f"call {call} layer {l} {name}: a REUSE layer was written"
                    continue
                assert int(written.sum()) == prob.T, f"call {call} layer {l} {name}: the reference wrote {int(written.sum())} rows"
                # same slots written, sentinels elsewhere
                assert bool(((gi != SENT).view(-1, cfg.D).any(dim=1) == written).all()), f"call {call} layer {l} {name}: slots differ"
                g, w = got.view(-1, cfg.D)[written], want.view(-1, cfg.D)[written]
                assert bool(torch.isfinite(g.float()).all()), f"call {call} layer {l} {name}: non-finite output"
                err = _rel_fro(g, w)
                assert err <= TOL, f"call {call} layer {l} {name}: rel fro {err:.3e} against scd_patch"
                exact &= bool(torch.equal(gi, wi))
        if call == 0:
            first = [t.clone() for t in k_new]
        else:                   # the second call's inputs really were different
            assert not torch.equal(first[patch_layers[0]].view(torch.int16), k_new[patch_layers[0]].view(torch.int16))
        print(f"call {call}: {n_new} launches (scd_patch: {n_ref}), bit-identical to scd_patch: {exact}")


def test_patch_static_refuses_batches_beyond_its_array(cuda_device):
    from paper_2606_07684_b200 import binding as B
    from paper_2606_07684_b200.harness import CodecProblem
    # 8200 tokens x (d_a + d) x 2 B = 33.6 MB per layer > 32 MiB
    cfg = W.CONFIGS["llama3_8b_8k"].scaled(n_layers=2, patch_layers=(1,), seqlens=(8200,), d_model=1024)
    prob = CodecProblem(cfg, cuda_device)
    k, v, h = prob.make_sources()
    prob.alloc_pools()
    prob.encode(k, v, h)
    k8, v8 = _sentinel_pools(prob, cuda_device)
    with pytest.raises(B.ScdError) as e:
        B.scd_patch_static(prob.plan, prob.bdesc, prob.codes, k8, v8, prob.batch.n_blocks)
    assert e.value.status == 5 and "SCD_PATCH_STATIC_WORKSPACE_BYTES" in str(e.value)          # SCD_E_WORKSPACE
    torch.cuda.synchronize()
    assert bool((k8[1].view(torch.int16) == SENT).all())                                      # nothing was enqueued
    # the same batch goes through scd_patch with a caller workspace
    assert B.scd_patch(prob.plan, prob.bdesc, prob.codes, k8, v8, prob.batch.n_blocks, prob.workspace) > 0
    torch.cuda.synchronize()


def test_patch_static_on_the_fp32_path(cuda_device):
    """Tiny (fp32 states, SIMT kernels): the static array serves that path too; pools must equal scd_patch's bit for bit."""
    from paper_2606_07684_b200 import binding as B
    from paper_2606_07684_b200.harness import CodecProblem
    prob = CodecProblem(W.CONFIGS["tiny"], cuda_device)
    k, v, h = prob.make_sources()
    prob.alloc_pools()
    prob.encode(k, v, h)
    nb, L = prob.batch.n_blocks, prob.cfg.n_layers
    ref_k = [torch.full_like(p, float("nan")) for p in prob.k_pool]
    ref_v = [torch.full_like(p, float("nan")) for p in prob.v_pool]
    new_k = [t.clone() for t in ref_k]
    new_v = [t.clone() for t in ref_v]
    B.scd_patch(prob.plan, prob.bdesc, prob.codes, ref_k, ref_v, nb, prob.workspace)
    B.scd_patch_static(prob.plan, prob.bdesc, prob.codes, new_k, new_v, nb)
    torch.cuda.synchronize()
    wrote = False
    for l in range(L):
        for got, want in ((new_k[l], ref_k[l]), (new_v[l], ref_v[l])):
            assert torch.equal(got.view(torch.int32), want.view(torch.int32)), f"layer {l}"
            wrote |= bool(torch.isfinite(want).any())
    assert wrote
