"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/scd.h
declares, validates arguments on the host, and its code-buffer layout / payload accounting
agrees with the oracle's.  No compute call is made (there is no GPU here)."""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import scd_oracle as O

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    import __graft_entry__ as ge
    ge.build()                                  # nvcc cross-compiles without a GPU
    from paper_2606_07684_b200 import binding
    return binding


def test_exports_every_declared_symbol(B):
    hdr = open(os.path.join(ROOT, "include", "scd.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(scd_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(B.EXPORTS), declared ^ set(B.EXPORTS)
    for name in declared:
        assert hasattr(B.lib, name), name
    assert "sm_100a" in B.version()


def _descs(B, kinds, r_k=128, r_v=64, r_h=32, code=None, state=None):
    code = B.SCD_BF16 if code is None else code
    state = B.SCD_BF16 if state is None else state
    model = B.model_desc(n_layers=len(kinds), d_model=512, n_kv_heads=2, head_dim=64, max_position=1024,
                         state_dtype=state, code_dtype=code, rope_theta_producer=1e4)
    layers = []
    for k in kinds:
        d = B.LayerDesc()
        d.kind = k
        d.r_k, d.r_v, d.r_h, d.d_aligner = (r_k, r_v, 0, 0) if k == B.SCD_REUSE else (0, 0, r_h, 512)
        layers.append(d)
    return model, layers


@pytest.mark.parametrize("code", ["bf16", "e4m3", "f32"])
def test_code_layout_matches_oracle_payload(B, code):
    cd = {"bf16": B.SCD_BF16, "e4m3": B.SCD_E4M3_ROWSCALE, "f32": B.SCD_F32}[code]
    st = B.SCD_F32 if code == "f32" else B.SCD_BF16
    kinds = [B.SCD_REUSE, B.SCD_PATCH, B.SCD_REUSE, B.SCD_REUSE, B.SCD_PATCH]
    model, layers = _descs(B, kinds, code=cd, state=st)
    T = 1000
    # oracle accounting of |Z| (Eq. 3)
    ol = [O.Layer(O.REUSE, enc_k=np.zeros((1, 128)), enc_v=np.zeros((1, 64))) if k == B.SCD_REUSE
          else O.Layer(O.PATCH, enc_h=np.zeros((1, 32))) for k in kinds]
    om = O.Model(n_layers=5, d_model=512, n_kv_heads=2, head_dim=64, code_dtype=cd)
    _, _, _, code_bytes, payload = B.scd_code_layout(model, layers, T)
    assert payload == O.payload_bytes(om, ol, T)
    # segments: disjoint, 128-B aligned, inside the buffer, ranks as declared, K/V only on REUSE, H only on PATCH
    cb = {B.SCD_BF16: 2, B.SCD_E4M3_ROWSCALE: 1, B.SCD_F32: 4}[cd]
    spans = []
    for l, k in enumerate(kinds):
        for br in range(3):
            legal = (k == B.SCD_REUSE and br < 2) or (k == B.SCD_PATCH and br == 2)
            if not legal:
                with pytest.raises(B.ScdError):
                    B.scd_code_layout(model, layers, T, l, br)
                continue
            off, soff, rank, _, _ = B.scd_code_layout(model, layers, T, l, br)
            assert rank == {0: 128, 1: 64, 2: 32}[br] and off % 128 == 0
            spans.append((off, off + T * rank * cb))
            if cd == B.SCD_E4M3_ROWSCALE:
                assert soff % 128 == 0
                spans.append((soff, soff + 4 * T))
            else:
                assert soff == B.NO_SCALE
    spans.sort()
    assert all(a[1] <= b[0] for a, b in zip(spans, spans[1:])) and spans[-1][1] <= code_bytes
    assert code_bytes - payload < 128 * len(spans)        # only alignment padding on top of the payload
    assert B.scd_code_layout(model, layers, 0)[3] == 0


def test_code_layout_per_head_reading(B):
    """reuse_per_head: r_k / r_v are per-head ranks, a token's code row is H * r wide; the
    library's layout and payload agree with the oracle's accounting, PATCH segments are unaffected, and the
    16-byte row-pitch rule applies to the effective width."""
    kinds = [B.SCD_REUSE, B.SCD_PATCH, B.SCD_REUSE]
    model, layers = _descs(B, kinds, r_k=12, r_v=4, r_h=32)          # H = 2: code rows 24 and 8 wide
    model.reuse_per_head = 1
    T = 777
    ol = [O.Layer(O.REUSE, enc_k=np.zeros((64, 12)), enc_v=np.zeros((64, 4))) if k == B.SCD_REUSE
          else O.Layer(O.PATCH, enc_h=np.zeros((1, 32))) for k in kinds]
    om = O.Model(n_layers=3, d_model=512, n_kv_heads=2, head_dim=64, code_dtype=B.SCD_BF16, reuse_per_head=True)
    _, _, _, code_bytes, payload = B.scd_code_layout(model, layers, T)
    assert payload == O.payload_bytes(om, ol, T) == T * 2 * (2 * 24 + 2 * 8 + 32)
    assert B.scd_code_layout(model, layers, T, 0, 0)[2] == 24 and B.scd_code_layout(model, layers, T, 2, 1)[2] == 8
    assert B.scd_code_layout(model, layers, T, 1, 2)[2] == 32
    layers[0].r_k = 2                                                # H * r = 4: not a multiple of 8 on the bf16 path
    with pytest.raises(B.ScdError) as e:
        B.scd_code_layout(model, layers, T)
    assert e.value.status == 3


def test_host_side_validation(B):
    model, layers = _descs(B, [B.SCD_REUSE, B.SCD_PATCH])
    arr = (B.LayerDesc * 2)(*layers)
    h = ctypes.c_void_p()
    assert B.lib.scd_plan(None, arr, None, ctypes.byref(h)) == 1 and b"NULL" in B.lib.scd_last_error()
    assert B.lib.scd_plan(ctypes.byref(model), None, None, ctypes.byref(h)) == 1
    assert B.lib.scd_plan(ctypes.byref(model), arr, None, None) == 1
    bad = B.model_desc(n_layers=2, d_model=512, n_kv_heads=2, head_dim=48, max_position=64, state_dtype=B.SCD_BF16,
                       code_dtype=B.SCD_BF16, rope_theta_producer=1e4)
    assert B.lib.scd_plan(ctypes.byref(bad), arr, None, ctypes.byref(h)) == 3          # head_dim unsupported
    bad = B.model_desc(n_layers=500, d_model=512, n_kv_heads=2, head_dim=64, max_position=64,
                       state_dtype=B.SCD_BF16, code_dtype=B.SCD_BF16, rope_theta_producer=1e4)
    assert B.lib.scd_plan(ctypes.byref(bad), arr, None, ctypes.byref(h)) == 1
    layers[0].r_k = 20                                                              # not a multiple of 8 on bf16
    with pytest.raises(B.ScdError) as e:
        B.scd_code_layout(model, layers, 10)
    assert e.value.status == 3
    layers[0].r_k = 0
    with pytest.raises(B.ScdError) as e:
        B.scd_code_layout(model, layers, 10)
    assert e.value.status == 2
    # hot calls reject a NULL plan before touching CUDA
    assert B.lib.scd_encode(None, None, None, None, None) == 1
    assert B.lib.scd_reuse_decode(None, None, None, None, None) == 1
    assert B.lib.scd_patch(None, None, None, None, None, 0, None) == 1
    assert B.lib.scd_plan_query(None, 1, None, None, None) == 1
    assert B.lib.scd_plan_destroy(None) == 0


def test_workload_generator_basis_is_a_pca_basis():
    """The seeded generator's calibration fit (a library eigen-solver) against numpy's SVD:
    same projector, orthonormal rows; and the Tiny spectrum gives the truncation error the
    SURVEY quotes (~0.073 for r = 32)."""
    import torch
    from paper_2606_07684_b200 import workloads as W
    cfg = W.CONFIGS["tiny"]
    x = W.make_state(cfg, 0, 1, 512, "cpu")
    b, mu = W.fit_basis(x, cfg.rank)
    b, mu, xn = b.numpy(), mu.numpy(), x.double().numpy()
    np.testing.assert_allclose(b @ b.T, np.eye(cfg.rank), atol=1e-10)
    _, s, vt = np.linalg.svd(xn - mu, full_matrices=False)
    np.testing.assert_allclose(b.T @ b, vt[:cfg.rank].T @ vt[:cfg.rank], atol=1e-8)
    rel = np.sqrt((s[cfg.rank:] ** 2).sum() / (s ** 2).sum())
    assert 0.06 < rel < 0.085
    # regenerating a row range gives the same bits
    y = W.make_state(cfg, 0, 1, 100, "cpu", row_offset=200)
    assert torch.equal(y, x[200:300])


def test_int4_layout_matches_oracle_payload_and_rejects_bad_groups(B):
    """scd_int4_layout (pure host): payload = oracle's |Z| for the INT4 codec (Eq. 3 :86); segments
    disjoint and 128-B aligned; unsupported groups rejected."""
    from oracle import int4_oracle as Q
    for group in (32, 64, 128):
        desc = B.Int4Desc(8, 128, 16, group)
        for T, n in ((1000, 3), (1, 1), (8192, 64)):
            stride, moff, total, payload = B.scd_int4_layout(desc, T, n)
            assert payload == Q.payload_bytes(T, 1024, group, n)
            assert stride % 128 == 0 and moff % 128 == 0 and total == stride * n
            assert T * 512 <= moff and moff + T * (1024 // group) * 4 <= stride
    for bad in (B.Int4Desc(8, 128, 16, 16), B.Int4Desc(8, 64, 16, 128), B.Int4Desc(0, 128, 16, 32)):
        with pytest.raises(B.ScdError):
            B.scd_int4_layout(bad, 10, 1)


def test_struct_layouts_agree_with_the_library(B):
    """The ctypes structs of the binding have the sizes the C compiler gave the ABI structs (scd_struct_size)."""
    import ctypes as C
    for which, cls in enumerate((B.ModelDesc, B.LayerDesc, B.BatchDesc, B.SrcDesc, B.PagedKV, B.Int4Desc, B.FitDesc)):
        assert B.lib.scd_struct_size(which) == C.sizeof(cls), cls.__name__
    assert B.lib.scd_struct_size(99) == -1


def test_fit_query_is_pure_host_arithmetic(B):
    """scd_fit_query validates the descriptor and sizes the workspace without touching a device: the K-major copy of
    X = [A B] (2 W x ceil(N / 64) * 64 bf16) dominates; bad descriptors come back with the documented statuses."""
    d = B.FitDesc(1024, 128, 1, 1e-3, B.SCD_BF16, B.SCD_BF16)
    ws = B.scd_fit_query(d, 100000)
    xt = 2 * 1024 * ((100000 + 63) // 64 * 64) * 2
    assert xt < ws < xt + 200 * (1 << 20) and B.scd_fit_query(d, 1) < B.scd_fit_query(d, 100000)
    for desc, status in ((B.FitDesc(60, 8, 0, 1e-3, B.SCD_BF16, B.SCD_F32), 2), (B.FitDesc(2048, 8, 0, 1e-3, B.SCD_BF16, B.SCD_F32), 3),
                         (B.FitDesc(64, 0, 0, 1e-3, B.SCD_BF16, B.SCD_F32), 2), (B.FitDesc(64, 8, 0, 1e-3, B.SCD_F32, B.SCD_F32), 3),
                         (B.FitDesc(64, 8, 0, 1e-3, B.SCD_BF16, B.SCD_E4M3_ROWSCALE), 1)):
        with pytest.raises(B.ScdError) as e:
            B.scd_fit_query(desc, 64)
        assert e.value.status == status
    with pytest.raises(B.ScdError):
        B.scd_fit_query(d, 0)
